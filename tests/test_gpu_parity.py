"""GPU parity: the CUDA path (through the C ABI and its Python binding) against
the fp64 CPU oracle on the same seeded inputs.

Bars (BASELINE.json north_star): integer ray table
(j0, n) bit-exact; signal within 1e-4 relative per pixel; line integrals within
1e-4 relative plus a floor of 1e-6 of the image maximum (grazing rays).
"""
import math
import zlib

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from parity_util import (check_line_integrals, check_ray_table, check_signal,  # noqa: E402
                         compare_full)
from test_oracle_pins import tiny_workload  # noqa: E402
from workloads import make_workload  # noqa: E402


@pytest.fixture(scope="module")
def gdrr():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    import paper_1204_6367_b200 as g
    return g


LAYOUTS = [0, 1, 2]


# ---------------------------------------------------------------- C0 .. C2, full images

@pytest.mark.parametrize("layout", LAYOUTS)
@pytest.mark.parametrize("name", ["C0", "C1"])
def test_full_image_parity_small(gdrr, workloads_cache, name, layout):
    w = workloads_cache(name)
    ref = oracle.project(w)
    with gdrr.Projector(w, layout=layout) as pr:
        stats = compare_full(pr, w, ref, f"{name} layout {layout}")
        assert pr.count_samples() == int(ref["ray_table"][..., 1].sum())
    print(name, layout, stats)


@pytest.mark.parametrize("phi_deg", [0.0, 37.0])
def test_full_image_parity_c2(gdrr, workloads_cache, phi_deg):
    """C2 at its timed angle and at 37 degrees, so that no axis alignment can
    hide an indexing slip."""
    w = workloads_cache("C2").with_phis([math.radians(phi_deg)])
    ref = oracle.project(w)
    with gdrr.Projector(w) as pr:
        stats = compare_full(pr, w, ref, f"C2 phi {phi_deg}")
    print("C2", phi_deg, stats)


def test_multi_projection_batch_and_ranges(gdrr, workloads_cache):
    """Several angles in one launch, and sub-ranges (proj_begin / proj_count)
    give the same images as the oracle's per-angle results."""
    phis = np.radians([0.0, 37.0, 90.0, 123.4, 180.0, 270.0, 315.0])
    w = workloads_cache("C1").with_phis(phis)
    ref = oracle.project(w)
    with gdrr.Projector(w) as pr:
        compare_full(pr, w, ref, "C1 x 7 angles")
        sig, li, tab = pr.project(proj_begin=2, proj_count=3, want_li=True, want_table=True)
        check_ray_table(tab.cpu().numpy(), ref["ray_table"][2:5])
        check_signal(sig.cpu().numpy(), ref["signal"][2:5])
        check_line_integrals(li.cpu().numpy(), ref["line_integrals"][2:5])


@pytest.mark.parametrize("sampler", [1, 2])
def test_both_packed_samplers_against_the_oracle(gdrr, workloads_cache, sampler):
    """GDRR_SAMPLER_GATHER (1) and GDRR_SAMPLER_STAGED (2) explicitly: C1 at 7 angles (bounding boxes fit the
    staged box), C0 (they do not: every chunk takes the gather fallback inside the staged kernel) and a ragged
    three-material volume."""
    phis = np.radians([0.0, 37.0, 90.0, 123.4, 180.0, 270.0, 315.0])
    w = workloads_cache("C1").with_phis(phis)
    with gdrr.Projector(w, sampler=sampler) as pr:
        compare_full(pr, w, oracle.project(w), f"C1 x 7 angles sampler {sampler}")
    w = workloads_cache("C0")
    with gdrr.Projector(w, sampler=sampler) as pr:
        compare_full(pr, w, oracle.project(w), f"C0 sampler {sampler}")
    rng = np.random.default_rng(8)
    rho = rng.uniform(0.0, 2.0, size=(19, 23, 29)).astype(np.float32)
    mat = rng.integers(0, 3, size=rho.shape).astype(np.uint8)
    w = tiny_workload(rho, mat, n_materials=3, spacing=(1.0, 1.0, 1.3), nu=45, nv=39, du=0.8, dv=0.8,
                      phis=np.radians([15.0, 100.0, 222.0]), step=0.5, mu_hat=rng.uniform(0.01, 0.03, size=(3, 1)))
    with gdrr.Projector(w, sampler=sampler) as pr:
        compare_full(pr, w, oracle.project(w), f"ragged sampler {sampler}")
    # one material (untagged words, no purity vote) with a beam that fits the staged box
    w1 = tiny_workload(rho, None, n_materials=1, spacing=(1.0, 1.0, 1.3), nu=45, nv=39, du=0.8, dv=0.8,
                       phis=np.radians([15.0, 100.0, 222.0]), step=0.5)
    with gdrr.Projector(w1, sampler=sampler) as pr:
        compare_full(pr, w1, oracle.project(w1), f"one material sampler {sampler}")
    # long steps: 2.5 voxels per step (no chunk fits the staged box) and 10 voxels per step (16 steps would
    # overflow the in-chunk fixed point: the library must fall back to the gather kernel's short chunks)
    for step in (2.5, 10.0):
        ws = tiny_workload(rho, mat, n_materials=3, spacing=(1.0, 1.0, 1.3), nu=45, nv=39, du=0.8, dv=0.8,
                           phis=np.radians([15.0, 222.0]), step=step, mu_hat=rng.uniform(0.01, 0.03, size=(3, 1)))
        with gdrr.Projector(ws, sampler=sampler) as pr:
            compare_full(pr, ws, oracle.project(ws), f"step {step} sampler {sampler}")


@pytest.mark.parametrize("phantom", ["noisy3", "random"])
@pytest.mark.parametrize("sampler", [1, 2])
def test_c2_phantom_variants_full_image(gdrr, phantom, sampler):
    """The mixed-cell paths at clinical size: C2 with 3 % voxel noise before the material thresholds (13 % of its cells
    mix two materials: the masked second blend) and with a material drawn per voxel (every cell mixes three or four:
    the routed corners), every pixel of a projection at 37 degrees against the oracle, both samplers."""
    w = make_workload("C2", phantom=phantom).with_phis([math.radians(37.0)])
    ref = oracle.project(w)
    with gdrr.Projector(w, sampler=sampler) as pr:
        stats = compare_full(pr, w, ref, f"C2 {phantom} sampler {sampler}")
    print(phantom, sampler, stats)


def test_staged_and_gather_samplers_agree(gdrr, workloads_cache):
    """Same samples, same blend; only the summation chunks (16 vs 32) and the re-basing of the position differ."""
    w = workloads_cache("C2").with_phis(np.radians([0.0, 37.0, 211.0]))
    with gdrr.Projector(w, sampler=1) as a, gdrr.Projector(w, sampler=2) as b:
        sa, la, ta = a.project(want_li=True, want_table=True)
        sb, lb, tb = b.project(want_li=True, want_table=True)
    assert torch.equal(ta, tb)
    assert ((sa - sb).abs() / sa).max().item() < 2e-5
    assert (la - lb).abs().max().item() < 2e-5 * la.max().item()
    with pytest.raises(gdrr.GdrrError):
        with gdrr.Projector(workloads_cache("C0"), sampler=7):
            pass


# ---------------------------------------------------------------- C3 / C4 at full size, sampled

def _sampled_scan_parity(gdrr, w, projections, n_pix, seed, what):
    rng = np.random.default_rng(seed)
    with gdrr.Projector(w) as pr:
        total_err = 0.0
        for p in projections:
            ii = rng.integers(0, w.nu, n_pix)
            jj = rng.integers(0, w.nv, n_pix)
            # always include the corners and the centre of the detector
            ii[:5] = [0, w.nu - 1, 0, w.nu - 1, w.nu // 2]
            jj[:5] = [0, 0, w.nv - 1, w.nv - 1, w.nv // 2]
            pix = np.stack([np.full(n_pix, p), ii, jj], axis=1)
            ref = oracle.project(w, pixels=pix)
            sig, li, tab = pr.project(proj_begin=p, proj_count=1, want_li=True, want_table=True)
            sig = sig[0].cpu().numpy()[jj, ii]
            li = li[0].cpu().numpy()[:, jj, ii].T
            tab = tab[0].cpu().numpy()[jj, ii]
            check_ray_table(tab, ref["ray_table"], f"{what} p={p}")
            check_line_integrals(li, ref["line_integrals"], f"{what} p={p}")
            total_err = max(total_err, check_signal(sig, ref["signal"], f"{what} p={p}"))
        print(what, "max relative signal error", total_err)


def test_c3_full_size_sampled(gdrr, workloads_cache):
    """C3 in the launch configuration bench.py times, 8 projections x 3000
    sampled pixels against the oracle (p = 0, N/8, 37, N/4, ...)."""
    w = workloads_cache("C3")
    n = w.n_proj
    _sampled_scan_parity(gdrr, w, [0, n // 8, 37, n // 4, n // 3, n // 2, int(0.7 * n), n - 1],
                         3000, 33, "C3")


def test_c3_batched_launch_equals_single_launches(gdrr, workloads_cache):
    """The batched launch bench.py uses (many projections per launch) returns
    bit-identical images to one launch per projection."""
    w = workloads_cache("C3")
    with gdrr.Projector(w) as pr:
        batch, _, _ = pr.project(proj_begin=40, proj_count=6)
        for k in range(6):
            one, _, _ = pr.project(proj_begin=40 + k, proj_count=1)
            assert torch.equal(batch[k], one[0])


def test_c4_full_size_sampled(gdrr, workloads_cache):
    w = workloads_cache("C4")
    n = w.n_proj
    _sampled_scan_parity(gdrr, w, [0, n // 8, n // 3, n - 1], 2000, 44, "C4")


# ---------------------------------------------------------------- closed forms on the GPU path itself

def test_empty_volume_gives_flat_field(gdrr, workloads_cache):
    w0 = workloads_cache("C2")
    import copy
    w = copy.copy(w0)
    w.rho = np.zeros_like(w0.rho)
    rng = np.random.default_rng(5)
    w.fluence_map = rng.uniform(0.5, 1.5, size=(w.nv, w.nu)).astype(np.float32)
    flat = np.zeros((w.nv, w.nu))
    for e in range(w.n_energy):
        flat += (w.phi_weight[e] * w.response[e]
                 * np.exp(-w.bowtie_mu[e] * w.bowtie_thickness)[None, :] * w.fluence_map)
    with gdrr.Projector(w) as pr:
        sig, li, _ = pr.project(want_li=True)
    assert float(li.abs().max()) == 0.0
    check_signal(sig[0].cpu().numpy(), flat, "flat field")


def test_uniform_volume_integrates_to_n_times_step(gdrr):
    """rho = const everywhere: LI = rho0 * n * dl exactly up to fp32 rounding
    (clamp-to-edge, reading Q7; oracle pin P3)."""
    rho = np.full((12, 20, 16), 1.25, dtype=np.float32)
    w = tiny_workload(rho, spacing=(2.0, 1.5, 3.0), nu=40, nv=36, du=2.0, dv=2.0,
                      phis=np.radians([0.0, 30.0, 90.0, 200.0]), step=0.37)
    with gdrr.Projector(w) as pr:
        _, li, tab = pr.project(want_li=True, want_table=True)
    n = tab[..., 1].cpu().numpy().astype(np.float64)
    got = li[:, 0].cpu().numpy().astype(np.float64)
    np.testing.assert_allclose(got, 1.25 * n * 0.37, rtol=2e-6, atol=0)


# ---------------------------------------------------------------- edge cases

def _random_volume(rng, shape, n_mat):
    rho = rng.uniform(0.0, 2.0, size=shape).astype(np.float32)
    rho[rng.uniform(size=shape) < 0.2] = 0.0
    mat = rng.integers(0, n_mat, size=shape).astype(np.uint8)
    return rho, mat


@pytest.mark.parametrize("layout", LAYOUTS)
@pytest.mark.parametrize("case", ["ragged", "odd_aniso_offcentre", "theta_offset", "three_materials",
                                  "long_step", "one_voxel", "thin_slab", "long_thin"])
def test_edge_cases(gdrr, case, layout):
    rng = np.random.default_rng(zlib.crc32(case.encode()))
    kw = dict(nu=37, nv=29, du=2.5, dv=2.5, step=0.5,
              phis=np.radians([0.0, 17.0, 90.0, 181.0, 271.5]))
    n_mat, shape, spacing = 2, (14, 18, 22), (2.0, 2.0, 2.0)
    if case == "ragged":
        kw.update(nu=33, nv=17)                       # not multiples of the 16 x 16 tile
    elif case == "odd_aniso_offcentre":
        shape, spacing = (9, 13, 17), (1.3, 2.1, 3.7)
        kw.update(centre=(12.0, -7.5, 4.0), nu=50, nv=40)
    elif case == "theta_offset":
        kw.update(theta=math.radians(9.0), nu=61, du=4.0)
    elif case == "three_materials":
        n_mat = 3
    elif case == "long_step":
        kw.update(step=5.3)                           # several voxels per step
    elif case == "one_voxel":
        shape, spacing = (1, 1, 1), (30.0, 30.0, 30.0)
        kw.update(step=1.0)
    elif case == "thin_slab":
        shape = (1, 24, 24)
        kw.update(step=0.25)
    elif case == "long_thin":                         # 1500 voxels along x: cell indices beyond 1024, rays of 3000 samples
        shape, spacing = (5, 6, 1500), (0.25, 0.5, 0.5)
        kw.update(step=0.125, nu=40, nv=8, du=0.3, dv=0.3, phis=np.radians([0.0, 2.0, 90.0, 178.5]))
    rho, mat = _random_volume(rng, shape, n_mat)
    energies = np.array([30.0, 60.0, 90.0])
    mu_hat = rng.uniform(0.01, 0.05, size=(n_mat, 3))
    w = tiny_workload(rho, mat, spacing=spacing, n_materials=n_mat, energies=energies, mu_hat=mu_hat,
                      phi_weight=np.array([0.2, 0.5, 0.3]), response=energies, **kw)
    if case == "theta_offset":
        w.u_off, w.v_off = 11.0, -6.0
    ref = oracle.project(w)
    with gdrr.Projector(w, layout=layout) as pr:
        stats = compare_full(pr, w, ref, f"{case} layout {layout}")
    assert ref["ray_table"][..., 1].max() > 0
    print(case, layout, stats)


@pytest.mark.parametrize("n_energy", [1, 7, 512])
def test_energy_grid_sizes_up_to_the_maximum(gdrr, n_energy):
    """1, an odd number and GDRR_MAX_ENERGIES = 512 energy bins (the tables then take 12 KB of every CTA's shared memory:
    the staged kernel runs two CTAs per SM instead of three), three materials, every layout and sampler."""
    rng = np.random.default_rng(n_energy)
    rho, mat = _random_volume(rng, (18, 22, 26), 3)
    energies = np.linspace(20.0, 140.0, n_energy) if n_energy > 1 else np.array([60.0])
    w = tiny_workload(rho, mat, n_materials=3, spacing=(1.0, 1.2, 1.4), nu=44, nv=38, du=0.9, dv=0.9,
                      phis=np.radians([12.0, 200.0]), step=0.45, energies=energies,
                      mu_hat=rng.uniform(0.01, 0.05, size=(3, n_energy)),
                      phi_weight=rng.dirichlet(np.ones(n_energy)), response=energies / 60.0)
    w.bowtie_mu = rng.uniform(0.02, 0.08, size=n_energy)
    w.bowtie_thickness = rng.uniform(1.0, 10.0, size=w.nu)
    ref = oracle.project(w)
    for layout, sampler in ((2, 1), (2, 2), (0, 0), (1, 0)):
        with gdrr.Projector(w, layout=layout, sampler=sampler) as pr:
            compare_full(pr, w, ref, f"{n_energy} bins layout {layout} sampler {sampler}")
    with pytest.raises(gdrr.GdrrError) as e:
        gdrr.gdrr_set_spectrum(gdrr.gdrr_create_context(0), np.ones(513) / 513, np.ones(513), np.ones((1, 513)))
    assert e.value.code == gdrr.GDRR_ERR_INVALID_ARG


def test_rays_parallel_to_axes_and_all_miss(gdrr):
    """Odd detector: the central ray is exactly axis parallel at phi = 0 and has
    a zero direction component (reading Q17); a far-off detector misses the box."""
    rng = np.random.default_rng(8)
    rho, mat = _random_volume(rng, (10, 10, 10), 1)
    w = tiny_workload(rho, None, nu=17, nv=17, du=4.0, dv=4.0,
                      phis=np.radians([0.0, 90.0, 180.0, 270.0]))
    ref = oracle.project(w)
    with gdrr.Projector(w) as pr:
        compare_full(pr, w, ref, "axis parallel")
    w2 = tiny_workload(rho, None, nu=16, nv=16, du=1.0, dv=1.0, phis=[0.3])
    w2.v_off = 400.0
    ref2 = oracle.project(w2)
    assert ref2["ray_table"][..., 1].max() == 0
    with gdrr.Projector(w2) as pr:
        out = compare_full(pr, w2, ref2, "all miss")
    assert out["signal"] <= 1e-6


def test_cell_indices_agree_with_oracle_positions(gdrr, workloads_cache):
    """Reading Q9: the kernel's in-chunk fixed-point positions give the same cell
    as the oracle's fp64 positions except within 2^-12 of a cell face.  Checked
    through the line integrals of a volume whose value IS its cell index along
    x (a ramp): tri-linear interpolation reproduces gx exactly, so LI / (n dl)
    is the mean x index coordinate of the samples."""
    n = 32
    ramp = np.broadcast_to(np.arange(n, dtype=np.float32)[None, None, :], (n, n, n)).copy()
    w = tiny_workload(ramp, nu=48, nv=48, du=1.5, dv=1.5, step=0.5,
                      phis=np.radians([0.0, 33.0, 77.0]))
    ref = oracle.project(w)
    with gdrr.Projector(w) as pr:
        _, li, tab = pr.project(want_li=True, want_table=True)
    check_ray_table(tab.cpu().numpy(), ref["ray_table"])
    got = li[:, 0].cpu().numpy().astype(np.float64)
    want = ref["line_integrals"][:, 0]
    hit = ref["ray_table"][..., 1] > 4
    mean_pos_err = np.abs(got - want)[hit] / (ref["ray_table"][..., 1][hit] * 0.5)
    assert mean_pos_err.max() < 2e-5, mean_pos_err.max()   # index units


# ---------------------------------------------------------------- the ABI's error behaviour on a live device

def test_error_codes_on_device(gdrr):
    ctx = gdrr.gdrr_create_context(0)
    try:
        sig = torch.empty((1, 8, 8), dtype=torch.float32, device="cuda")
        rho = torch.ones((4, 4, 4), dtype=torch.float32, device="cuda")
        mat = torch.zeros((4, 4, 4), dtype=torch.uint8, device="cuda")
        ws = torch.empty(gdrr.gdrr_volume_workspace_bytes(4, 4, 4, 1, 0), dtype=torch.uint8, device="cuda")
        vol = gdrr.gdrr_create_volume(ctx, rho, mat, (4, 4, 4), (1, 1, 1), None, 1, 0, ws)
        with pytest.raises(gdrr.GdrrError) as e:
            gdrr.gdrr_project(ctx, vol, 0, 1, sig)
        assert e.value.code == gdrr.GDRR_ERR_NOT_READY
        gdrr.gdrr_set_geometry(ctx, 1000, 1500, 0, 8, 8, 1, 1, 0, 0, [0.0, 1.0], 0.0)
        with pytest.raises(gdrr.GdrrError) as e:
            gdrr.gdrr_project(ctx, vol, 0, 1, sig)
        assert e.value.code == gdrr.GDRR_ERR_NOT_READY
        gdrr.gdrr_set_spectrum(ctx, [1.0], [1.0], [[0.02], [0.03]])
        with pytest.raises(gdrr.GdrrError) as e:                    # 2 materials vs 1
            gdrr.gdrr_project(ctx, vol, 0, 1, sig)
        assert e.value.code == gdrr.GDRR_ERR_NOT_READY
        gdrr.gdrr_set_spectrum(ctx, [1.0], [1.0], [[0.02]])
        with pytest.raises(gdrr.GdrrError) as e:                    # range
            gdrr.gdrr_project(ctx, vol, 1, 2, torch.empty((2, 8, 8), dtype=torch.float32, device="cuda"))
        assert e.value.code == gdrr.GDRR_ERR_INVALID_ARG
        with pytest.raises(ValueError):                             # the binding checks what the C ABI cannot see:
            gdrr.gdrr_project(ctx, vol, 0, 2, sig)                  # an output tensor smaller than the request
        gdrr.gdrr_project(ctx, vol, 0, 1, sig)
        torch.cuda.synchronize()
        # a material index out of range is caught on the device: gdrr_create_volume does not wait for the check,
        # gdrr_volume_status does, and every later call on the volume refuses it
        gdrr.gdrr_volume_status(ctx, vol)                       # the good volume
        mat_bad = mat.clone()
        mat_bad[1, 2, 3] = 5
        ws2 = torch.empty_like(ws)
        bad = gdrr.gdrr_create_volume(ctx, rho, mat_bad, (4, 4, 4), (1, 1, 1), None, 1, 0, ws2)
        with pytest.raises(gdrr.GdrrError) as e:
            gdrr.gdrr_volume_status(ctx, bad)
        assert e.value.code == gdrr.GDRR_ERR_INVALID_ARG
        with pytest.raises(gdrr.GdrrError) as e:
            gdrr.gdrr_project(ctx, bad, 0, 1, sig)
        assert e.value.code == gdrr.GDRR_ERR_INVALID_ARG
        gdrr.gdrr_destroy_volume(bad)
        # ... also without gdrr_volume_status, by the first call that finds the ingest finished
        for layout in (0, 1, 2):
            wsl = torch.empty(gdrr.gdrr_volume_workspace_bytes(4, 4, 4, 1, layout), dtype=torch.uint8, device="cuda")
            bad = gdrr.gdrr_create_volume(ctx, rho, mat_bad, (4, 4, 4), (1, 1, 1), None, 1, layout, wsl)
            torch.cuda.synchronize()
            with pytest.raises(gdrr.GdrrError) as e:
                gdrr.gdrr_project(ctx, bad, 0, 1, sig)
            assert e.value.code == gdrr.GDRR_ERR_INVALID_ARG
            gdrr.gdrr_destroy_volume(bad)
        gdrr.gdrr_project(ctx, vol, 0, 1, sig)                  # the good volume still works
        # workspace too small
        with pytest.raises(gdrr.GdrrError) as e:
            gdrr.gdrr_create_volume(ctx, rho, mat, (4, 4, 4), (1, 1, 1), None, 1, 0, ws[:100])
        assert e.value.code == gdrr.GDRR_ERR_WORKSPACE
        # source inside the volume box
        big = tiny_workload(np.ones((4, 4, 4), dtype=np.float32), spacing=(600.0, 600.0, 600.0))
        with pytest.raises(gdrr.GdrrError) as e:
            with gdrr.Projector(big) as pr:
                pr.project()
        assert e.value.code == gdrr.GDRR_ERR_INVALID_ARG
        gdrr.gdrr_destroy_volume(vol)
    finally:
        gdrr.gdrr_destroy_context(ctx)


def test_host_buffer_entry_points(gdrr, workloads_cache):
    """gdrr_create_volume_host + gdrr_project_host (the e2e path of bench.py)
    give the same bits as the device-buffer path."""
    w = workloads_cache("C1").with_phis(np.radians([0.0, 45.0, 90.0, 135.0, 200.0]))
    with gdrr.Projector(w) as pr:
        want, _, _ = pr.project()
        want = want.cpu()
    with gdrr.Projector(w, from_host=True) as pr:
        rho_h = torch.from_numpy(w.rho).pin_memory()
        mat_h = torch.from_numpy(w.mat).pin_memory()
        pr.ingest_host(rho_h, mat_h)
        out = torch.empty((w.n_proj, w.nv, w.nu), dtype=torch.float32).pin_memory()
        for stage_proj in (1, 2, 4, 5, 8):
            out.zero_()
            stage = torch.empty((stage_proj, w.nv, w.nu), dtype=torch.float32, device="cuda")
            gdrr.gdrr_project_host(pr.ctx, pr.vol, 0, w.n_proj, out, stage, stage_proj)
            assert torch.equal(out, want), stage_proj
