"""GPU parity on general source paths (gdrr_set_geometry_poses; helical and C-arm
orbits, free poses) against the oracle's pose path, which tests/test_oracle_pose_pins.py pins.

Bars as in test_gpu_parity.py: integer ray table bit-exact, signal 1e-4 relative, line integrals 1e-4
relative plus the grazing-ray floor; Siddon as in test_gpu_siddon.py."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from parity_util import check_line_integrals, check_ray_table, check_signal, compare_full  # noqa: E402
from test_oracle_pins import tiny_workload  # noqa: E402
from workloads import trajectories  # noqa: E402


@pytest.fixture(scope="module")
def gdrr():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    import paper_1204_6367_b200 as g
    return g


def _helix(w, n, turns=1.5, pitch=60.0):
    phis = 2 * math.pi * turns * np.arange(n) / n
    return trajectories.helical_poses(w.sad, w.sdd, phis, pitch, z0_mm=-0.5 * pitch * turns)


def _c_arm(w, n, tilt_deg=25.0):
    phis = 2 * math.pi * np.arange(n) / n + 0.1
    return trajectories.c_arm_poses(w.sad, w.sdd, phis, math.radians(tilt_deg))


@pytest.mark.parametrize("layout", [0, 1, 2])
def test_circular_poses_reproduce_the_gantry_bit_for_bit(gdrr, workloads_cache, layout):
    """gdrr_set_geometry is gdrr_set_geometry_poses on the circle's poses: same kernels, same numbers."""
    phis = np.radians([0.0, 37.0, 123.4, 270.0])
    w = workloads_cache("C1").with_phis(phis)
    wp = w.with_poses(trajectories.circular_poses(w.sad, w.sdd, w.theta, phis))
    with gdrr.Projector(w, layout=layout) as a, gdrr.Projector(wp, layout=layout) as b:
        sa, la, ta = a.project(want_li=True, want_table=True)
        sb, lb, tb = b.project(want_li=True, want_table=True)
        assert torch.equal(ta, tb) and torch.equal(sa, sb) and torch.equal(la, lb)


@pytest.mark.parametrize("sampler", [1, 2])
@pytest.mark.parametrize("path", ["helix", "c_arm", "free"])
def test_pose_paths_full_image_parity_c1(gdrr, workloads_cache, path, sampler):
    w0 = workloads_cache("C1")
    poses = {"helix": lambda: _helix(w0, 6), "c_arm": lambda: _c_arm(w0, 6),
             "free": lambda: trajectories.free_poses(6, w0.sad, w0.sdd, seed=2024)}[path]()
    w = w0.with_poses(poses)
    ref = oracle.project(w)
    assert int(ref["ray_table"][..., 1].sum()) > 1e6
    with gdrr.Projector(w, sampler=sampler) as pr:
        stats = compare_full(pr, w, ref, f"C1 {path} sampler {sampler}")
        assert pr.count_samples() == int(ref["ray_table"][..., 1].sum())
        sig, li, tab = pr.project(proj_begin=2, proj_count=3, want_li=True, want_table=True)
        check_ray_table(tab.cpu().numpy(), ref["ray_table"][2:5])
        check_signal(sig.cpu().numpy(), ref["signal"][2:5])
    print(path, sampler, stats)


@pytest.mark.parametrize("layout", [0, 1])
def test_pose_paths_exact_layouts_ragged_volume(gdrr, layout):
    rng = np.random.default_rng(31)
    nx, ny, nz = 45, 37, 29
    rho = rng.uniform(0.0, 1.8, size=(nz, ny, nx)).astype(np.float32)
    mat = rng.integers(0, 3, size=(nz, ny, nx)).astype(np.uint8)
    w = tiny_workload(rho, mat, spacing=(1.7, 2.1, 2.6), n_materials=3, nu=53, nv=41, du=2.5, dv=2.9,
                      step=0.6, mu_hat=[[0.02, 0.018], [0.03, 0.022], [0.06, 0.04]],
                      energies=[50.0, 80.0], centre=(4.0, -3.0, 6.0))
    w.u_off, w.v_off = 6.0, -4.0
    w = w.with_poses(np.concatenate([_helix(w, 3, 0.7, 30.0), _c_arm(w, 3, 40.0),
                                     trajectories.free_poses(3, w.sad, w.sdd, seed=5)]))
    ref = oracle.project(w)
    with gdrr.Projector(w, layout=layout) as pr:
        print(layout, compare_full(pr, w, ref, f"ragged poses layout {layout}"))


def test_pose_paths_c2_tilted_orbit_sampled_pixels(gdrr, workloads_cache):
    """C2 at full size on a tilted C-arm orbit and a helix, on sampled pixels the oracle computes one by one."""
    w0 = workloads_cache("C2")
    w = w0.with_poses(np.concatenate([_c_arm(w0, 2, 20.0), _helix(w0, 2, 0.4, 80.0)]))
    rng = np.random.default_rng(8)
    pix = np.stack([rng.integers(0, 4, 3000), rng.integers(0, w.nu, 3000), rng.integers(0, w.nv, 3000)], axis=1)
    ref = oracle.project(w, pixels=pix)
    with gdrr.Projector(w) as pr:
        sig, li, tab = pr.project(want_li=True, want_table=True)
    sig, li, tab = sig.cpu().numpy(), li.cpu().numpy(), tab.cpu().numpy()
    p, i, j = pix[:, 0], pix[:, 1], pix[:, 2]
    check_ray_table(tab[p, j, i], ref["ray_table"])
    check_signal(sig[p, j, i], ref["signal"], "C2 poses")
    check_line_integrals(li[p, :, j, i], ref["line_integrals"], "C2 poses")
    assert (ref["ray_table"][:, 1] > 0).mean() > 0.5


def test_pose_paths_siddon(gdrr, workloads_cache):
    w0 = workloads_cache("C1")
    w = w0.with_poses(np.concatenate([_helix(w0, 2), _c_arm(w0, 2), trajectories.free_poses(2, w0.sad, w0.sdd, 6)]))
    ref = oracle.project(w, method="siddon")
    for layout in (1, 2):
        with gdrr.Projector(w, layout=layout, method=gdrr.GDRR_METHOD_SIDDON) as pr:
            sig, li, tab = pr.project(want_li=True, want_table=True)
        li, sig = li.cpu().numpy().astype(np.float64), sig.cpu().numpy().astype(np.float64)
        scale = ref["line_integrals"].max()
        err = np.abs(li - ref["line_integrals"])
        assert np.all(err <= 1e-4 * np.abs(ref["line_integrals"]) + 2e-6 * scale), float(err.max())
        check_signal(sig, ref["signal"], f"siddon poses layout {layout}")
        check_ray_table(tab.cpu().numpy(), ref["ray_table"])


def test_pose_edge_cases(gdrr):
    """A pose looking away from the volume: flat field, n = 0 everywhere; a source inside the volume box: error."""
    rho = np.ones((8, 8, 8), dtype=np.float32)
    w = tiny_workload(rho, spacing=(2.0, 2.0, 2.0), nu=20, nv=18, du=4.0, dv=4.0, sad=300.0, sdd=500.0)
    away = trajectories.circular_poses(300.0, 500.0, 0.0, [0.0, 1.0])
    away[:, 3:6] = 2.6 * away[:, 0:3]                       # detector behind the source
    ref = oracle.project(w.with_poses(away))
    for layout in (0, 1, 2):
        with gdrr.Projector(w.with_poses(away), layout=layout) as pr:
            sig, li, tab = pr.project(want_li=True, want_table=True)
            check_ray_table(tab.cpu().numpy(), ref["ray_table"])
            assert torch.count_nonzero(li).item() == 0
            check_signal(sig.cpu().numpy(), ref["signal"], "away")
    inside = trajectories.circular_poses(300.0, 500.0, 0.0, [0.0])
    inside[0, 0:3] = (1.0, -2.0, 0.5)
    with gdrr.Projector(w.with_poses(inside)) as pr:
        with pytest.raises(gdrr.GdrrError):
            pr.project()


@pytest.mark.parametrize("sampler", [1, 2])
def test_skewed_and_stretched_detector_frames(gdrr, workloads_cache, sampler):
    """u_hat and v_hat are used as given: a frame that is neither unit nor orthogonal (pixels 1.25 x wider along u, v
    leaning 12 degrees towards u) and a detector rotated in its own plane.  The staged sampler's bound on how far a
    tile's rays leave the hull of its corner rays scales with these vectors (gdrr_api.cu hull_margins): a wrong bound
    would show as quads read outside the staged box."""
    w0 = workloads_cache("C1")
    phis = np.radians([5.0, 95.0, 230.0])
    poses = trajectories.circular_poses(w0.sad, w0.sdd, 0.0, phis)
    skew = poses.copy()
    skew[:, 6:9] *= 1.25                                                   # stretched u
    skew[:, 9:12] = np.cos(0.21) * poses[:, 9:12] + np.sin(0.21) * poses[:, 6:9]   # v leaning towards u
    c, s_ = math.cos(0.6), math.sin(0.6)
    rot = poses.copy()
    rot[:, 6:9] = c * poses[:, 6:9] + s_ * poses[:, 9:12]                 # detector rotated by 34 degrees in its plane
    rot[:, 9:12] = -s_ * poses[:, 6:9] + c * poses[:, 9:12]
    for what, ps in (("skewed", skew), ("rotated", rot)):
        w = w0.with_poses(ps)
        with gdrr.Projector(w, sampler=sampler) as pr:
            stats = compare_full(pr, w, oracle.project(w), f"{what} frame sampler {sampler}")
        print(what, sampler, stats)


def test_pose_argument_errors(gdrr):
    ctx = gdrr.gdrr_create_context(0)
    try:
        good = trajectories.circular_poses(1000.0, 1500.0, 0.0, [0.0, 1.0])
        gdrr.gdrr_set_geometry_poses(ctx, 8, 8, 1.0, 1.0, 0.0, 0.0, good, 0.5)
        bad = good.copy(); bad[1, 9:12] = bad[1, 6:9]               # u_hat parallel to v_hat
        with pytest.raises(gdrr.GdrrError):
            gdrr.gdrr_set_geometry_poses(ctx, 8, 8, 1.0, 1.0, 0.0, 0.0, bad, 0.5)
        bad = good.copy(); bad[0, 0:3] = bad[0, 3:6]                # source in the detector plane
        with pytest.raises(gdrr.GdrrError):
            gdrr.gdrr_set_geometry_poses(ctx, 8, 8, 1.0, 1.0, 0.0, 0.0, bad, 0.5)
        bad = good.copy(); bad[0, 4] = np.nan
        with pytest.raises(gdrr.GdrrError):
            gdrr.gdrr_set_geometry_poses(ctx, 8, 8, 1.0, 1.0, 0.0, 0.0, bad, 0.5)
    finally:
        gdrr.gdrr_destroy_context(ctx)
