"""Pins for the oracle's Siddon option (oracle/gdrr_oracle.c, ray_siddon) against things other
than itself.  PAPER.md:151 and 413 name Siddon's exact radiological path (piecewise-constant
voxels) as gDRR's optional line integral; the paper prints no value for it, so it is pinned by
the definition LI_m = sum_voxels rho [mat = m] |ray /\\ voxel| evaluated another way (one slab
clip per voxel, brute force), by closed forms, and by the fine-step limit of a nearest-voxel
midpoint rule written here in numpy."""
import math

import numpy as np
import pytest

import oracle
from test_oracle_pins import np_ray, tiny_workload


def brute_force_li(w, phi, i, j):
    """|ray /\\ voxel| for EVERY voxel by clipping the source->pixel segment against that voxel's own
    box (independent of any traversal order), summed per material."""
    S, d, L, t_in, t_out = np_ray(w, phi, i, j)
    nx, ny, nz = w.dims
    lo = np.array(w.centre) - 0.5 * np.array(w.dims) * np.array(w.spacing)
    li = np.zeros(w.n_materials)
    for iz in range(nz):
        for iy in range(ny):
            for ix in range(nx):
                a, b = 0.0, L
                for ax, idx in enumerate((ix, iy, iz)):
                    v0 = lo[ax] + idx * w.spacing[ax]
                    v1 = v0 + w.spacing[ax]
                    if d[ax] != 0.0:
                        t1, t2 = (v0 - S[ax]) / d[ax], (v1 - S[ax]) / d[ax]
                        a, b = max(a, min(t1, t2)), min(b, max(t1, t2))
                    elif not (v0 <= S[ax] < v1):
                        a, b = 1.0, 0.0
                if b > a:
                    li[w.mat[iz, iy, ix]] += float(w.rho[iz, iy, ix]) * (b - a)
    return li


def test_s1_brute_force_per_voxel_clipping():
    rng = np.random.default_rng(11)
    rho = rng.uniform(0.2, 2.0, size=(4, 5, 6)).astype(np.float32)
    mat = rng.integers(0, 3, size=rho.shape).astype(np.uint8)
    for phi_deg, spacing, centre in ((0.0, (2.0, 3.0, 2.5), (0, 0, 0)), (33.0, (2.0, 2.0, 2.0), (1.5, -2.0, 0.7)),
                                     (90.0, (1.0, 2.0, 3.0), (0, 0, 0)), (211.0, (2.5, 1.5, 2.0), (0, 0, 0))):
        # even detector dims: no ray lies IN a lattice plane (u = 0 or v = 0 with even voxel counts), where the
        # voxel a ray belongs to is a tie and either neighbour is a correct answer
        w = tiny_workload(rho, mat, spacing=spacing, n_materials=3, nu=8, nv=6, du=2.4, dv=2.9,
                          phis=(math.radians(phi_deg),), centre=centre, mu_hat=np.full((3, 1), 0.02))
        ref = oracle.project(w, method="siddon")
        for j in range(w.nv):
            for i in range(w.nu):
                bf = brute_force_li(w, w.phis[0], i, j)
                np.testing.assert_allclose(ref["line_integrals"][0, :, j, i], bf, rtol=1e-11, atol=1e-11)
    assert ref["line_integrals"].max() > 0


@pytest.mark.parametrize("phi_deg", [0.0, 17.0, 45.0, 90.0, 180.0, 263.0])
def test_s2_uniform_volume_is_rho_times_chord(phi_deg):
    rho = np.full((10, 12, 14), 1.3, dtype=np.float32)
    w = tiny_workload(rho, spacing=(2.0, 1.5, 2.5), nu=20, nv=16, phis=(math.radians(phi_deg),))
    ref = oracle.project(w, method="siddon")
    hits = 0
    for j in range(w.nv):
        for i in range(w.nu):
            S, d, L, t_in, t_out = np_ray(w, w.phis[0], i, j)
            chord = max(t_out - t_in, 0.0)
            assert abs(ref["line_integrals"][0, 0, j, i] - float(np.float32(1.3)) * chord) <= 1e-10 * (1 + chord)
            hits += chord > 0
    assert hits > 50


def test_s3_axis_parallel_rows_and_segment_count():
    """The central ray at phi = 0 runs along +x through one row of voxels: LI = dx * sum of that row."""
    rng = np.random.default_rng(5)
    rho = rng.uniform(0.5, 1.5, size=(5, 7, 9)).astype(np.float32)
    w = tiny_workload(rho, spacing=(2.0, 2.0, 2.0), nu=1, nv=1, du=1.0, dv=1.0, phis=(0.0, math.pi / 2))
    # one pixel at u = v = 0: the ray is the x axis (phi = 0) or the y axis (phi = 90), through the
    # centre voxel row (odd dims, so it runs through voxel centres, away from any lattice plane)
    ref = oracle.project(w, method="siddon")
    assert abs(ref["line_integrals"][0, 0, 0, 0] - 2.0 * float(rho[2, 3, :].astype(np.float64).sum())) < 1e-10
    assert abs(ref["line_integrals"][1, 0, 0, 0] - 2.0 * float(rho[2, :, 4].astype(np.float64).sum())) < 1e-9
    assert ref["n_segments"][0, 0, 0] == 9 and ref["n_segments"][1, 0, 0] == 7


def test_s4_fine_step_limit_of_a_nearest_voxel_midpoint_rule():
    """Siddon's sum is the exact integral of the piecewise-constant field; a midpoint rule on the
    NEAREST-voxel field with a tiny step converges to it (error <= step * jumps)."""
    rng = np.random.default_rng(2)
    rho = rng.uniform(0.0, 2.0, size=(6, 6, 6)).astype(np.float32)
    w = tiny_workload(rho, spacing=(2.0, 2.0, 2.0), nu=5, nv=5, du=2.0, dv=2.0, phis=(math.radians(28.0),))
    ref = oracle.project(w, method="siddon")
    lo = -0.5 * np.array(w.dims) * np.array(w.spacing)
    h = 1e-3
    for j in range(w.nv):
        for i in range(w.nu):
            S, d, L, t_in, t_out = np_ray(w, w.phis[0], i, j)
            if t_out <= t_in:
                assert ref["line_integrals"][0, 0, j, i] == 0.0
                continue
            n = int(round((t_out - t_in) / h))
            t = t_in + (np.arange(n) + 0.5) * ((t_out - t_in) / n)
            x = S[None, :] + t[:, None] * d[None, :]
            idx = np.clip(np.floor((x - lo) / np.array(w.spacing)).astype(int), 0, np.array(w.dims) - 1)
            approx = float(rho[idx[:, 2], idx[:, 1], idx[:, 0]].astype(np.float64).sum()) * ((t_out - t_in) / n)
            assert abs(approx - ref["line_integrals"][0, 0, j, i]) < 2.0 * h * 40


def test_s5_sphere_chord_and_beer_lambert():
    n, vox, R = 48, 1.0, 18.0
    c = (np.arange(n) - (n - 1) / 2) * vox
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    rho = (X * X + Y * Y + Z * Z <= R * R).astype(np.float32) * 1.1
    w = tiny_workload(rho, spacing=(vox,) * 3, nu=33, nv=3, du=1.5, dv=1.5, phis=(math.radians(40.0),),
                      mu_hat=np.array([[0.03]]))
    ref = oracle.project(w, method="siddon")
    for i in range(w.nu):
        S, d, L, t_in, t_out = np_ray(w, w.phis[0], i, 1)
        b = np.linalg.norm(np.cross(-S, d))                      # impact parameter of the ray
        if b < 0.8 * R:
            assert abs(ref["line_integrals"][0, 0, 1, i] - 1.1 * 2 * math.sqrt(R * R - b * b)) < 1.1 * 1.5 * vox + 1e-5
    # mono-energetic: P = exp(-mu_hat * LI)   (Eq. (1) with one channel, phi = R = 1)
    np.testing.assert_allclose(-np.log(ref["signal"][0]) / 0.03, ref["line_integrals"][0, 0], rtol=1e-12, atol=1e-12)


def test_s6_material_routing_sums_to_the_unsegmented_volume(workloads_cache):
    w = workloads_cache("C1")
    pix = np.array([[0, i, j] for j in range(8, w.nv, 37) for i in range(5, w.nu, 41)], dtype=np.int32)
    seg = oracle.project(w, pixels=pix, method="siddon")
    one = tiny_workload(w.rho, None, spacing=w.spacing, nu=w.nu, nv=w.nv, du=w.du, dv=w.dv, phis=w.phis,
                        step=w.step_mm, sad=w.sad, sdd=w.sdd)
    tot = oracle.project(one, pixels=pix, method="siddon")
    np.testing.assert_allclose(seg["line_integrals"].sum(axis=1), tot["line_integrals"][:, 0], rtol=1e-12)
    assert (seg["line_integrals"][:, 1] > 0).any()               # bone is crossed somewhere


def test_siddon_golden_regression(workloads_cache):
    """tests/golden/oracle_siddon_regression.txt (written by tests/golden/make_golden.py, which calls only oracle/):
    a guard against accidental changes of the oracle's arithmetic, not a pin."""
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "oracle_siddon_regression.txt")
    rows = [l.split() for l in open(path) if not l.startswith("#")]
    assert len(rows) == 10
    for row in rows:
        w = workloads_cache(row[0])
        p, i, j, nseg = map(int, row[1:5])
        out = oracle.project(w, pixels=np.array([[p, i, j]]), method="siddon")
        assert int(out["n_segments"][0]) == nseg
        assert out["signal"][0] == pytest.approx(float(row[5]), rel=1e-13)
        assert np.allclose(out["line_integrals"][0], [float(x) for x in row[6:]], rtol=1e-13, atol=1e-13)
