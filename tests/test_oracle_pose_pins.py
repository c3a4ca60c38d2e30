"""Pins of the oracle's general-pose path (helical / C-arm source paths, SURVEY.md NEXT-4,
PAPER.md:405 "with simple modifications"; reading Q31) against things other than itself:

  G1  poses of the circular gantry built here from PAPER.md:93-95 give the circular oracle's integer
      ray table bit for bit and its signal exactly (the circular path carries pins P1-P10)
  G2  a helix is the circle seen from a shifted table: pose shifted by z == volume centre shifted by -z
  G3  a C-arm orbit tilted 90 degrees about x == the untilted orbit on the volume with y and z exchanged
  G4  Siddon through a uniform box == rho x the chord of the box, the chord clipped here in numpy, free poses
  G5  a small ball shadows where the line source->ball meets the detector plane (ray-plane intersection
      done here), free poses: pins P, u_hat, v_hat and the pixel indexing
  G6  flipping u_hat mirrors the image in u; rolling the frame by 90 degrees turns a square image
"""
import math

import numpy as np
import pytest

import oracle
from workloads import trajectories
from test_oracle_pins import tiny_workload


def _phantom(n=(20, 18, 16), seed=5):
    rng = np.random.default_rng(seed)
    nx, ny, nz = n
    rho = rng.uniform(0.2, 1.6, size=(nz, ny, nx)).astype(np.float32)
    mat = rng.integers(0, 2, size=(nz, ny, nx)).astype(np.uint8)
    return rho, mat


def _gantry_poses(sad, sdd, theta, phis):
    """PAPER.md:93-95 written out here (not taken from the oracle or workloads.trajectories)."""
    out = []
    for phi in phis:
        psi = phi + theta
        aid = sdd - sad
        out.append([-(sad * math.cos(phi)), -(sad * math.sin(phi)), 0.0,
                    aid * math.cos(psi), aid * math.sin(psi), 0.0,
                    -math.sin(psi), math.cos(psi), 0.0,
                    0.0, 0.0, 1.0])
    return np.array(out)


@pytest.mark.parametrize("method", ["trilinear", "siddon"])
def test_g1_circular_gantry_as_poses_is_bit_identical(method):
    rho, mat = _phantom()
    phis = np.radians([0.0, 17.0, 90.0, 133.0, 270.0])
    kw = dict(spacing=(2.0, 2.2, 2.5), n_materials=2, nu=25, nv=21, du=3.0, dv=3.3, step=0.7,
              mu_hat=[[0.02], [0.05]])
    for theta, u_off in ((0.0, 0.0), (math.radians(7.0), 11.5)):
        w = tiny_workload(rho, mat, phis=phis, theta=theta, **kw)
        w.u_off, w.v_off = u_off, -0.4 * u_off
        a = oracle.project(w, method=method)
        b = oracle.project(w.with_poses(_gantry_poses(w.sad, w.sdd, theta, phis)), method=method)
        assert np.array_equal(a["ray_table"], b["ray_table"])
        assert np.array_equal(a["signal"], b["signal"])
        assert np.array_equal(a["line_integrals"], b["line_integrals"])
        # and the trajectory generator the GPU tests use says the same thing
        t = trajectories.circular_poses(w.sad, w.sdd, theta, phis)
        assert np.array_equal(oracle.project(w.with_poses(t), method=method)["ray_table"], a["ray_table"])


def test_g2_helix_is_the_circle_with_the_table_shifted():
    rho, mat = _phantom((22, 22, 30))
    phis = np.radians([10.0, 100.0, 200.0, 300.0])
    pitch = 40.0
    w = tiny_workload(rho, mat, phis=phis, spacing=(2.0, 2.0, 2.0), n_materials=2, nu=24, nv=30,
                      du=3.0, dv=3.0, mu_hat=[[0.02], [0.04]])
    hel = oracle.project(w.with_poses(trajectories.helical_poses(w.sad, w.sdd, phis, pitch, z0_mm=-9.0)))
    for p, phi in enumerate(phis):
        z = -9.0 + pitch * phi / (2 * math.pi)
        ws = tiny_workload(rho, mat, phis=[phi], spacing=(2.0, 2.0, 2.0), n_materials=2, nu=24, nv=30,
                           du=3.0, dv=3.0, mu_hat=[[0.02], [0.04]], centre=(0.0, 0.0, -z))
        ref = oracle.project(ws)
        assert np.allclose(hel["line_integrals"][p], ref["line_integrals"][0], rtol=1e-9, atol=1e-9)
        assert np.allclose(hel["signal"][p], ref["signal"][0], rtol=1e-10)
    # the shift matters: projections at different z differ
    assert np.max(np.abs(hel["line_integrals"][0] - hel["line_integrals"][3])) > 1.0


@pytest.mark.parametrize("method", ["trilinear", "siddon"])
def test_g3_c_arm_tilted_90_degrees_is_an_axis_exchange(method):
    """R = rotation by +90 deg about x: (x, y, z) -> (x, -z, y).  Projecting f on the poses R*pose equals
    projecting f'(x) = f(R x) on the untilted poses; on the lattice f'[k][j][i] = f[j][ny-1-k][i]."""
    rho, mat = _phantom((20, 16, 24))
    phis = np.radians([0.0, 35.0, 120.0, 251.0])
    common = dict(n_materials=2, nu=24, nv=22, du=3.0, dv=3.0, mu_hat=[[0.02], [0.04]], step=0.6)
    w = tiny_workload(rho, mat, phis=phis, spacing=(2.0, 2.5, 1.5), **common)
    tilted = oracle.project(w.with_poses(trajectories.c_arm_poses(w.sad, w.sdd, phis, math.pi / 2)),
                            method=method)
    rho2 = np.ascontiguousarray(rho.transpose(1, 0, 2)[::-1])
    mat2 = np.ascontiguousarray(mat.transpose(1, 0, 2)[::-1])
    w2 = tiny_workload(rho2, mat2, phis=phis, spacing=(2.0, 1.5, 2.5), **common)
    ref = oracle.project(w2, method=method)
    scale = np.max(ref["line_integrals"])
    assert np.max(np.abs(tilted["line_integrals"] - ref["line_integrals"])) < 1e-9 * scale
    assert np.allclose(tilted["signal"], ref["signal"], rtol=1e-10)
    assert scale > 10.0


def _clip_chord(S, D, lo, hi):
    """Length of the segment S->D inside the box [lo, hi] (numpy, independent of the oracle)."""
    d = D - S
    t0, t1 = 0.0, 1.0
    for a in range(3):
        if d[a] == 0.0:
            if not (lo[a] <= S[a] <= hi[a]):
                return 0.0
            continue
        ta, tb = (lo[a] - S[a]) / d[a], (hi[a] - S[a]) / d[a]
        t0, t1 = max(t0, min(ta, tb)), min(t1, max(ta, tb))
    return max(t1 - t0, 0.0) * float(np.linalg.norm(d))


def test_g4_uniform_box_chord_on_free_poses():
    n, sp = (18, 14, 10), (2.0, 3.0, 2.5)
    rho = np.full((n[2], n[1], n[0]), 1.25, dtype=np.float32)
    poses = trajectories.free_poses(6, 400.0, 700.0, seed=77)
    w = tiny_workload(rho, spacing=sp, nu=20, nv=16, du=4.0, dv=4.0, step=0.5, sad=400.0, sdd=700.0)
    w = w.with_poses(poses)
    w.u_off, w.v_off = 3.0, -2.0
    sid = oracle.project(w, method="siddon")["line_integrals"][:, 0]
    tri = oracle.project(w, method="trilinear")["line_integrals"][:, 0]
    half = 0.5 * np.array(n) * np.array(sp)
    n_hit = 0
    for p in range(6):
        S, P, uh, vh = poses[p, 0:3], poses[p, 3:6], poses[p, 6:9], poses[p, 9:12]
        for j in range(w.nv):
            for i in range(w.nu):
                u = (i - (w.nu - 1) / 2) * w.du + w.u_off
                v = (j - (w.nv - 1) / 2) * w.dv + w.v_off
                chord = _clip_chord(S, P + u * uh + v * vh, -half, half)
                assert sid[p, j, i] == pytest.approx(1.25 * chord, abs=1e-9)
                assert abs(tri[p, j, i] - 1.25 * chord) <= 1.25 * w.step_mm + 1e-9   # midpoint count: +-1 step
                n_hit += chord > 0
    assert n_hit > 600


def test_g5_ball_shadow_on_free_poses():
    nvox, vox = 48, 2.0
    ball = np.array([14.0, -9.0, 11.0])
    ax = (np.arange(nvox) - (nvox - 1) / 2) * vox
    z, y, x = np.meshgrid(ax, ax, ax, indexing="ij")
    rho = np.where((x - ball[0]) ** 2 + (y - ball[1]) ** 2 + (z - ball[2]) ** 2 <= 25.0, 5.0, 0.0)
    poses = trajectories.free_poses(5, 500.0, 800.0, seed=3)
    w = tiny_workload(rho, spacing=(vox,) * 3, nu=72, nv=64, du=2.0, dv=2.0, sad=500.0, sdd=800.0)
    w = w.with_poses(poses)
    w.u_off, w.v_off = 4.0, -6.0
    li = oracle.project(w)["line_integrals"][:, 0]
    us = (np.arange(w.nu) - (w.nu - 1) / 2) * w.du + w.u_off
    vs = (np.arange(w.nv) - (w.nv - 1) / 2) * w.dv + w.v_off
    for p in range(5):
        S, P, uh, vh = poses[p, 0:3], poses[p, 3:6], poses[p, 6:9], poses[p, 9:12]
        nrm = np.cross(uh, vh)
        s_hit = np.dot(P - S, nrm) / np.dot(ball - S, nrm)
        H = S + s_hit * (ball - S)
        u_want, v_want = np.dot(H - P, uh), np.dot(H - P, vh)
        assert abs(u_want) < 60 and abs(v_want) < 50 and (abs(u_want) > 4 or abs(v_want) > 4)
        tot = li[p].sum()
        assert tot > 0
        assert (li[p].sum(axis=0) * us).sum() / tot == pytest.approx(u_want, abs=w.du)
        assert (li[p].sum(axis=1) * vs).sum() / tot == pytest.approx(v_want, abs=w.dv)


def test_g6_detector_frame_flip_and_roll():
    rho, mat = _phantom((20, 20, 20), seed=9)
    poses = trajectories.c_arm_poses(1000.0, 1500.0, np.radians([40.0, 200.0]), math.radians(25.0))
    w = tiny_workload(rho, mat, spacing=(2.0, 2.0, 2.0), n_materials=2, nu=22, nv=22, du=3.0, dv=3.0,
                      mu_hat=[[0.02], [0.04]])
    base = oracle.project(w.with_poses(poses))["line_integrals"]
    flip = poses.copy()
    flip[:, 6:9] *= -1.0
    got = oracle.project(w.with_poses(flip))["line_integrals"]
    assert np.allclose(got, base[..., ::-1], rtol=1e-10, atol=1e-10)
    roll = poses.copy()
    roll[:, 6:9], roll[:, 9:12] = poses[:, 9:12], -poses[:, 6:9]       # u' = v, v' = -u
    got = oracle.project(w.with_poses(roll))["line_integrals"]
    # pixel (i', j') of the rolled frame sits at u = -v' , v = u'  ->  (i, j) = (nv-1-j', i')
    want = base.transpose(0, 1, 3, 2)[..., ::-1, :]
    assert np.allclose(got, want, rtol=1e-10, atol=1e-10)
    assert np.max(np.abs(base - base[..., ::-1])) > 0.1


def test_pose_ray_geometry_matches_a_direct_construction():
    rho = np.ones((8, 8, 8), dtype=np.float32)
    w = tiny_workload(rho, spacing=(3.0, 3.0, 3.0), nu=10, nv=8, du=5.0, dv=6.0)
    w.u_off, w.v_off = 1.5, -2.5
    pose = trajectories.free_poses(1, 300.0, 500.0, seed=11)[0]
    r = oracle.ray_pose(w, pose, 7, 2)
    u = (7 - 4.5) * 5.0 + 1.5
    v = (2 - 3.5) * 6.0 - 2.5
    D = pose[3:6] + u * pose[6:9] + v * pose[9:12]
    d = D - pose[0:3]
    assert np.allclose(r["S"], pose[0:3])
    assert r["L"] == pytest.approx(np.linalg.norm(d), rel=1e-14)
    assert np.allclose(r["dir"], d / np.linalg.norm(d), atol=1e-14)


def test_trajectory_generators_give_orthonormal_frames_at_the_stated_distances():
    phis = np.radians([0.0, 33.0, 180.0, 311.0])
    for poses in (trajectories.circular_poses(1000.0, 1500.0, 0.0, phis),
                  trajectories.helical_poses(1000.0, 1500.0, phis, 40.0, z0_mm=-5.0),
                  trajectories.c_arm_poses(1000.0, 1500.0, phis, 0.4),
                  trajectories.free_poses(4, 1000.0, 1500.0, seed=1)):
        S, P, uh, vh = poses[:, 0:3], poses[:, 3:6], poses[:, 6:9], poses[:, 9:12]
        assert np.allclose(np.linalg.norm(uh, axis=1), 1.0, atol=1e-12)
        assert np.allclose(np.linalg.norm(vh, axis=1), 1.0, atol=1e-12)
        assert np.allclose(np.sum(uh * vh, axis=1), 0.0, atol=1e-12)
        nrm = np.cross(uh, vh)
        # source-to-detector distance along the detector normal is SDD
        assert np.allclose(np.abs(np.sum((P - S) * nrm, axis=1)), 1500.0, rtol=1e-12)


def test_pose_that_looks_away_from_the_volume_gives_the_flat_field():
    rho = np.ones((8, 8, 8), dtype=np.float32)
    w = tiny_workload(rho, spacing=(2.0, 2.0, 2.0), nu=6, nv=5, du=4.0, dv=4.0, sad=300.0, sdd=500.0)
    pose = trajectories.circular_poses(300.0, 500.0, 0.0, [0.0])
    pose[0, 3] = -800.0                      # detector behind the source: every ray leaves the volume behind
    out = oracle.project(w.with_poses(pose))
    assert np.all(out["ray_table"][..., 1] == 0)
    assert np.all(out["line_integrals"] == 0.0)
    assert np.allclose(out["signal"], 1.0, rtol=1e-15)
