"""Source/detector trajectories as pose tables (inputs only).

A pose is what the user of a general-geometry projector supplies per projection:
the source position S, the detector origin P (where pixel coordinates (u, v) =
(0, 0) sit), and the detector's in-plane unit vectors u_hat, v_hat -- 12 doubles,
world coordinates, mm.  How rays are formed from a pose (pixel centre, clipping,
sampling) is the projector's business and is NOT here.

PAPER.md:93-95 defines the circular gantry; PAPER.md:405 says other scanner
geometries need "simple modifications".  The trajectories below are the usual
ones: the circle itself (for cross-checks), a helix (the gantry circle with a
table feed along z), a C-arm orbit (the circle's plane tilted about the x
axis), and seeded free poses.
"""
import numpy as np

from .prng import SplitMix64


def _rot_x(alpha):
    c, s = np.cos(alpha), np.sin(alpha)
    return np.array([[1.0, 0.0, 0.0], [0.0, c, -s], [0.0, s, c]])


def circular_poses(sad, sdd, theta, phis):
    """The gantry of PAPER.md:93-95 as poses: S = -SAD (cos phi, sin phi, 0),
    P = (SDD - SAD)(cos psi, sin psi, 0), u_hat = (-sin psi, cos psi, 0), v_hat = +z,
    psi = phi + theta."""
    phis = np.asarray(phis, dtype=np.float64)
    psi = phis + theta
    aid = sdd - sad
    out = np.zeros((phis.shape[0], 12))
    out[:, 0] = -(sad * np.cos(phis))
    out[:, 1] = -(sad * np.sin(phis))
    out[:, 3] = aid * np.cos(psi)
    out[:, 4] = aid * np.sin(psi)
    out[:, 6] = -np.sin(psi)
    out[:, 7] = np.cos(psi)
    out[:, 11] = 1.0
    return out


def helical_poses(sad, sdd, phis, pitch_mm, z0_mm=0.0):
    """Helix: the circular gantry whose source and detector move along z by
    pitch_mm per turn, z = z0 + pitch * phi / (2 pi)."""
    out = circular_poses(sad, sdd, 0.0, phis)
    z = z0_mm + pitch_mm * np.asarray(phis, dtype=np.float64) / (2.0 * np.pi)
    out[:, 2] += z
    out[:, 5] += z
    return out


def c_arm_poses(sad, sdd, phis, tilt_rad):
    """C-arm orbit: the circular gantry's plane tilted about the world x axis by
    tilt_rad (cranio-caudal angulation); the detector frame tilts with it."""
    out = circular_poses(sad, sdd, 0.0, phis)
    R = _rot_x(tilt_rad)
    for k in range(4):
        out[:, 3 * k:3 * k + 3] = out[:, 3 * k:3 * k + 3] @ R.T
    return out


def free_poses(n, sad, sdd, seed):
    """Seeded free poses: source on the sphere of radius sad in a random direction,
    detector origin opposite at sdd - sad, detector frame rotated in its plane."""
    rng = SplitMix64(seed)
    out = np.zeros((n, 12))
    for p in range(n):
        z = rng.uniform(-0.6, 0.6)
        a = rng.uniform(0.0, 2.0 * np.pi)
        r = np.sqrt(1.0 - z * z)
        nrm = np.array([r * np.cos(a), r * np.sin(a), z])          # source -> detector direction
        helper = np.array([0.0, 0.0, 1.0])
        e1 = np.cross(helper, nrm)
        e1 /= np.linalg.norm(e1)
        e2 = np.cross(nrm, e1)
        roll = rng.uniform(0.0, 2.0 * np.pi)
        out[p, 0:3] = -sad * nrm
        out[p, 3:6] = (sdd - sad) * nrm
        out[p, 6:9] = np.cos(roll) * e1 + np.sin(roll) * e2
        out[p, 9:12] = -np.sin(roll) * e1 + np.cos(roll) * e2
    return out
