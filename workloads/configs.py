"""The five CBCT-shaped workloads C0..C4 of BASELINE.json, as seeded arrays.

Naming follows SURVEY.md section 0: C0 tiny mono, C1 small poly, C2 clinical single
projection, C3 full scan, C4 high-resolution scan.  Everything is drawn from
one SplitMix64 stream per config (seed = 12046367 + 1000*index), in the order
the code below consumes it.  Units: mm, g/cm^3, keV; mu_hat in mm^-1 per g/cm^3.

Array conventions: rho[iz][iy][ix], x fastest; the volume is
centred on the isocentre O; voxel (ix,iy,iz) has its centre at
((ix,iy,iz) - (N-1)/2) * spacing.
"""
from dataclasses import dataclass, field
import hashlib
import math
from typing import Optional

import numpy as np

from . import curves
from .prng import SplitMix64

WORKLOAD_NAMES = ("C0", "C1", "C2", "C3", "C4")
BASE_SEED = 12046367
TEXTURE_AMPLITUDE = 0.015          # +-1.5 % smooth density modulation in tissue
TEXTURE_PERIOD_MM = (37.0, 29.0, 41.0)
SEGMENT_THRESHOLDS = (0.2, 0.98, 1.15)   # air | adipose | soft | bone


@dataclass
class Workload:
    name: str
    # volume
    rho: np.ndarray                 # float32 [nz][ny][nx]
    mat: np.ndarray                 # uint8   [nz][ny][nx], values < n_materials
    spacing: tuple                  # (dx, dy, dz) mm
    n_materials: int
    # geometry
    sad: float
    sdd: float
    theta: float
    nu: int
    nv: int
    du: float
    dv: float
    u_off: float
    v_off: float
    phis: np.ndarray                # float64 [n_proj], radians
    step_mm: float
    # source / detector tables
    energies: np.ndarray            # float64 [n_energy], keV (bin centres)
    phi_weight: np.ndarray          # float64 [n_energy], sums to 1
    response: np.ndarray            # float64 [n_energy]
    mu_hat: np.ndarray              # float64 [n_materials][n_energy]
    fluence_map: Optional[np.ndarray] = None   # float32 [nv][nu] or None (= 1)
    bowtie_mu: Optional[np.ndarray] = None     # float64 [n_energy] or None
    bowtie_thickness: Optional[np.ndarray] = None  # float64 [nu] or None
    centre: tuple = (0.0, 0.0, 0.0)
    notes: dict = field(default_factory=dict)
    # general source path (helical, C-arm): float64 [n_proj][12] = per projection source S, detector
    # origin P, u_hat, v_hat (world, mm); None = the circular gantry (sad, sdd, theta, phis)
    poses: Optional[np.ndarray] = None
    # pixel-dependent detector response ("could also be pixel dependent"; reading Q32):
    # float32 [n_energy][nv][nu] gain g(E, u), the pixel's response is response[E] * g; None = 1
    response_gain: Optional[np.ndarray] = None

    @property
    def dims(self):
        nz, ny, nx = self.rho.shape
        return nx, ny, nz

    @property
    def n_proj(self):
        return int(self.phis.shape[0] if self.poses is None else self.poses.shape[0])

    @property
    def n_energy(self):
        return int(self.energies.shape[0])

    def with_phis(self, phis):
        """Same inputs, other projection angles (radians)."""
        import copy
        w = copy.copy(self)
        w.phis = np.ascontiguousarray(np.asarray(phis, dtype=np.float64))
        return w

    def with_poses(self, poses):
        """Same inputs on a general source path: poses [n_proj][12] (see workloads/trajectories.py)."""
        import copy
        w = copy.copy(self)
        w.poses = np.ascontiguousarray(np.asarray(poses, dtype=np.float64)).reshape(-1, 12)
        return w

    def sha256(self):
        h = hashlib.sha256()
        for a in (self.rho, self.mat, self.phis, self.phi_weight, self.response,
                  self.mu_hat):
            h.update(np.ascontiguousarray(a).tobytes())
        return h.hexdigest()


# --------------------------------------------------------------------------
# phantom painting (inputs only)
# --------------------------------------------------------------------------

def _axes(n, d):
    return (np.arange(n, dtype=np.float64) - 0.5 * (n - 1)) * d


def _paint_ellipsoid(rho, spacing, centre, semi, value, mask=None, matarr=None,
                     matval=None):
    """rho[...] = value at voxels whose centre lies inside the ellipsoid (and
    inside ``mask`` when given).  Works on the bounding box only."""
    nz, ny, nx = rho.shape
    dims = (nx, ny, nz)
    sl = []
    grids = []
    for a in range(3):
        n, d = dims[a], spacing[a]
        lo = (centre[a] - semi[a]) / d + 0.5 * (n - 1)
        hi = (centre[a] + semi[a]) / d + 0.5 * (n - 1)
        i0 = max(0, int(math.floor(lo)))
        i1 = min(n, int(math.ceil(hi)) + 1)
        if i1 <= i0:
            return
        sl.append(slice(i0, i1))
        x = (np.arange(i0, i1, dtype=np.float64) - 0.5 * (n - 1)) * d
        grids.append(((x - centre[a]) / semi[a]) ** 2)
    gx, gy, gz = grids
    inside = (gz[:, None, None] + gy[None, :, None] + gx[None, None, :]) <= 1.0
    view = (sl[2], sl[1], sl[0])
    if mask is not None:
        inside &= mask[view]
    rho[view][inside] = value
    if matarr is not None:
        matarr[view][inside] = matval


def _elliptic_cylinder_mask(shape, spacing, a, b):
    nz, ny, nx = shape
    x = _axes(nx, spacing[0])
    y = _axes(ny, spacing[1])
    m2 = ((y[:, None] / b) ** 2 + (x[None, :] / a) ** 2) <= 1.0
    return np.broadcast_to(m2[None, :, :], shape)


def _texture(shape, spacing):
    nz, ny, nx = shape
    x = _axes(nx, spacing[0])
    y = _axes(ny, spacing[1])
    z = _axes(nz, spacing[2])
    px, py, pz = TEXTURE_PERIOD_MM
    sx = np.sin(2 * np.pi * x / px).astype(np.float32)
    cy = np.cos(2 * np.pi * y / py).astype(np.float32)
    cz = np.cos(2 * np.pi * z / pz).astype(np.float32)
    return (np.float32(1.0) + np.float32(TEXTURE_AMPLITUDE)
            * cz[:, None, None] * cy[None, :, None] * sx[None, None, :])


def _segment(rho):
    t0, t1, t2 = SEGMENT_THRESHOLDS
    mat = np.zeros(rho.shape, dtype=np.uint8)
    mat[rho >= np.float32(t0)] = 1
    mat[rho >= np.float32(t1)] = 2
    mat[rho >= np.float32(t2)] = 3
    return mat


# --------------------------------------------------------------------------
# the volumes
# --------------------------------------------------------------------------

def _volume_c0(rng):
    n, d = 32, 2.0
    spacing = (d, d, d)
    extent = n * d
    rho = np.zeros((n, n, n), dtype=np.float32)
    _paint_ellipsoid(rho, spacing, (0.0, 0.0, 0.0), (24.0, 24.0, 24.0), 1.0)
    for _ in range(3):
        c = tuple(-0.5 * extent + rng.u01() * extent for _ in range(3))
        s = tuple(rng.uniform(4.0, 12.0) for _ in range(3))
        val = 0.3 + 1.5 * rng.u01()
        _paint_ellipsoid(rho, spacing, c, s, val)
    mat = np.zeros_like(rho, dtype=np.uint8)
    return rho, mat, spacing, 1


def _volume_c1(rng):
    n, d = 128, 2.0
    spacing = (d, d, d)
    ext = (n * d, n * d, n * d)
    shape = (n, n, n)
    a_body, b_body = 0.42 * ext[0], 0.32 * ext[1]
    body = _elliptic_cylinder_mask(shape, spacing, a_body, b_body)
    rho = np.where(body, np.float32(1.0), np.float32(0.0)).astype(np.float32)
    mat = np.zeros(shape, dtype=np.uint8)
    for k in range(12):
        c = (rng.uniform(-0.6, 0.6) * a_body, rng.uniform(-0.6, 0.6) * b_body,
             rng.uniform(-0.4, 0.4) * ext[2])
        s = tuple(rng.uniform(0.04, 0.14) * ext[a] for a in range(3))
        if k < 8:
            val, m = rng.uniform(0.9, 1.1), 0
        else:
            val, m = rng.uniform(1.2, 1.9), 1
        _paint_ellipsoid(rho, spacing, c, s, val, mask=body, matarr=mat, matval=m)
    tex = _texture(shape, spacing)
    soft = body & (mat == 0)
    bone = mat == 1
    rho = rho * tex
    rho[soft] = np.clip(rho[soft], 0.9, 1.1)
    rho[bone] = np.clip(rho[bone], 1.2, 1.9)
    rho[~body] = 0.0
    return rho.astype(np.float32), mat, spacing, 2


PHANTOMS = ("smooth", "noisy1", "noisy3", "random")


def _volume_pelvis(rng, dims, spacing, phantom="smooth", seed=0):
    """Pelvis-like ellipsoid phantom, 4 materials by density thresholds
    (used for C2, C3, C4 scaled to the extent).

    phantom: "smooth" (the recipe of BASELINE.md: noise-free densities, so 98.8 % of C3's cells have 8 corners of
    one material); "noisy1" / "noisy3": the same densities times (1 + sigma z), z seeded unit Gaussian voxel
    noise, sigma = 1 % / 3 %, applied to tissue BEFORE the thresholds, as in a reconstructed CT whose voxel noise
    straddles the adipose / soft threshold; "random": the same densities with a material drawn uniformly per
    voxel (no spatial structure at all: the worst case for any scheme that exploits material coherence)."""
    nx, ny, nz = dims
    shape = (nz, ny, nx)
    X, Y, Z = nx * spacing[0], ny * spacing[1], nz * spacing[2]
    rho = np.full(shape, 0.0012, dtype=np.float32)
    body = _elliptic_cylinder_mask(shape, spacing, 0.40 * X, 0.28 * Y)
    rho[body] = rng.uniform(0.92, 0.96)
    inner = _elliptic_cylinder_mask(shape, spacing, 0.34 * X, 0.22 * Y)
    rho[inner] = rng.uniform(1.02, 1.07)
    inner = np.ascontiguousarray(inner)
    # femoral-head-like pair
    for sx in (-1.0, 1.0):
        c = (sx * 0.26 * X, rng.uniform(-0.03, 0.03) * Y, -0.15 * Z)
        r = 0.045 * X
        _paint_ellipsoid(rho, spacing, c, (r, r, 1.1 * r), rng.uniform(1.3, 1.9),
                         mask=inner)
    # iliac-wing-like pair
    for sx in (-1.0, 1.0):
        c = (sx * 0.20 * X, 0.03 * Y, 0.15 * Z)
        _paint_ellipsoid(rho, spacing, c, (0.09 * X, 0.03 * Y, 0.22 * Z),
                         rng.uniform(1.3, 1.9), mask=inner)
    # sacrum-like
    _paint_ellipsoid(rho, spacing, (0.0, -0.12 * Y, 0.10 * Z),
                     (0.07 * X, 0.06 * Y, 0.20 * Z), rng.uniform(1.3, 1.9),
                     mask=inner)
    # bowel gas
    c = (rng.uniform(-0.1, 0.1) * X, rng.uniform(0.0, 0.1) * Y,
         rng.uniform(-0.2, 0.2) * Z)
    _paint_ellipsoid(rho, spacing, c, (0.05 * X, 0.035 * Y, 0.06 * Z), 0.0012,
                     mask=inner)
    # further seeded inserts
    for k in range(10):
        c = (rng.uniform(-0.30, 0.30) * X, rng.uniform(-0.18, 0.18) * Y,
             rng.uniform(-0.45, 0.45) * Z)
        s = tuple(rng.uniform(0.02, 0.07) * e for e in (X, Y, Z))
        val = (rng.uniform(0.92, 0.96), rng.uniform(1.02, 1.07),
               rng.uniform(1.3, 1.9))[k % 3]
        _paint_ellipsoid(rho, spacing, c, s, val, mask=inner)
    tex = _texture(shape, spacing)
    tissue = rho > np.float32(0.2)
    np.multiply(rho, tex, out=rho, where=tissue)
    if phantom in ("noisy1", "noisy3"):
        sigma = np.float32(0.01 if phantom == "noisy1" else 0.03)
        gen = np.random.Generator(np.random.PCG64(seed))
        for z in range(nz):                             # slab by slab: no second volume-sized array
            noise = gen.standard_normal((ny, nx), dtype=np.float32)
            np.multiply(rho[z], np.float32(1.0) + sigma * noise, out=rho[z], where=tissue[z])
        np.maximum(rho, np.float32(0.0), out=rho)
    mat = _segment(rho)
    if phantom == "random":
        gen = np.random.Generator(np.random.PCG64(seed))
        mat = gen.integers(0, 4, size=shape, dtype=np.uint8)
    elif phantom not in PHANTOMS:
        raise ValueError(f"unknown phantom {phantom!r}")
    return rho, mat, spacing, 4


def with_tissue_classes(w, n_classes):
    """The same volume segmented into `n_classes` materials (5..8) instead of four: density edges at 0.2 (air), 0.98
    (fat), then tissue and bone split further.  The mass attenuation curves of the new classes are those of the class
    they were split from, scaled by a few per cent (a seeded stand-in: only the count of materials matters here)."""
    import copy
    if not 5 <= n_classes <= 8 or w.n_materials != 4:
        raise ValueError("with_tissue_classes: 5..8 classes of a four-material workload")
    edges_all = [0.2, 0.98, 1.03, 1.15, 1.35, 1.6, 1.75]           # 8 classes
    parent_all = [0, 1, 2, 2, 3, 3, 3, 3]
    keep = {5: [0, 1, 2, 3], 6: [0, 1, 2, 3, 4], 7: [0, 1, 2, 3, 4, 5], 8: [0, 1, 2, 3, 4, 5, 6]}[n_classes]
    edges = np.array([edges_all[k] for k in keep], dtype=np.float32)
    parents = [0] + [parent_all[k + 1] for k in keep]
    out = copy.copy(w)
    out.mat = np.digitize(w.rho, edges).astype(np.uint8)
    out.n_materials = n_classes
    rng = SplitMix64(BASE_SEED + 77 + n_classes)
    out.mu_hat = np.ascontiguousarray(np.stack([w.mu_hat[p] * rng.uniform(0.97, 1.03) for p in parents]))
    out.notes = dict(w.notes, tissue_classes=n_classes)
    return out


def pure_cell_fraction(mat):
    """Fraction of the (nx-1)(ny-1)(nz-1) cells of the voxel lattice whose 8 corner voxels have one material
    (an input statistic: the CUDA sampler's fast path needs such cells)."""
    m = mat
    same = np.ones(tuple(n - 1 for n in m.shape), dtype=bool)
    ref = m[:-1, :-1, :-1]
    for dz in (0, 1):
        for dy in (0, 1):
            for dx in (0, 1):
                if dz or dy or dx:
                    same &= m[dz:m.shape[0] - 1 + dz, dy:m.shape[1] - 1 + dy, dx:m.shape[2] - 1 + dx] == ref
    return float(same.mean())


# --------------------------------------------------------------------------
# spectra and tables
# --------------------------------------------------------------------------

def _draw_mu_hat(rng, energies, materials):
    rows = {}
    # soft and bone are always drawn first, in this order; adipose after them
    a, b = rng.uniform(0.0025, 0.0035), rng.uniform(0.0170, 0.0185)
    rows["soft"] = curves.mu_hat_curve(energies, a, b)
    a, b = rng.uniform(0.010, 0.016), rng.uniform(0.0165, 0.0180)
    rows["bone"] = curves.mu_hat_curve(energies, a, b)
    if "adipose" in materials:
        a, b = rng.uniform(0.0015, 0.0022), rng.uniform(0.0172, 0.0182)
        rows["adipose"] = curves.mu_hat_curve(energies, a, b)
    rows["air"] = rows["soft"]
    return np.ascontiguousarray(np.stack([rows[m] for m in materials]))


def _even_angles(n):
    return 2.0 * np.pi * np.arange(n, dtype=np.float64) / n


# --------------------------------------------------------------------------
# public entry
# --------------------------------------------------------------------------

def make_workload(name: str, n_proj: Optional[int] = None, phantom: str = "smooth") -> Workload:
    """Build workload ``name`` in {"C0".."C4"}.  ``n_proj`` overrides the number
    of evenly spaced projections (C3/C4 default to 360/656; C0..C2 to one at 0).
    ``phantom`` (C2..C4 only): see _volume_pelvis; "smooth" is the configuration of BASELINE.json."""
    if name not in WORKLOAD_NAMES:
        raise ValueError(f"unknown workload {name!r}")
    if phantom != "smooth" and name not in ("C2", "C3", "C4"):
        raise ValueError("phantom variants exist for C2, C3 and C4")
    idx = WORKLOAD_NAMES.index(name)
    rng = SplitMix64(BASE_SEED + 1000 * idx)
    sad, sdd = 1000.0, 1500.0
    if name == "C0":
        rho, mat, spacing, M = _volume_c0(rng)
        E = np.array([60.0])
        wl = Workload(name, rho, mat, spacing, M, sad, sdd, 0.0, 64, 48, 3.1, 3.1,
                      0.0, 0.0, _even_angles(n_proj or 1), 0.5, E,
                      np.array([1.0]), np.array([1.0]), np.array([[0.0206]]))
    elif name == "C1":
        rho, mat, spacing, M = _volume_c1(rng)
        E = 22.5 + 5.0 * np.arange(20, dtype=np.float64)
        mu_hat = _draw_mu_hat(rng, E, ("soft", "bone"))
        wl = Workload(name, rho, mat, spacing, M, sad, sdd, 0.0, 256, 192, 1.552,
                      1.552, 0.0, 0.0, _even_angles(n_proj or 1), 1.0, E,
                      curves.kramers_spectrum(E, 120.0), curves.response_linear(E),
                      mu_hat)
    else:
        if name == "C2":
            dims, spacing = (256, 256, 128), (1.95, 1.95, 2.5)
            nu, nv, dpix, step, default_np = 512, 384, 0.776, 0.975, 1
        elif name == "C3":
            dims, spacing = (512, 512, 256), (0.98, 0.98, 1.25)
            nu, nv, dpix, step, default_np = 512, 384, 0.776, 0.49, 360
        else:
            dims, spacing = (512, 512, 512), (0.5, 0.5, 0.5)
            nu, nv, dpix, step, default_np = 1024, 768, 0.388, 0.25, 656
        rho, mat, spacing, M = _volume_pelvis(rng, dims, spacing, phantom, BASE_SEED + 1000 * idx + 7)
        if name == "C4":
            E = 15.0 + (np.arange(120, dtype=np.float64) + 0.5) * 110.0 / 120.0
            e_max = 125.0
        else:
            E = 21.0 + np.arange(100, dtype=np.float64)
            e_max = 120.0
        mu_hat = _draw_mu_hat(rng, E, ("air", "adipose", "soft", "bone"))
        wl = Workload(name, rho, mat, spacing, M, sad, sdd, 0.0, nu, nv, dpix, dpix,
                      0.0, 0.0, _even_angles(n_proj or default_np), step, E,
                      curves.kramers_spectrum(E, e_max), curves.response_csi(E),
                      mu_hat, None, curves.mu_al(E),
                      curves.bowtie_thickness(nu, dpix))
    wl.rho = np.ascontiguousarray(wl.rho, dtype=np.float32)
    wl.mat = np.ascontiguousarray(wl.mat, dtype=np.uint8)
    wl.notes["seed"] = BASE_SEED + 1000 * idx
    wl.notes["phantom"] = phantom
    return wl


def shard_projections(n_proj: int, world_size: int, rank: int):
    """Contiguous block of projection indices owned by ``rank``: (begin, count).
    Projections are independent, so this is the whole
    multi-GPU story: no exchange step."""
    if not (0 <= rank < world_size):
        raise ValueError("rank out of range")
    base, rem = divmod(n_proj, world_size)
    begin = rank * base + min(rank, rem)
    return begin, base + (1 if rank < rem else 0)
