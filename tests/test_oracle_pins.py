"""Pins for the CPU oracle (oracle/gdrr_oracle.c) against things other than itself.

The paper prints no numeric value of P(u) or of a line integral,
so nothing can be pinned by a worked example.  These tests pin the oracle to
what the paper's model and the mathematics fix:
closed forms, invariants, special cases, an independent exact integrator
written here in numpy, and brute force on tiny inputs.  Each is chosen so that
a plausible slip (dropped term, wrong sign or index, transposed axis) fails.
"""
import math

import numpy as np
import pytest

import oracle
from workloads import Workload, make_workload

SQRT3 = math.sqrt(3.0)


# --------------------------------------------------------------------------
# helpers: tiny workloads and an INDEPENDENT numpy statement of the field
# --------------------------------------------------------------------------

def tiny_workload(rho, mat=None, spacing=(2.0, 2.0, 2.0), n_materials=1, nu=24, nv=20,
                  du=3.0, dv=3.0, phis=(0.0,), step=0.5, sad=1000.0, sdd=1500.0,
                  mu_hat=None, phi_weight=None, response=None, energies=None,
                  theta=0.0, centre=(0.0, 0.0, 0.0), **kw):
    rho = np.ascontiguousarray(rho, dtype=np.float32)
    if mat is None:
        mat = np.zeros(rho.shape, dtype=np.uint8)
    if energies is None:
        energies = np.array([60.0])
    ne = len(energies)
    if mu_hat is None:
        mu_hat = np.full((n_materials, ne), 0.02)
    if phi_weight is None:
        phi_weight = np.full(ne, 1.0 / ne)
    if response is None:
        response = np.ones(ne)
    return Workload("tiny", rho, np.ascontiguousarray(mat, dtype=np.uint8), tuple(spacing),
                    n_materials, sad, sdd, theta, nu, nv, du, dv, 0.0, 0.0,
                    np.asarray(phis, dtype=np.float64), step, np.asarray(energies, float),
                    np.asarray(phi_weight, float), np.asarray(response, float),
                    np.asarray(mu_hat, float), centre=tuple(centre), **kw)


def np_trilinear(rho, g):
    """Clamp-to-edge tri-linear interpolant, written independently of the C
    oracle: g = (gx, gy, gz) index coordinates."""
    nz, ny, nx = rho.shape
    val = 0.0
    base = [math.floor(c) for c in g]
    frac = [c - b for c, b in zip(g, base)]
    for qz in (0, 1):
        for qy in (0, 1):
            for qx in (0, 1):
                ix = min(max(base[0] + qx, 0), nx - 1)
                iy = min(max(base[1] + qy, 0), ny - 1)
                iz = min(max(base[2] + qz, 0), nz - 1)
                w = ((frac[0] if qx else 1 - frac[0]) * (frac[1] if qy else 1 - frac[1])
                     * (frac[2] if qz else 1 - frac[2]))
                val += w * float(rho[iz, iy, ix])
    return val


def np_ray(w, phi, i, j):
    """Source, unit direction and box chord [t_in, t_out] of pixel (i, j),
    written independently of the C oracle (numpy vectors, no shared order of
    operations): PAPER.md:93-95 with readings Q1-Q4."""
    psi = phi + w.theta
    S = np.array([-w.sad * math.cos(phi), -w.sad * math.sin(phi), 0.0])
    n_hat = np.array([math.cos(psi), math.sin(psi), 0.0])
    u_hat = np.cross([0.0, 0.0, 1.0], n_hat)
    u = (i - (w.nu - 1) / 2) * w.du + w.u_off
    v = (j - (w.nv - 1) / 2) * w.dv + w.v_off
    D = (w.sdd - w.sad) * n_hat + u * u_hat + v * np.array([0.0, 0.0, 1.0])
    L = np.linalg.norm(D - S)
    d = (D - S) / L
    n = np.array(w.dims, dtype=float)
    sp = np.array(w.spacing)
    c = np.array(w.centre)
    lo, hi = c - n * sp / 2, c + n * sp / 2
    t_in, t_out = 0.0, L
    for a in range(3):
        if d[a] != 0:
            t1, t2 = (lo[a] - S[a]) / d[a], (hi[a] - S[a]) / d[a]
            t_in, t_out = max(t_in, min(t1, t2)), min(t_out, max(t1, t2))
        elif S[a] < lo[a] or S[a] > hi[a]:
            return S, d, L, 0.0, 0.0
    return S, d, L, t_in, t_out


def exact_line_integral(w, phi, i, j):
    """Exact integral of the clamped tri-linear field of w.rho over the box
    chord: split at every t where an index coordinate crosses an integer; on
    each piece the field is a cubic in t, so 2-point Gauss-Legendre is exact
    (SURVEY.md 'O-exact')."""
    S, d, L, t_in, t_out = np_ray(w, phi, i, j)
    if t_out <= t_in:
        return 0.0
    n = np.array(w.dims, dtype=float)
    sp = np.array(w.spacing)
    c = np.array(w.centre)
    g_s = (S - c) / sp + (n - 1) / 2
    slope = d / sp
    cuts = [t_in, t_out]
    for a in range(3):
        if slope[a] == 0:
            continue
        ga, gb = g_s[a] + t_in * slope[a], g_s[a] + t_out * slope[a]
        for m in range(math.floor(min(ga, gb)), math.ceil(max(ga, gb)) + 1):
            t = (m - g_s[a]) / slope[a]
            if t_in < t < t_out:
                cuts.append(t)
    cuts = sorted(set(cuts))
    total = 0.0
    for ta, tb in zip(cuts[:-1], cuts[1:]):
        mid, half = 0.5 * (ta + tb), 0.5 * (tb - ta)
        for s in (-1.0, 1.0):
            t = mid + s * half / SQRT3
            total += half * np_trilinear(w.rho, g_s + t * slope)
    return total


def gaussian_blob_volume(n=16, seed=3):
    rng = np.random.default_rng(seed)
    z, y, x = np.meshgrid(*(np.arange(n, dtype=float),) * 3, indexing="ij")
    vol = np.zeros((n, n, n))
    for _ in range(4):
        c = rng.uniform(0.35 * n, 0.65 * n, size=3)
        s = rng.uniform(0.08 * n, 0.14 * n)
        vol += rng.uniform(0.5, 1.5) * np.exp(-((x - c[0]) ** 2 + (y - c[1]) ** 2
                                                + (z - c[2]) ** 2) / (2 * s * s))
    vol[:2], vol[-2:], vol[:, :2], vol[:, -2:], vol[:, :, :2], vol[:, :, -2:] = (0,) * 6
    return vol.astype(np.float32)


# --------------------------------------------------------------------------
# P1  empty volume: flat field (PAPER.md:147 with mu = 0; normalisation :121)
# --------------------------------------------------------------------------

def test_p1_empty_volume_flat_field():
    w = make_workload("C2")
    w.rho = np.zeros((8, 8, 8), dtype=np.float32)
    w.mat = np.zeros((8, 8, 8), dtype=np.uint8)
    rng = np.random.default_rng(0)
    w.fluence_map = rng.uniform(0.5, 1.5, size=(w.nv, w.nu)).astype(np.float32)
    pix = np.array([[0, i, j] for i in (0, 17, 255, 256, 511) for j in (0, 100, 383)])
    out = oracle.project(w, pixels=pix)
    for (p, i, j), got in zip(pix, out["signal"]):
        want = 0.0
        for e in range(w.n_energy):       # the separate 5-line loop of SURVEY P1
            want += (w.phi_weight[e] * float(w.fluence_map[j, i])
                     * math.exp(-w.bowtie_mu[e] * w.bowtie_thickness[i]) * w.response[e])
        assert got == pytest.approx(want, rel=1e-14)
    # w = 1, no bowtie, sum(phi) = 1, R = 1  =>  P = 1 everywhere
    w0 = make_workload("C0")
    w0.rho[:] = 0
    assert np.all(np.abs(oracle.project(w0)["signal"] - 1.0) < 1e-15)


# --------------------------------------------------------------------------
# P2  mono-energetic Beer-Lambert: -ln(P/(phi R))/mu_hat = LI
# --------------------------------------------------------------------------

def test_p2_monoenergetic_beer_lambert(workloads_cache):
    w = workloads_cache("C0")
    out = oracle.project(w)
    li = out["line_integrals"][0, 0]
    back = -np.log(out["signal"][0] / (w.phi_weight[0] * w.response[0])) / w.mu_hat[0, 0]
    assert np.max(np.abs(back - li)) < 1e-11
    assert li.max() > 40.0        # the sphere is really there (diameter 48 mm)


# --------------------------------------------------------------------------
# P3  uniform volume: LI = rho0 * n * dl exactly; |LI - rho0*chord| < rho0*dl
# --------------------------------------------------------------------------

@pytest.mark.parametrize("phi_deg", [0.0, 37.0, 90.0, 211.3])
def test_p3_uniform_volume_chord(phi_deg):
    rho0 = 1.37
    rho = np.full((10, 14, 12), rho0, dtype=np.float32)      # nz, ny, nx all different
    w = tiny_workload(rho, spacing=(2.0, 1.5, 2.5), phis=[math.radians(phi_deg)],
                      step=0.4, nu=32, nv=24, du=2.0, dv=2.0)
    out = oracle.project(w)
    li = out["line_integrals"][0, 0]
    tab = out["ray_table"][0]
    rho0f = float(np.float32(rho0))
    assert np.max(np.abs(li - rho0f * tab[..., 1] * w.step_mm)) < 1e-11
    n_hit = 0
    for j in range(w.nv):
        for i in range(w.nu):
            S, d, L, t_in, t_out = np_ray(w, w.phis[0], i, j)
            chord = max(t_out - t_in, 0.0)
            assert abs(li[j, i] - rho0f * chord) < rho0f * w.step_mm * (1 + 1e-9)
            n_hit += chord > 0
    assert n_hit > 100


# --------------------------------------------------------------------------
# P4  tri-affine reproduction;  P5  nodes and cell centres
# --------------------------------------------------------------------------

def test_p4_triaffine_reproduction():
    nx, ny, nz = 7, 6, 5
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")

    def f(x, y, z):
        return (0.5 + 0.25 * x) * (1.5 - 0.125 * y) * (0.75 + 0.5 * z)
    rho = f(x, y, z).astype(np.float32)      # exactly representable values
    rng = np.random.default_rng(1)
    pts = rng.uniform([0, 0, 0], [nx - 1, ny - 1, nz - 1], size=(500, 3))
    got = oracle.trilinear(rho, pts)
    want = f(pts[:, 0], pts[:, 1], pts[:, 2])
    assert np.max(np.abs(got - want)) < 1e-13
    # the axes are not interchangeable: a transposed index would fail here
    assert abs(f(1.5, 2.5, 3.5) - f(3.5, 2.5, 1.5)) > 0.1


def test_p5_nodes_cell_centres_and_clamp():
    rng = np.random.default_rng(2)
    rho = rng.uniform(0, 2, size=(4, 5, 6)).astype(np.float32)
    nodes = np.array([[x, y, z] for z in range(4) for y in range(5) for x in range(6)], float)
    assert np.array_equal(oracle.trilinear(rho, nodes), rho.astype(np.float64).ravel())
    centres = np.array([[x + .5, y + .5, z + .5] for z in range(3) for y in range(4)
                        for x in range(5)])
    want = [rho[z:z + 2, y:y + 2, x:x + 2].astype(np.float64).mean()
            for z in range(3) for y in range(4) for x in range(5)]
    assert np.max(np.abs(oracle.trilinear(rho, centres) - want)) < 1e-15
    # clamp-to-edge in the half-voxel shell (Q7): constant along the clamped axis
    assert oracle.trilinear(rho, [[-0.4, 2.0, 1.0]])[0] == pytest.approx(float(rho[1, 2, 0]), rel=1e-15)
    assert oracle.trilinear(rho, [[5.3, 2.0, 1.0]])[0] == pytest.approx(float(rho[1, 2, 5]), rel=1e-15)
    assert oracle.trilinear(rho, [[2.0, 4.45, 3.2]])[0] == pytest.approx(float(rho[3, 4, 2]), rel=1e-15)
    got = oracle.trilinear(rho, [[2.25, -0.3, 1.0]])[0]
    assert got == pytest.approx(0.75 * float(rho[1, 0, 2]) + 0.25 * float(rho[1, 0, 3]), rel=1e-15)
    # cross-check against the independent numpy statement on random points
    pts = rng.uniform([-0.5, -0.5, -0.5], [5.5, 4.5, 3.5], size=(300, 3))
    want = [np_trilinear(rho, p) for p in pts]
    assert np.max(np.abs(oracle.trilinear(rho, pts) - want)) < 1e-14


# --------------------------------------------------------------------------
# P6  exact tri-linear line integral and step-halving convergence
# --------------------------------------------------------------------------

def test_p6_exact_integrator_reproduces_box_chord():
    rho = np.full((6, 6, 6), 1.0, dtype=np.float32)
    w = tiny_workload(rho, phis=[math.radians(23.0)], nu=8, nv=8)
    for (i, j) in [(0, 7), (4, 2), (3, 3)]:
        S, d, L, t_in, t_out = np_ray(w, w.phis[0], i, j)
        assert exact_line_integral(w, w.phis[0], i, j) == pytest.approx(max(t_out - t_in, 0.0), abs=1e-10)
    assert t_out - t_in > 5.0


def test_p6_midpoint_rule_converges_to_exact_integral():
    rho = gaussian_blob_volume(16)
    phi = math.radians(31.0)
    pix = [(7, 6), (9, 10), (12, 8), (5, 9), (8, 8)]
    pixels = np.array([[0, i, j] for i, j in pix])
    base = tiny_workload(rho, phis=[phi], nu=16, nv=16, du=3.0, dv=3.0)
    exact = np.array([exact_line_integral(base, phi, i, j) for i, j in pix])
    assert exact.min() > 1.0
    errs = []
    for step in (1.0, 0.5, 0.25, 0.125, 0.0625, 0.001):
        li = oracle.project(base, pixels=pixels, step=step)["line_integrals"][:, 0]
        errs.append(np.max(np.abs(li - exact) / exact))
    assert errs[0] < 3e-2
    assert errs[3] < errs[0] / 16          # error(dl/8) < error(dl)/16  (~ O(dl^2))
    assert errs[4] < errs[1] / 16
    assert errs[5] < 1e-7                  # dl -> 0: the line integral itself
    # default step = half the smallest voxel edge (Q8)
    w_aniso = tiny_workload(rho, spacing=(2.0, 1.0, 3.0), phis=[phi], nu=16, nv=16)
    a = oracle.project(w_aniso, pixels=pixels, step=0.0)["ray_table"]
    b = oracle.project(w_aniso, pixels=pixels, step=0.5)["ray_table"]
    assert np.array_equal(a, b)


def test_p6_midpoints_are_laid_from_the_source():
    """Q9: interval k has midpoint (k + 1/2) dl measured from the SOURCE and
    counts iff t_in <= t_k < t_out: brute force over k."""
    rho = np.ones((8, 8, 8), dtype=np.float32)
    w = tiny_workload(rho, phis=[math.radians(12.0)], nu=12, nv=10, du=2.0, dv=2.0, step=0.37)
    for (i, j) in [(5, 5), (0, 0), (11, 4), (6, 9)]:
        r = oracle.ray(w, w.phis[0], i, j)
        S, d, L, t_in, t_out = np_ray(w, w.phis[0], i, j)
        ks = [k for k in range(0, int(L / w.step_mm) + 2)
              if t_in <= (k + 0.5) * w.step_mm < t_out]
        if ks:
            assert (r["j0"], r["n"]) == (ks[0], len(ks))
        else:
            assert r["n"] == 0
        assert r["t_in"] == pytest.approx(t_in, abs=1e-9)
        assert r["t_out"] == pytest.approx(t_out, abs=1e-9)


def test_p6_linear_ramp_midpoint_rule_is_exact():
    """For a field linear along the ray the midpoint rule is exact on
    [j0*dl, (j0+n)*dl]: LI = n*dl*f(centre of that range).  A sample placed at
    k*dl instead of (k+1/2)*dl ("midpoint of each interval")
    shifts the sum by dl/2 times the slope and fails this."""
    nz, ny, nx = 40, 8, 8
    a, b = 0.5, 0.0625                                   # rho = a + b*iz, exact in fp32
    rho = np.broadcast_to((a + b * np.arange(nz))[:, None, None], (nz, ny, nx)).astype(np.float32)
    w = tiny_workload(rho, spacing=(2.0, 2.0, 2.0), phis=[math.radians(40.0)], nu=6, nv=40,
                      du=1.0, dv=2.0, step=0.5)
    out = oracle.project(w)
    li, tab = out["line_integrals"][0, 0], out["ray_table"][0]
    checked = 0
    for j in range(w.nv):
        for i in range(w.nu):
            S, d, L, t_in, t_out = np_ray(w, w.phis[0], i, j)
            j0, n = tab[j, i]
            if n == 0:
                continue
            t_a, t_b = j0 * w.step_mm, (j0 + n) * w.step_mm
            gz = lambda t: (S[2] + t * d[2]) / w.spacing[2] + (nz - 1) / 2
            if min(gz(t_a), gz(t_b)) < 0 or max(gz(t_a), gz(t_b)) > nz - 1:
                continue                                  # touches the clamped shell in z
            want = (t_b - t_a) * (a + b * gz(0.5 * (t_a + t_b)))
            assert li[j, i] == pytest.approx(want, abs=1e-10)
            shift = 0.5 * w.step_mm * (t_b - t_a) * b * abs(d[2]) / w.spacing[2]
            checked += shift > 1e-5                       # the wrong rule would be visible
    assert checked > 100


# --------------------------------------------------------------------------
# P7  homogeneous sphere: LI ~ rho0 * 2 sqrt(R^2 - b^2)
# --------------------------------------------------------------------------

def _sphere_errors(n, vox, R, rho0):
    ax = (np.arange(n) - (n - 1) / 2) * vox
    z, y, x = np.meshgrid(ax, ax, ax, indexing="ij")
    rho = np.where(x * x + y * y + z * z <= R * R, rho0, 0.0).astype(np.float32)
    w = tiny_workload(rho, spacing=(vox,) * 3, phis=[math.radians(17.0)], nu=40, nv=40,
                      du=2.4, dv=2.4, step=0.5 * vox)
    li = oracle.project(w)["line_integrals"][0, 0]
    errs = []
    for j in range(w.nv):
        for i in range(w.nu):
            S, d, L, _, _ = np_ray(w, w.phis[0], i, j)
            b = np.linalg.norm(np.cross(-S, d))          # impact parameter wrt O
            if b < 0.8 * R:
                errs.append(li[j, i] - rho0 * 2 * math.sqrt(R * R - b * b))
    return np.abs(np.array(errs))


def test_p7_sphere_chord():
    R, rho0 = 24.0, 1.0
    e_coarse = _sphere_errors(32, 2.0, R, rho0)
    e_fine = _sphere_errors(64, 1.0, R, rho0)
    assert len(e_coarse) > 300
    assert e_coarse.max() < 2.0 * rho0            # within one 2 mm voxel
    assert e_fine.max() < 1.0 * rho0
    assert e_fine.mean() < 0.6 * e_coarse.mean()  # the error shrinks with the voxel size


# --------------------------------------------------------------------------
# P8  linearity / additivity / literal form identity (Q10)
# --------------------------------------------------------------------------

def test_p8_material_routing_and_linearity(workloads_cache):
    w = workloads_cache("C1")
    rng = np.random.default_rng(5)
    pix = np.stack([np.zeros(40, int), rng.integers(0, w.nu, 40), rng.integers(0, w.nv, 40)], 1)
    a = oracle.project(w, pixels=pix)
    # sum over materials = LI of the un-segmented density
    w1 = tiny_workload(w.rho, spacing=w.spacing, nu=w.nu, nv=w.nv, du=w.du, dv=w.dv,
                       step=w.step_mm)
    b = oracle.project(w1, pixels=pix)
    tot = a["line_integrals"].sum(axis=1)
    assert np.max(np.abs(tot - b["line_integrals"][:, 0])) < 1e-10 * tot.max()
    assert a["line_integrals"][:, 1].max() > 1.0      # bone is hit by some ray
    # scaling rho by 2 (exact in fp32) scales every LI by 2
    w2 = w.with_phis(w.phis)
    w2.rho = w.rho * np.float32(2.0)
    c = oracle.project(w2, pixels=pix)
    assert np.max(np.abs(c["line_integrals"] - 2 * a["line_integrals"])) < 1e-10
    # a voxel belongs to exactly one material: swapping labels swaps the LIs
    w3 = w.with_phis(w.phis)
    w3.mat = (1 - w.mat).astype(np.uint8)
    d = oracle.project(w3, pixels=pix)
    assert np.array_equal(d["line_integrals"][:, ::-1], a["line_integrals"])


def test_p8_many_materials_are_the_line_integrals_of_the_masked_fields():
    """Up to 16 materials (reading Q33): LI_m of a volume of 11 materials equals the line integral of the
    one-material volume rho * [mat == m], for every m -- the linearity the CUDA path's groups of four rest on."""
    rng = np.random.default_rng(21)
    shape = (10, 12, 14)
    rho = rng.uniform(0.1, 2.0, size=shape).astype(np.float32)
    mat = rng.integers(0, 11, size=shape).astype(np.uint8)
    kw = dict(spacing=(2.0, 2.5, 3.0), nu=20, nv=16, du=3.0, dv=3.0, phis=np.radians([20.0, 200.0]), step=0.7)
    w = tiny_workload(rho, mat, n_materials=11, mu_hat=rng.uniform(0.01, 0.05, size=(11, 1)), **kw)
    full = oracle.project(w)
    tau = np.zeros_like(full["signal"])
    for m in range(11):
        one = tiny_workload(np.where(mat == m, rho, np.float32(0.0)), **kw)
        li_m = oracle.project(one)["line_integrals"][:, 0]
        np.testing.assert_allclose(full["line_integrals"][:, m], li_m, rtol=1e-12, atol=1e-12)
        tau += w.mu_hat[m, 0] * li_m
    np.testing.assert_allclose(full["signal"], np.exp(-tau), rtol=1e-12)


@pytest.mark.parametrize("name,npix", [("C0", 60), ("C1", 40), ("C2", 12)])
def test_p8_paper_literal_form_equals_factored_form(workloads_cache, name, npix):
    """O5' (one trace per energy channel on mu_E = rho*mu_hat[mat][E], as the
    paper states it) == O5+O6 (per-material traces, mu_hat applied after)."""
    w = workloads_cache(name)
    rng = np.random.default_rng(7)
    pix = np.stack([np.zeros(npix, int), rng.integers(0, w.nu, npix),
                    rng.integers(0, w.nv, npix)], 1)
    fac = oracle.project(w, pixels=pix)
    lit = oracle.project_literal(w, pixels=pix)
    tau_fac = fac["line_integrals"] @ w.mu_hat
    assert np.max(np.abs(lit["tau"] - tau_fac) / (1 + np.abs(lit["tau"]))) < 1e-12
    assert np.max(np.abs(lit["signal"] - fac["signal"]) / fac["signal"]) < 1e-11


# --------------------------------------------------------------------------
# P9  symmetry, rotation equivariance, orientation of u and v (Q1-Q3, Q6)
# --------------------------------------------------------------------------

def test_p9_z_mirror_symmetry():
    rng = np.random.default_rng(11)
    half = rng.uniform(0, 1.5, size=(6, 10, 12)).astype(np.float32)
    rho = np.concatenate([half, half[::-1]], axis=0)
    w = tiny_workload(rho, phis=[math.radians(52.0)], nu=20, nv=18, du=2.5, dv=2.5)
    p = oracle.project(w)["signal"][0]
    assert np.max(np.abs(p - p[::-1, :])) < 1e-13
    assert np.max(np.abs(p - p[:, ::-1])) > 1e-3      # no accidental u symmetry


def test_p9_rotation_equivariance():
    rng = np.random.default_rng(12)
    rho = rng.uniform(0, 1.5, size=(8, 12, 12)).astype(np.float32)
    rho[:, :2], rho[:, -2:], rho[:, :, :2], rho[:, :, -2:] = 0, 0, 0, 0
    mat = (rho > 0.8).astype(np.uint8)
    # rotate the object by +90 deg about z: voxel (ix, iy) -> (N-1-iy, ix)
    rot = lambda a: np.ascontiguousarray(a.transpose(0, 2, 1)[:, :, ::-1])
    kw = dict(n_materials=2, nu=20, nv=14, du=2.5, dv=2.5, step=0.7,
              mu_hat=[[0.02], [0.05]])
    for phi_deg in (0.0, 28.0, 135.0):
        w_a = tiny_workload(rho, mat, phis=[math.radians(phi_deg)], **kw)
        w_b = tiny_workload(rot(rho), rot(mat), phis=[math.radians(phi_deg + 90.0)], **kw)
        a, b = oracle.project(w_a), oracle.project(w_b)
        assert np.max(np.abs(a["signal"] - b["signal"])) < 1e-11
        assert np.max(np.abs(a["line_integrals"] - b["line_integrals"])) < 1e-9
    # theta != 0 moves the detector relative to SO (Q2): with the detector
    # rotated by theta the central pixel's ray is the one at angle phi + theta
    # seen from O only if sad == 0; so just check it changes the image and
    # that theta = 2*pi does not
    w0 = tiny_workload(rho, mat, phis=[0.3], theta=0.0, **kw)
    w1 = tiny_workload(rho, mat, phis=[0.3], theta=0.2, **kw)
    w2 = tiny_workload(rho, mat, phis=[0.3], theta=2 * math.pi, **kw)
    p0, p1, p2 = (oracle.project(x)["signal"] for x in (w0, w1, w2))
    assert np.max(np.abs(p0 - p1)) > 1e-3
    assert np.max(np.abs(p0 - p2)) < 1e-9


@pytest.mark.parametrize("phi_deg", [0.0, 60.0])
def test_p9_shadow_position_of_a_small_ball(phi_deg):
    """A dense ball at (x', y', z) in the frame rotated by phi shadows at
    u = SDD*y'/(SAD + x'), v = SDD*z/(SAD + x')  (+y' -> +u, +z -> +v)."""
    n, vox = 48, 2.0
    phi = math.radians(phi_deg)
    ax = (np.arange(n) - (n - 1) / 2) * vox
    z, y, x = np.meshgrid(ax, ax, ax, indexing="ij")
    xr, yr, zr = 10.0, 22.0, -14.0                      # rotated-frame position
    cx = xr * math.cos(phi) - yr * math.sin(phi)
    cy = xr * math.sin(phi) + yr * math.cos(phi)
    rho = np.where((x - cx) ** 2 + (y - cy) ** 2 + (z - zr) ** 2 <= 5.0 ** 2, 5.0, 0.0)
    w = tiny_workload(rho, spacing=(vox,) * 3, phis=[phi], nu=64, nv=64, du=2.0, dv=2.0)
    li = oracle.project(w)["line_integrals"][0, 0]
    us = (np.arange(w.nu) - (w.nu - 1) / 2) * w.du
    vs = (np.arange(w.nv) - (w.nv - 1) / 2) * w.dv
    u_c = (li.sum(axis=0) * us).sum() / li.sum()
    v_c = (li.sum(axis=1) * vs).sum() / li.sum()
    assert u_c == pytest.approx(1500.0 * yr / (1000.0 + xr), abs=w.du)
    assert v_c == pytest.approx(1500.0 * zr / (1000.0 + xr), abs=w.dv)


def test_p9_detector_angle_theta_orientation():
    """Q2/Q3 with theta != 0: P = AID*(cos(phi+theta), sin(phi+theta), 0), the
    detector plane is perpendicular to OP, u_hat = z_hat x n_hat.  A small ball
    shadows where the line S->ball meets that plane (ray-plane intersection
    done here, independently of the oracle's pixel->ray construction)."""
    n, vox = 64, 2.5
    phi, theta = math.radians(20.0), math.radians(8.0)
    sad, sdd = 1000.0, 1500.0
    S = -sad * np.array([math.cos(phi), math.sin(phi), 0.0])
    n_hat = np.array([math.cos(phi + theta), math.sin(phi + theta), 0.0])
    u_hat = np.array([-math.sin(phi + theta), math.cos(phi + theta), 0.0])
    P = (sdd - sad) * n_hat
    lam = -np.dot(S, P - S) / np.dot(P - S, P - S)        # closest approach of SP to O
    ball = S + lam * (P - S) + 9.0 * u_hat + np.array([0.0, 0.0, -12.0])
    assert np.max(np.abs(ball)) < 0.5 * n * vox - 10
    s_hit = np.dot(P - S, n_hat) / np.dot(ball - S, n_hat)
    H = S + s_hit * (ball - S)
    u_want, v_want = np.dot(H - P, u_hat), H[2]
    assert u_want > 5 and v_want < -5
    ax = (np.arange(n) - (n - 1) / 2) * vox
    z, y, x = np.meshgrid(ax, ax, ax, indexing="ij")
    rho = np.where((x - ball[0]) ** 2 + (y - ball[1]) ** 2 + (z - ball[2]) ** 2 <= 36.0, 4.0, 0.0)
    w = tiny_workload(rho, spacing=(vox,) * 3, phis=[phi], theta=theta, nu=64, nv=64,
                      du=1.5, dv=1.5)
    li = oracle.project(w)["line_integrals"][0, 0]
    us = (np.arange(w.nu) - (w.nu - 1) / 2) * w.du
    vs = (np.arange(w.nv) - (w.nv - 1) / 2) * w.dv
    assert li.sum() > 0
    assert (li.sum(axis=0) * us).sum() / li.sum() == pytest.approx(u_want, abs=w.du)
    assert (li.sum(axis=1) * vs).sum() / li.sum() == pytest.approx(v_want, abs=w.dv)


# --------------------------------------------------------------------------
# P10 bounds; hit/miss table = shadow of the box
# --------------------------------------------------------------------------

def test_p10_bounds(workloads_cache):
    w = workloads_cache("C1")
    out = oracle.project(w)
    flat = float((w.phi_weight * w.response).sum())
    assert out["signal"].min() > 0 and out["signal"].max() <= flat * (1 + 1e-15)
    assert out["line_integrals"].min() >= 0
    diag = math.sqrt(sum((n * d) ** 2 for n, d in zip(w.dims, w.spacing)))
    assert out["ray_table"][..., 1].max() <= math.ceil(diag / w.step_mm) + 1
    assert out["ray_table"][..., 1].min() > 0          # hit fraction 1.0


@pytest.mark.parametrize("phi_deg", [0.0, 37.0])
def test_hit_mask_is_the_shadow_of_the_box(workloads_cache, phi_deg):
    from scipy.spatial import Delaunay
    w = workloads_cache("C0")
    phi = math.radians(phi_deg)
    half = [n * d / 2 for n, d in zip(w.dims, w.spacing)]
    pts = []
    for sx in (-1, 1):
        for sy in (-1, 1):
            for sz in (-1, 1):
                x, y, z = sx * half[0], sy * half[1], sz * half[2]
                xr = x * math.cos(phi) + y * math.sin(phi)
                yr = -x * math.sin(phi) + y * math.cos(phi)
                pts.append((w.sdd * yr / (w.sad + xr), w.sdd * z / (w.sad + xr)))
    hull = Delaunay(np.array(pts))
    us = (np.arange(w.nu) - (w.nu - 1) / 2) * w.du
    vs = (np.arange(w.nv) - (w.nv - 1) / 2) * w.dv
    uu, vv = np.meshgrid(us, vs)
    inside = hull.find_simplex(np.stack([uu.ravel(), vv.ravel()], 1)) >= 0
    hit = np.array([[oracle.ray(w, phi, i, j)["hit"] for i in range(w.nu)]
                    for j in range(w.nv)])
    assert np.array_equal(hit.ravel(), inside)
    if phi_deg == 0.0:
        assert hit.mean() == pytest.approx(1 / 3, abs=0.01)   # 0.333
    n = oracle.project(w.with_phis([phi]))["ray_table"][0, ..., 1]
    assert np.all(n[~hit] == 0)
    assert (n[hit] > 0).mean() > 0.99       # a grazing chord < dl may hold no midpoint


# --------------------------------------------------------------------------
# energy sum: bowtie and response enter exactly as Eq. (1) / Q13 say
# --------------------------------------------------------------------------

def test_energy_sum_against_direct_evaluation(workloads_cache):
    w = workloads_cache("C2")
    rng = np.random.default_rng(13)
    pix = np.stack([np.zeros(25, int), rng.integers(0, w.nu, 25), rng.integers(0, w.nv, 25)], 1)
    out = oracle.project(w, pixels=pix)
    for q, (p, i, j) in enumerate(pix):
        tau = w.mu_hat.T @ out["line_integrals"][q]
        want = np.sum(w.phi_weight * np.exp(-w.bowtie_mu * w.bowtie_thickness[i])
                      * w.response * np.exp(-tau))
        assert out["signal"][q] == pytest.approx(want, rel=1e-13)
    # listed pixels == the same pixels of the full image
    full = oracle.project(w)
    assert np.array_equal(full["signal"][0, pix[:, 2], pix[:, 1]], out["signal"])
    assert np.array_equal(full["ray_table"][0, pix[:, 2], pix[:, 1]], out["ray_table"])


def test_workload_sample_counts_match_survey(workloads_cache):
    """SURVEY.md section 8 workload table: samples per projection and max per ray."""
    want = {"C0": (1.23e5, 129), "C1": (1.20e7, 259), "C2": (1.01e8, 519)}
    for name, (tot, mx) in want.items():
        w = workloads_cache(name)
        n = oracle.project(w, want_li=False)["ray_table"][..., 1]
        assert n.sum() == pytest.approx(tot, rel=0.01)
        assert n.max() == mx


def test_golden_regression(workloads_cache):
    """tests/golden/oracle_regression.txt (written by tests/golden/make_golden.py,
    which calls only oracle/): guards against accidental changes; the paper
    prints no value to store instead."""
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "oracle_regression.txt")
    rows = [l.split() for l in open(path) if not l.startswith("#")]
    assert len(rows) == 10
    for row in rows:
        w = workloads_cache(row[0])
        p, i, j, j0, n = map(int, row[1:6])
        out = oracle.project(w, pixels=np.array([[p, i, j]]))
        assert tuple(out["ray_table"][0]) == (j0, n)
        assert out["signal"][0] == pytest.approx(float(row[6]), rel=1e-13)
        want_li = np.array([float(x) for x in row[7:]])
        assert np.allclose(out["line_integrals"][0], want_li, rtol=1e-13, atol=1e-13)
