"""Randomised differential test: seeded random workloads (volume kind, size, spacing, offset, material count 1..9,
geometry, detector offset, bowtie, fluence map, response gain, helical and C-arm poses, step length) through a random
kernel of the library (midpoint rule or Siddon; packed, brick or linear layout; AUTO, gather or staged sampler) against
the oracle, with the bars of every other parity test (tests/parity_util.py).  The default run takes 120 seeds in blocks
of 20; `python -m pytest tests/test_gpu_random_workloads.py -m gpu --random-cases N` takes N more from another seed range
(round 2 ran 14,900 further cases with volumes up to 150 voxels and detectors up to 220 pixels a side: no failure, worst
relative signal error 8.0e-6)."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from parity_util import (check_line_integrals, check_ray_table, check_signal, face_tie_checker,  # noqa: E402
                         siddon_sliver_checker)
from test_oracle_pins import tiny_workload  # noqa: E402
from workloads import trajectories  # noqa: E402


@pytest.fixture(scope="module")
def gdrr():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    import paper_1204_6367_b200 as g
    return g


def structured_volume(rng, shape, n_mat):
    nz, ny, nx = shape
    z, y, x = np.meshgrid(np.linspace(-1, 1, nz), np.linspace(-1, 1, ny), np.linspace(-1, 1, nx), indexing="ij")
    rho = np.zeros(shape, dtype=np.float32); mat = np.zeros(shape, dtype=np.uint8)
    kind = rng.integers(0, 3)
    if kind == 0:                                  # random voxels
        rho = rng.uniform(0, 2, size=shape).astype(np.float32); rho[rng.uniform(size=shape) < 0.2] = 0
        mat = rng.integers(0, n_mat, size=shape).astype(np.uint8)
    else:                                          # ellipsoids of random materials in a body, optional noise
        body = (x / 0.9) ** 2 + (y / 0.8) ** 2 + (z / 0.95) ** 2 < 1
        rho[body] = 1.0
        for _ in range(rng.integers(3, 12)):
            c = rng.uniform(-0.6, 0.6, 3); r = rng.uniform(0.1, 0.4, 3)
            e = ((x - c[0]) / r[0]) ** 2 + ((y - c[1]) / r[1]) ** 2 + ((z - c[2]) / r[2]) ** 2 < 1
            rho[e] = rng.uniform(0.2, 1.9); mat[e] = rng.integers(0, n_mat)
        if kind == 2:
            flip = rng.uniform(size=shape) < 0.05
            mat = np.where(flip, rng.integers(0, n_mat, size=shape), mat).astype(np.uint8)
            rho = (rho * rng.normal(1.0, 0.02, size=shape)).astype(np.float32).clip(0)
    return rho, mat

def random_case(seed, max_dim=72, max_nu=90):
    rng = np.random.default_rng(seed)
    n_mat = int(rng.choice([1, 2, 3, 4, 4, 4, 5, 7, 9]))
    shape = tuple(int(v) for v in rng.integers(8, max_dim, 3))
    if rng.uniform() < 0.5: shape = shape[:2] + (4 * max(2, shape[2] // 4),)       # rows 4-voxel aligned: vector ingest
    rho, mat = structured_volume(rng, shape, n_mat)
    spacing = tuple(float(v) for v in rng.uniform(0.6, 2.5, 3))
    extent = max(shape[2] * spacing[0], shape[1] * spacing[1], shape[0] * spacing[2])
    sad = float(rng.uniform(1.5, 6.0) * extent); sdd = float(sad * rng.uniform(1.2, 2.0))
    nu, nv = int(rng.integers(10, max_nu)), int(rng.integers(10, 70))
    fan = extent * sdd / sad * rng.uniform(0.6, 1.4)
    du, dv = float(fan / nu), float(fan / nv * rng.uniform(0.6, 1.2))
    ne = int(rng.choice([1, 3, 8]))
    energies = np.linspace(30, 110, ne)
    n_proj = int(rng.integers(1, 5))
    kw = dict(spacing=spacing, n_materials=n_mat, nu=nu, nv=nv, du=du, dv=dv, sad=sad, sdd=sdd,
              phis=rng.uniform(0, 2 * math.pi, n_proj), step=float(rng.uniform(0.3, 0.9) * min(spacing)),
              energies=energies, mu_hat=rng.uniform(0.01, 0.05, size=(n_mat, ne)), phi_weight=np.full(ne, 1.0 / ne),
              response=rng.uniform(0.5, 1.5, ne), theta=float(rng.choice([0.0, 0.0, rng.uniform(-0.2, 0.2)])),
              centre=tuple(float(v) for v in rng.uniform(-0.1, 0.1, 3) * extent))
    w = tiny_workload(rho, mat, **kw)
    if rng.uniform() < 0.3: w.u_off = float(rng.uniform(-0.2, 0.2) * fan)
    if rng.uniform() < 0.3: w.fluence_map = rng.uniform(0.5, 1.5, size=(nv, nu)).astype(np.float32)
    if rng.uniform() < 0.3:
        w.bowtie_mu = rng.uniform(0.01, 0.03, ne); w.bowtie_thickness = rng.uniform(0, 20, nu)
    if rng.uniform() < 0.2: w.response_gain = rng.uniform(0.5, 1.5, size=(ne, nv, nu)).astype(np.float32)
    pose = rng.uniform()
    if pose < 0.15: w = w.with_poses(trajectories.helical_poses(w.sad, w.sdd, w.phis, float(rng.uniform(5, 40))))
    elif pose < 0.3: w = w.with_poses(trajectories.c_arm_poses(w.sad, w.sdd, w.phis, float(rng.uniform(0, 0.7))))
    method = "siddon" if rng.uniform() < 0.3 else "trilinear"
    layout = int(rng.choice([2, 2, 2, 0, 1]))
    sampler = int(rng.choice([0, 1, 2])) if layout == 2 else 0
    return w, method, layout, sampler

def run_case(g, seed, max_dim=72, max_nu=90):
    w, method, layout, sampler = random_case(seed, max_dim, max_nu)
    what = f"seed {seed} {method} layout {layout} sampler {sampler} shape {w.rho.shape} nmat {w.n_materials} det {w.nu}x{w.nv} proj {len(w.phis)} poses {w.poses is not None}"
    ref = oracle.project(w, method=method)
    kw = dict(method=g.GDRR_METHOD_SIDDON) if method == "siddon" else {}
    with g.Projector(w, layout=layout, sampler=sampler, **kw) as pr:
        sig, li, tab = pr.project(want_li=True, want_table=True)
    check_ray_table(tab.cpu().numpy(), ref["ray_table"], what)
    idx = list(range(len(w.phis)))
    checker = siddon_sliver_checker(w, idx) if method == "siddon" else face_tie_checker(w, idx)
    check_line_integrals(li.cpu().numpy(), ref["line_integrals"], what, checker)
    return check_signal(sig.cpu().numpy(), ref["signal"], what), what


@pytest.mark.parametrize("block", range(6))
def test_random_workloads_match_the_oracle(gdrr, block):
    worst = 0.0
    for seed in range(20 * block, 20 * block + 20):
        err, what = run_case(gdrr, seed)
        worst = max(worst, err)
    print(f"seeds {20 * block}..{20 * block + 19}: worst relative signal error {worst:.2e}")


def test_more_random_workloads(gdrr, request):
    """--random-cases N: N further cases, larger volumes and detectors (0 by default)."""
    n = int(request.config.getoption("--random-cases"))
    worst = 0.0
    for seed in range(100000, 100000 + n):
        err, what = run_case(gdrr, seed, max_dim=150, max_nu=220)
        worst = max(worst, err)
    print(f"{n} further cases: worst relative signal error {worst:.2e}")
