"""Pins of the oracle's pixel-dependent detector response ("In principle, the detector response could
also be pixel dependent"; reading Q32: r(E, u) = r(E) g(E, u), g float32 [n_energy][nv][nu]).  Each pin
is a closed form or a reduction to something already pinned, never the oracle's own formula retyped."""
import copy

import numpy as np

import oracle
from test_oracle_pins import tiny_workload


def _workload(seed=3, n_mat=2):
    rng = np.random.default_rng(seed)
    rho = rng.uniform(0.2, 1.8, size=(10, 12, 14)).astype(np.float32)
    mat = rng.integers(0, n_mat, size=rho.shape).astype(np.uint8)
    energies = np.array([30.0, 50.0, 70.0, 90.0])
    w = tiny_workload(rho, mat, n_materials=n_mat, nu=22, nv=18, du=2.5, dv=2.5, spacing=(2.0, 2.5, 3.0),
                      phis=np.radians([0.0, 40.0, 200.0]), step=0.7, energies=energies,
                      mu_hat=rng.uniform(0.01, 0.05, size=(n_mat, 4)), phi_weight=np.array([0.1, 0.4, 0.3, 0.2]),
                      response=energies / 50.0)
    w.fluence_map = rng.uniform(0.5, 1.5, size=(w.nv, w.nu)).astype(np.float32)
    w.bowtie_mu = rng.uniform(0.02, 0.1, size=4)
    w.bowtie_thickness = rng.uniform(1.0, 20.0, size=w.nu)
    return w, rng


def test_r1_flat_field_with_a_random_per_pixel_response_has_a_closed_form():
    """Empty volume: P(u) = w(u) sum_E phi_E r_E g(E, u) exp(-mu_bt,E t_bt(u)), written out in numpy."""
    w, rng = _workload()
    w.rho = np.zeros_like(w.rho)
    w.response_gain = rng.uniform(0.2, 1.7, size=(4, w.nv, w.nu)).astype(np.float32)
    out = oracle.project(w)
    want = np.zeros((w.nv, w.nu))
    for e in range(4):
        want += (w.phi_weight[e] * w.response[e] * w.response_gain[e].astype(np.float64)
                 * np.exp(-w.bowtie_mu[e] * w.bowtie_thickness)[None, :])
    want *= w.fluence_map.astype(np.float64)
    for p in range(w.n_proj):
        np.testing.assert_allclose(out["signal"][p], want, rtol=1e-13)
    assert np.all(out["line_integrals"] == 0.0)


def test_r2_unit_gain_is_the_pixel_independent_case_bit_for_bit():
    w, _ = _workload()
    ref = oracle.project(w)
    w1 = copy.copy(w)
    w1.response_gain = np.ones((4, w.nv, w.nu), dtype=np.float32)
    got = oracle.project(w1)
    assert np.array_equal(got["signal"], ref["signal"])
    assert np.array_equal(got["line_integrals"], ref["line_integrals"])
    assert np.array_equal(got["ray_table"], ref["ray_table"])
    # and through the listed-pixel path and the Siddon method
    pix = np.array([[0, 3, 4], [2, 21, 17], [1, 0, 0]])
    assert np.array_equal(oracle.project(w1, pixels=pix)["signal"], oracle.project(w, pixels=pix)["signal"])
    assert np.array_equal(oracle.project(w1, method="siddon")["signal"], oracle.project(w, method="siddon")["signal"])


def test_r3_an_energy_independent_gain_is_a_fluence_map():
    """g(E, u) = a(u): the response factors out of the energy sum, exactly as w(u) does."""
    w, rng = _workload(seed=5)
    a = rng.uniform(0.3, 2.0, size=(w.nv, w.nu)).astype(np.float32)
    w1 = copy.copy(w)
    w1.response_gain = np.broadcast_to(a, (4, w.nv, w.nu)).copy()
    w2 = copy.copy(w)
    w2.fluence_map = (w.fluence_map.astype(np.float64) * a.astype(np.float64))       # float64: no rounding of the product
    got, want = oracle.project(w1)["signal"], oracle.project(w2)["signal"]
    # w2's map is rounded to float32 by the oracle's interface: 6e-8 relative
    np.testing.assert_allclose(got, want, rtol=2e-7)


def test_r4_a_gain_that_selects_one_energy_gives_the_mono_energetic_beer_lambert_term():
    """g(E, u) = [E = E_k] for a pixel-dependent k(u): P = w phi_k r_k exp(-mu_bt,k t) exp(-sum_m mu_hat[m][k] LI_m),
    evaluated in numpy from the line integrals."""
    w, rng = _workload(seed=8)
    k = rng.integers(0, 4, size=(w.nv, w.nu))
    g = np.zeros((4, w.nv, w.nu), dtype=np.float32)
    for e in range(4):
        g[e][k == e] = 1.0
    w.response_gain = g
    out = oracle.project(w)
    li = out["line_integrals"]                                    # [P][M][nv][nu]
    mu_k = w.mu_hat[:, k]                                         # [M][nv][nu]
    tau = np.einsum("mji,pmji->pji", mu_k, li)
    want = (w.fluence_map.astype(np.float64) * w.phi_weight[k] * w.response[k]
            * np.exp(-w.bowtie_mu[k] * w.bowtie_thickness[None, :]))[None] * np.exp(-tau)
    np.testing.assert_allclose(out["signal"], want, rtol=1e-13)


def test_r5_gain_follows_the_pixel_on_a_general_source_path():
    """The same gain on the circular gantry given as poses: identical signals (the gain is indexed by the pixel)."""
    from workloads import trajectories
    w, rng = _workload(seed=11)
    w.response_gain = rng.uniform(0.5, 1.5, size=(4, w.nv, w.nu)).astype(np.float32)
    ref = oracle.project(w)
    wp = w.with_poses(trajectories.circular_poses(w.sad, w.sdd, w.theta, w.phis))
    got = oracle.project(wp)
    assert np.array_equal(got["ray_table"], ref["ray_table"])
    np.testing.assert_allclose(got["signal"], ref["signal"], rtol=1e-12)
