"""GPU parity of the pixel-dependent detector response (gdrr_set_response_gain, reading Q32) and of a
half-fan detector offset, against the oracle."""
import copy

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from parity_util import check_signal, compare_full  # noqa: E402


@pytest.fixture(scope="module")
def gdrr():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    import paper_1204_6367_b200 as g
    return g


def _with_gain(w, seed):
    rng = np.random.default_rng(seed)
    w = copy.copy(w)
    w.response_gain = rng.uniform(0.3, 1.8, size=(w.n_energy, w.nv, w.nu)).astype(np.float32)
    return w


@pytest.mark.parametrize("layout,sampler", [(2, 0), (2, 1), (0, 0), (1, 0)])
def test_response_gain_parity(gdrr, workloads_cache, layout, sampler):
    w = _with_gain(workloads_cache("C1").with_phis(np.radians([0.0, 37.0, 123.4])), 21)
    ref = oracle.project(w)
    with gdrr.Projector(w, layout=layout, sampler=sampler) as pr:
        stats = compare_full(pr, w, ref, f"gain layout {layout} sampler {sampler}")
    print(stats)
    # and it is not a no-op: the same scan without the gain differs
    plain = oracle.project(workloads_cache("C1").with_phis(np.radians([0.0, 37.0, 123.4])))
    assert np.abs(plain["signal"] / ref["signal"] - 1.0).max() > 0.1


def test_response_gain_on_c2_siddon_and_poses(gdrr, workloads_cache):
    from workloads import trajectories
    w = _with_gain(workloads_cache("C2").with_phis(np.radians([211.0])), 22)
    ref = oracle.project(w, method="siddon")
    with gdrr.Projector(w, method=gdrr.GDRR_METHOD_SIDDON) as pr:
        sig, _, _ = pr.project()
    check_signal(sig.cpu().numpy(), ref["signal"], "gain + siddon")
    wp = w.with_poses(trajectories.helical_poses(w.sad, w.sdd, np.radians([10.0, 100.0]), pitch_mm=60.0))
    with gdrr.Projector(wp) as pr:
        compare_full(pr, wp, oracle.project(wp), "gain + helix")


def test_unit_gain_and_clearing_give_the_plain_bits(gdrr, workloads_cache):
    w = workloads_cache("C1").with_phis(np.radians([15.0, 200.0]))
    with gdrr.Projector(w) as pr:
        plain, _, _ = pr.project()
        gdrr.gdrr_set_response_gain(pr.ctx, np.ones((w.n_energy, w.nv, w.nu), dtype=np.float32))
        unit, _, _ = pr.project()
        gdrr.gdrr_set_response_gain(pr.ctx, 2.0 * np.ones((w.n_energy, w.nv, w.nu), dtype=np.float32))
        twice, _, _ = pr.project()
        gdrr.gdrr_set_response_gain(pr.ctx, None)
        cleared, _, _ = pr.project()
        with pytest.raises(ValueError):
            gdrr.gdrr_set_response_gain(pr.ctx, np.ones((w.n_energy, 3, 3), dtype=np.float32))
    assert torch.equal(plain, unit) and torch.equal(plain, cleared)
    assert torch.equal(twice, 2.0 * plain)


def test_half_fan_detector_offset(gdrr, workloads_cache):
    """A half-fan scan: the detector shifted by 148 mm, so that the rays of its far edge cross only a corner of the
    volume; per-pixel parity on two full C2-sized projections."""
    w = copy.copy(workloads_cache("C2").with_phis(np.radians([0.0, 123.0])))
    w.u_off = 148.0
    ref = oracle.project(w)
    with gdrr.Projector(w) as pr:
        stats = compare_full(pr, w, ref, "half fan")
    n = ref["ray_table"][..., 1]
    assert n.min() < 0.5 * n.max()                                # chords from a corner of the box to its full width
    print(stats)
