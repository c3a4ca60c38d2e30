"""What GDRR_SAMPLER_AUTO picks is part of the measured performance (gdrr_api.cu beam_fits): pin it, so that a
regression shows as a failing test and not only as a slower number.  Also: the per-sample cell check of SURVEY.md Q9."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from workloads import trajectories  # noqa: E402


@pytest.fixture(scope="module")
def gdrr():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    import paper_1204_6367_b200 as g
    return g


def _picked(gdrr, w, count=None):
    with gdrr.Projector(w) as pr:                                    # GDRR_SAMPLER_AUTO
        assert gdrr.gdrr_last_sampler(pr.ctx) == 0
        pr.project(proj_begin=0, proj_count=count or w.n_proj)
        torch.cuda.synchronize()
        return gdrr.gdrr_last_sampler(pr.ctx)


def test_auto_picks_the_staged_kernel_on_the_timed_configs(gdrr, workloads_cache):
    for name in ("C1", "C2", "C3", "C4"):
        assert _picked(gdrr, workloads_cache(name)) == gdrr.GDRR_SAMPLER_STAGED, name
    # C0's 2 mm voxels under a 3.1 mm detector: a CTA's beam over 16 steps does not fit the box
    assert _picked(gdrr, workloads_cache("C0")) == gdrr.GDRR_SAMPLER_GATHER


def test_auto_choice_on_other_source_paths(gdrr, workloads_cache):
    w = workloads_cache("C3")
    phis = w.phis                                   # the whole orbit: the choice is made on the mean beam extent
    nz_mm = w.dims[2] * w.spacing[2]
    helix = w.with_poses(trajectories.helical_poses(w.sad, w.sdd, phis, pitch_mm=0.5 * nz_mm, z0_mm=-0.25 * nz_mm))
    assert _picked(gdrr, helix) == gdrr.GDRR_SAMPLER_STAGED
    for tilt, want in ((10.0, "STAGED"), (20.0, "STAGED"), (35.0, "GATHER")):
        tilted = w.with_poses(trajectories.c_arm_poses(w.sad, w.sdd, phis, np.deg2rad(tilt)))
        assert _picked(gdrr, tilted) == getattr(gdrr, "GDRR_SAMPLER_" + want), tilt
    # an explicit choice is honoured; exact layouts report 0
    with gdrr.Projector(w, sampler=gdrr.GDRR_SAMPLER_GATHER) as pr:
        pr.project(proj_begin=0, proj_count=1)
        assert gdrr.gdrr_last_sampler(pr.ctx) == gdrr.GDRR_SAMPLER_GATHER
    with gdrr.Projector(workloads_cache("C1"), layout=gdrr.GDRR_LAYOUT_LINEAR) as pr:
        pr.project(proj_begin=0, proj_count=1)
        assert gdrr.gdrr_last_sampler(pr.ctx) == 0


@pytest.mark.parametrize("sampler", [1, 2])
@pytest.mark.parametrize("name", ["C0", "C1"])
def test_per_sample_cells_agree_with_the_oracle(gdrr, workloads_cache, name, sampler):
    """the cell of every sample, formed by the kernel's own position arithmetic (gdrr_debug_ray_cells),
    equals floor() of the oracle's fp64 position except where that position is within 2^-12 of a cell face."""
    w = workloads_cache(name).with_phis(np.radians([0.0, 33.0, 90.0, 201.5]))
    rng = np.random.default_rng(9)
    checked = ties = 0
    with gdrr.Projector(w) as pr:
        cells = torch.empty((4096, 3), dtype=torch.int32, device="cuda")
        count = torch.zeros(1, dtype=torch.int32, device="cuda")
        for p in range(w.n_proj):
            pix = [(0, 0), (w.nu - 1, w.nv - 1), (w.nu // 2, w.nv // 2)] + \
                  [(int(rng.integers(w.nu)), int(rng.integers(w.nv))) for _ in range(40)]
            for i, j in pix:
                gdrr.gdrr_debug_ray_cells(pr.ctx, pr.vol, p, i, j, sampler, cells, count)
                n = int(count.item())
                gi, ref = oracle.ray_samples(w, float(w.phis[p]), i, j)
                assert n == len(gi)
                if n == 0:
                    continue
                got = cells[:n].cpu().numpy()
                diff = got != ref
                fr = gi - np.floor(gi)
                near = np.minimum(fr, 1.0 - fr)
                assert np.all(near[diff] < 2.0 ** -12), (name, p, i, j, got[diff.any(axis=1)][:3], gi[diff.any(axis=1)][:3])
                assert np.all(np.abs(got - ref) <= 1)
                checked += n
                ties += int(diff.sum())
    print(f"{name} sampler {sampler}: {checked} samples compared, {ties} face ties")
    assert checked > 1000
