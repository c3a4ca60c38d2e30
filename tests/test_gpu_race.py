"""Race evidence for the staged sampler's TMA ring (project_staged.cu): compute-sanitizer is closed on this GPU pool
(DESIGN.md section 8b), so the evidence that can be had is (a) bit-identical images over many repeats, (b) the same with
a co-running kernel on a second stream and with 1, 8 and 360 projections per launch (different CTA co-residency), and
(c) a build of the kernel whose warps are delayed into forced orders (gdrr_debug_set_skew) and must return the same
bits.  The happens-before argument for every shared word is in DESIGN.md section 5."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def gdrr():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    import paper_1204_6367_b200 as g
    return g


def _project(pr, begin, count):
    sig, li, _ = pr.project(proj_begin=begin, proj_count=count, want_li=True)
    return sig, li


@pytest.mark.parametrize("name,phis_deg,repeats", [("C2", [0.0, 37.0, 211.0], 60), ("C3", None, 50)])
def test_repeated_launches_are_bit_identical(gdrr, workloads_cache, name, phis_deg, repeats):
    """(a) the same launch `repeats` times: signal AND line integrals identical to the first, bit for bit."""
    w = workloads_cache(name)
    if phis_deg is not None:
        w = w.with_phis(np.radians(phis_deg))
    n = w.n_proj if phis_deg is not None else 8
    begin = 0 if phis_deg is not None else 41
    with gdrr.Projector(w, sampler=gdrr.GDRR_SAMPLER_STAGED) as pr:
        sig0, li0 = _project(pr, begin, n)
        assert gdrr.gdrr_last_sampler(pr.ctx) == gdrr.GDRR_SAMPLER_STAGED
        for k in range(repeats):
            sig, li = _project(pr, begin, n)
            assert torch.equal(sig, sig0) and torch.equal(li, li0), f"{name}: repeat {k} differs"


def test_co_running_kernel_and_launch_sizes(gdrr, workloads_cache):
    """(b) a matrix product spins on a second stream while C3 is projected with 1, 8 and 360 projections per launch: every
    image must equal the one a quiet single-projection launch gave."""
    w = workloads_cache("C3")
    side = torch.cuda.Stream()
    a = torch.randn((4096, 4096), device="cuda")
    with gdrr.Projector(w, sampler=gdrr.GDRR_SAMPLER_STAGED) as pr:
        quiet = {p: pr.project(proj_begin=p, proj_count=1)[0].clone() for p in (0, 7, 45, 100, 359)}
        torch.cuda.synchronize()
        for per_launch in (1, 8, 360):
            with torch.cuda.stream(side):
                for _ in range(40):
                    a = torch.tanh(a @ a * 1e-3)
            out = torch.empty((w.n_proj, w.nv, w.nu), dtype=torch.float32, device="cuda")
            for b in range(0, w.n_proj, per_launch):
                if per_launch == 1 and b not in quiet:
                    continue
                n = min(per_launch, w.n_proj - b)
                gdrr.gdrr_project(pr.ctx, pr.vol, b, n, out[b:b + n])
            torch.cuda.synchronize()
            for p, ref in quiet.items():
                assert torch.equal(out[p], ref[0]), f"{per_launch} projections per launch: projection {p} differs"


@pytest.mark.parametrize("mode", [1, 2, 3])
def test_forced_warp_orders_give_the_same_bits(gdrr, workloads_cache, mode):
    """(c) the skewed build of the staged kernel (warps sleep before every barrier operation of the ring, keyed on warp
    and chunk: pseudo-random / one warp always last / the producer late) against the product kernel."""
    for name, phis_deg in (("C1", [0.0, 37.0, 90.0, 123.4]), ("C2", [0.0, 211.0])):
        w = workloads_cache(name).with_phis(np.radians(phis_deg))
        with gdrr.Projector(w, sampler=gdrr.GDRR_SAMPLER_STAGED) as pr:
            sig0, li0 = _project(pr, 0, w.n_proj)
            gdrr.gdrr_debug_set_skew(pr.ctx, mode)
            sig1, li1 = _project(pr, 0, w.n_proj)
            gdrr.gdrr_debug_set_skew(pr.ctx, 0)
            sig2, li2 = _project(pr, 0, w.n_proj)
        assert torch.equal(sig0, sig1) and torch.equal(li0, li1), f"{name}: skew mode {mode} changed the result"
        assert torch.equal(sig0, sig2) and torch.equal(li0, li2)
    # a volume whose chunks do not fit the box (C0): the ring then carries only "gather this chunk" messages
    w = workloads_cache("C0")
    with gdrr.Projector(w, sampler=gdrr.GDRR_SAMPLER_STAGED) as pr:
        sig0, li0 = _project(pr, 0, 1)
        gdrr.gdrr_debug_set_skew(pr.ctx, mode)
        sig1, li1 = _project(pr, 0, 1)
    assert torch.equal(sig0, sig1) and torch.equal(li0, li1)
