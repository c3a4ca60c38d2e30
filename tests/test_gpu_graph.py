"""gdrr_project inside CUDA stream capture (include/gdrr.h: "only enqueues kernels on cuda_stream" once the volume's
ingest is known to have finished): the call is captured into a CUDA graph, the graph is replayed into the same output
buffers, and every replay gives the bits of the direct call.  Checked against the oracle once, so that "the same
bits" are the right ones.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from parity_util import check_signal  # noqa: E402


@pytest.fixture(scope="module")
def gdrr():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    import paper_1204_6367_b200 as g
    return g


def _capture(gdrr, pr, n, want_li, want_table):
    w = pr.w
    sig = torch.zeros((n, w.nv, w.nu), dtype=torch.float32, device="cuda")
    li = torch.zeros((n, w.n_materials, w.nv, w.nu), dtype=torch.float32, device="cuda") if want_li else None
    tab = torch.zeros((n, w.nv, w.nu, 2), dtype=torch.int32, device="cuda") if want_table else None
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        gdrr.gdrr_project(pr.ctx, pr.vol, 0, n, sig, li, tab)
    return graph, sig, li, tab


@pytest.mark.parametrize("name,sampler,method", [("C1", 0, "trilinear"), ("C1", 1, "trilinear"), ("C0", 0, "trilinear"),
                                                 ("C1", 0, "siddon")],
                         ids=["C1-auto", "C1-gather", "C0-auto", "C1-siddon"])
def test_project_replays_from_a_cuda_graph(gdrr, workloads_cache, name, sampler, method):
    w = workloads_cache(name)
    with gdrr.Projector(w, sampler=sampler) as pr:
        if method == "siddon":
            gdrr.gdrr_set_method(pr.ctx, gdrr.GDRR_METHOD_SIDDON)
        eager, li_e, tab_e = pr.project(0, 1, want_li=True, want_table=True)      # (Siddon: also makes the compact copy)
        gdrr.gdrr_volume_status(pr.ctx, pr.vol)              # ingest and copy have finished: gdrr_project only launches now
        torch.cuda.synchronize()
        launches = pr.kernel_launches()
        graph, sig, li, tab = _capture(gdrr, pr, 1, True, True)
        captured = pr.kernel_launches() - launches
        assert captured == 1, f"{captured} kernels captured for one projection call"
        for _ in range(3):
            sig.zero_(); li.zero_(); tab.zero_()
            graph.replay()
            torch.cuda.synchronize()
            assert torch.equal(sig, eager) and torch.equal(li, li_e) and torch.equal(tab, tab_e)
        if method == "trilinear":
            ref = oracle.project(w.with_phis(w.phis[:1]))
            check_signal(sig.cpu().numpy(), ref["signal"], f"{name} from a CUDA graph")
            assert np.array_equal(tab.cpu().numpy(), ref["ray_table"])


def test_graph_of_many_projection_calls(gdrr, workloads_cache):
    """A scan as 12 calls of one projection each, captured once: one graph launch instead of 12 kernel launches."""
    w = workloads_cache("C1")
    w = w.with_phis(np.linspace(0.0, 2.0 * np.pi, 12, endpoint=False))
    with gdrr.Projector(w) as pr:
        gdrr.gdrr_volume_status(pr.ctx, pr.vol)
        eager, _, _ = pr.project(0, 12)
        sig = torch.zeros_like(eager)
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            for p in range(12):
                gdrr.gdrr_project(pr.ctx, pr.vol, p, 1, sig[p:p + 1])
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(sig, eager)
