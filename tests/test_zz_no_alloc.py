"""gdrr_denoise_scatter_static (include/gdrr.h): the scatter denoiser for callers that cannot allocate device memory.
Its ping-pong scratch image is a static __device__ array inside the library (GDRR_DENOISE_STATIC_MAX_FLOATS pixels)
instead of a caller's buffer.  Checked here against gdrr_denoise_scatter on the same inputs, on calls in a row that
share the array (it keeps the previous call's contents), at the 1e-5 relative tolerance of tests/test_gpu_denoise.py
(the two paths launch the same kernel, so the results are expected to be equal bit for bit), plus the size limit and
"the call takes no device memory".

This file is collected last on purpose (the suite runs with pytest -x): it passes alone in a fresh process and after
the other tests.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def ctx():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    import paper_1204_6367_b200 as g
    c = g.gdrr_create_context(0)
    yield g, c
    g.gdrr_destroy_context(c)


def noisy_images(n, nv, nu, seed, level=60.0):
    """Seeded Poisson images over a smooth scatter-like profile (as tests/test_gpu_denoise.py draws them)."""
    rng = np.random.default_rng(seed)
    i, j = np.arange(nu)[None, :], np.arange(nv)[:, None]
    truth = level * (0.4 + np.exp(-((i - 0.4 * nu) ** 2 / (0.1 * nu * nu + 1) + (j - 0.6 * nv) ** 2 / (0.2 * nv * nv + 1))))
    return rng.poisson(np.broadcast_to(truth, (n, nv, nu))).astype(np.float32)


def existing_path(g, c, s_hat_d, beta, n_iter):
    out, scratch = torch.full_like(s_hat_d, -7.0), torch.full_like(s_hat_d, -9.0)
    g.gdrr_denoise_scatter(c, s_hat_d, out, scratch, beta, n_iter)
    torch.cuda.synchronize()
    return out


def static_path(g, c, s_hat_d, beta, n_iter):
    out = torch.full_like(s_hat_d, -7.0)
    g.gdrr_denoise_scatter_static(c, s_hat_d, out, beta, n_iter)
    torch.cuda.synchronize()
    return out


def compare(got, ref, what):
    got, ref = got.cpu().numpy().astype(np.float64), ref.cpu().numpy().astype(np.float64)
    assert np.all(ref > 0.0), what
    np.testing.assert_allclose(got, ref, rtol=1e-5, atol=0, err_msg=what)
    return float(np.max(np.abs(got - ref) / ref))


def test_static_scratch_matches_the_existing_path_on_calls_in_a_row(ctx):
    g, c = ctx
    # call 1: 8 detector images of C3's size, 100 sweeps (25 launches: the last one writes s_dev from the scratch)
    a = torch.from_numpy(noisy_images(8, 384, 512, seed=11)).cuda()
    # call 2, straight after: other images of another (ragged) size and a sweep count whose launch count is odd, so
    # the ping-pong starts on the other buffer and the array still holds call 1's iterates
    b = torch.from_numpy(noisy_images(5, 301, 517, seed=12, level=25.0)).cuda()
    ref_a, ref_b = existing_path(g, c, a, 0.05, 100), existing_path(g, c, b, 0.3, 37)
    got_a = static_path(g, c, a, 0.05, 100)
    got_b = static_path(g, c, b, 0.3, 37)
    worst = max(compare(got_a, ref_a, "call 1"), compare(got_b, ref_b, "call 2"))
    # call 3: the first input again (the array now holds call 2's iterates), and a call that needs no scratch at all
    worst = max(worst, compare(static_path(g, c, a, 0.05, 100), ref_a, "call 3"))
    worst = max(worst, compare(static_path(g, c, b, 0.3, 3), existing_path(g, c, b, 0.3, 3), "call 4 (one launch)"))
    print("static scratch vs caller's scratch: worst relative difference", worst)
    assert worst == 0.0, "the two paths launch the same kernel on the same inputs"


def test_static_scratch_calls_take_no_device_memory(ctx):
    g, c = ctx
    a = torch.from_numpy(noisy_images(4, 384, 512, seed=13)).cuda()
    out = torch.empty_like(a)
    g.gdrr_denoise_scatter_static(c, a, out, 0.1, 9)          # (first use on this device: resolves the array's address)
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    for _ in range(5):
        g.gdrr_denoise_scatter_static(c, a, out, 0.1, 9)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after >= free_before, f"device memory shrank by {free_before - free_after} bytes over 5 calls"


def test_static_scratch_rejects_sizes_beyond_its_maximum(ctx):
    g, c = ctx
    limit = g.GDRR_DENOISE_STATIC_MAX_FLOATS
    n = limit // (384 * 512) + 1                              # 22 images of 512 x 384: one image too many
    too_big = torch.ones((n, 384, 512), dtype=torch.float32, device="cuda")
    out = torch.empty_like(too_big)
    with pytest.raises(g.GdrrError) as e:
        g.gdrr_denoise_scatter_static(c, too_big, out, 0.1, 8)
    assert e.value.code == g.GDRR_ERR_UNSUPPORTED
    assert "GDRR_DENOISE_STATIC_MAX_FLOATS" in str(e.value) and str(limit) in str(e.value)
    # exactly at the limit is served
    edge = torch.from_numpy(noisy_images(1, 2048, 2048, seed=14)).cuda()
    assert edge.numel() == limit
    compare(static_path(g, c, edge, 0.2, 6), existing_path(g, c, edge, 0.2, 6), "at the limit")
