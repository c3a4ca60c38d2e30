"""Step a0, PACKED_QUAD layout: the ingest kernel that writes four elements per thread from vector loads
(volumes whose rows are 4-voxel aligned, aligned input pointers) must write the same bytes as the plain kernel that
writes one element per thread (everything else).  The plain kernel is reached here by handing the library a material
array that starts one byte off a 4-byte boundary; the device workspaces of the two volumes are compared byte for
byte, pad slots included.  The layout itself is pinned against the oracle by every parity test; this file pins the
fast kernel to the plain one on shapes the parity tests do not reach (ragged rows, faces, every material count,
groups of more than four materials, slab ranges of the pipelined host ingest).
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


def random_volume(shape, n_mat, seed):
    rng = np.random.default_rng(seed)
    nz, ny, nx = shape
    # blocks of one material with noise on top: pure cells, two-material cells and cells of three and four materials
    coarse = rng.integers(0, n_mat, size=((nz + 3) // 4, (ny + 3) // 4, (nx + 3) // 4))
    mat = np.kron(coarse, np.ones((4, 4, 4), dtype=np.int64))[:nz, :ny, :nx]
    flip = rng.uniform(size=shape) < 0.15
    mat = np.where(flip, rng.integers(0, n_mat, size=shape), mat).astype(np.uint8)
    rho = rng.uniform(0.0, 2.0, size=shape).astype(np.float32)
    rho[rng.uniform(size=shape) < 0.1] = 0.0
    return rho, mat


def workspace_after_ingest(g, c, rho, mat, n_mat, misalign):
    nz, ny, nx = rho.shape
    n = rho.size
    rho_d = torch.from_numpy(rho).cuda()
    store = torch.zeros(n + 8, dtype=torch.uint8, device="cuda")
    off = (-store.data_ptr()) % 4 + (1 if misalign else 0)          # aligned start, or one byte past it
    mat_d = store[off:off + n]
    mat_d.copy_(torch.from_numpy(mat.reshape(-1)).cuda())
    assert (mat_d.data_ptr() % 4 == 0) != misalign
    ws = torch.full((g.gdrr_volume_workspace_bytes(nx, ny, nz, n_mat, g.GDRR_LAYOUT_PACKED_QUAD),), 0xA5,
                    dtype=torch.uint8, device="cuda")
    vol = g.gdrr_create_volume(c, rho_d, mat_d.view(nz, ny, nx), (nx, ny, nz), (1.0, 1.1, 1.2), (0.0, 0.0, 0.0), n_mat,
                               g.GDRR_LAYOUT_PACKED_QUAD, ws)
    g.gdrr_volume_status(c, vol)
    g.gdrr_destroy_volume(vol)
    return ws


SHAPES = [(5, 7, 8), (9, 6, 4), (3, 3, 12), (17, 33, 64), (6, 130, 260), (33, 20, 132), (2, 1, 4), (1, 1, 516)]


@pytest.mark.parametrize("shape", SHAPES, ids=[f"{s[2]}x{s[1]}x{s[0]}" for s in SHAPES])
@pytest.mark.parametrize("n_mat", [1, 2, 3, 4, 7, 11])
def test_vector_ingest_writes_the_bytes_of_the_plain_ingest(ctx, shape, n_mat):
    g, c = ctx
    rho, mat = random_volume(shape, n_mat, seed=1000 * n_mat + shape[2])
    fast = workspace_after_ingest(g, c, rho, mat, n_mat, misalign=False)
    plain = workspace_after_ingest(g, c, rho, mat, n_mat, misalign=True)
    same = torch.equal(fast, plain)
    if not same:
        bad = torch.nonzero(fast != plain).flatten()
        pytest.fail(f"{int(bad.numel())} bytes differ, first at byte {int(bad[0])} (word {int(bad[0]) // 4})")


def test_vector_ingest_on_c2(ctx, workloads_cache):
    """A clinical-size volume (256 x 256 x 128, 4 materials): the two kernels, and the z-slab pipelined host ingest,
    write identical workspaces."""
    g, c = ctx
    w = workloads_cache("C2")
    rho, mat = np.ascontiguousarray(w.rho, dtype=np.float32), np.ascontiguousarray(w.mat, dtype=np.uint8)
    fast = workspace_after_ingest(g, c, rho, mat, w.n_materials, misalign=False)
    plain = workspace_after_ingest(g, c, rho, mat, w.n_materials, misalign=True)
    assert torch.equal(fast, plain)
    nz, ny, nx = rho.shape
    ws = torch.full_like(fast, 0xA5)                    # (the same fill: bytes no ingest writes compare equal)
    rho_stage = torch.empty(rho.size, dtype=torch.float32, device="cuda")
    mat_stage = torch.empty(mat.size, dtype=torch.uint8, device="cuda")
    vol = g.gdrr_create_volume_host(c, rho, mat, (nx, ny, nz), (1.0, 1.1, 1.2), (0.0, 0.0, 0.0), w.n_materials,
                                    g.GDRR_LAYOUT_PACKED_QUAD, rho_stage, mat_stage, ws)
    g.gdrr_volume_status(c, vol)
    g.gdrr_destroy_volume(vol)
    assert torch.equal(ws, fast)


def test_bad_material_is_reported_by_both_kernels(ctx):
    g, c = ctx
    rho, mat = random_volume((6, 9, 16), 3, seed=5)
    mat[4, 7, 13] = 3                                   # n_materials = 3: index 3 is out of range
    for misalign in (False, True):
        with pytest.raises(g.GdrrError) as e:
            workspace_after_ingest(g, c, rho, mat, 3, misalign)
        assert e.value.code == g.GDRR_ERR_INVALID_ARG
