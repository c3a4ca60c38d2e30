// gdrr_debug_ray_cells: the cell (integer part of the index-space position) of every midpoint sample of ONE ray, formed
// exactly as the packed samplers form it -- the same device functions (chunk_base for the gather kernel's fp64 re-base
// every P.chunk samples, walk_init / walk_advance for the staged kernel's 5.27 fixed-point chunk bases, the 9.23 in-chunk
// steps) in the same order, with the chunk grid anchored as in the kernels (at the smallest first index of the ray's
// warp, or of its CTA).  tests/test_gpu_cells.py compares the cells with the oracle's fp64 positions (SURVEY.md Q9:
// they may differ only where a position is within 2^-12 of a cell face).  Not on any product path.
#include "packed_sampler.cuh"

namespace gdrr {

// one CTA = the 16 x 16 tile of the ray; `staged`: the staged kernel's walk, else the gather kernel's
__global__ void __launch_bounds__(kThreads)
gdrr_debug_ray_cells_kernel(const ProjectParams P, int pi, int pj, int staged, int32_t* cells, int max_samples,
                            int32_t* count) {
    __shared__ int krange[2];
    if (threadIdx.x == 0) { krange[0] = 0x7fffffff; krange[1] = (int)0x80000000; }
    __syncthreads();
    const int lane = threadIdx.x & 31;
    const int i = (pi / kTileU) * kTileU + ((threadIdx.x >> 5) & 3) * 4 + (lane & 3);
    const int j = (pj / kTileV) * kTileV + (threadIdx.x >> 7) * 8 + (lane >> 2);
    const bool valid = i < P.g.nu && j < P.g.nv;
    Ray r;
    ray_setup(P.g, P.g.proj_begin, min(i, P.g.nu - 1), min(j, P.g.nv - 1), r);
    if (!valid) r.n = 0;
    double gs[3], dg[3];
    index_line(P.g, r, gs, dg);
    const int j0 = r.j0, n = r.n;
    const int wmin = __reduce_min_sync(0xffffffffu, n > 0 ? j0 : 0x7fffffff);
    const int wmax = __reduce_max_sync(0xffffffffu, n > 0 ? j0 + n : (int)0x80000000);
    if (lane == 0 && wmin < wmax) {
        atomicMin(&krange[0], wmin);
        atomicMax(&krange[1], wmax);
    }
    __syncthreads();
    if (i != pi || j != pj) return;
    *count = n;
    const int dq[3] = {__double2int_rn(dg[0] * 8388608.0), __double2int_rn(dg[1] * 8388608.0),
                       __double2int_rn(dg[2] * 8388608.0)};
    if (staged) {
        const int kmin = krange[0], kmax = krange[1];
        if (kmin >= kmax) return;
        const int c_begin = kmin / kStageK;
        const int nchunks = (kmax - 1) / kStageK - c_begin + 1;
        ChunkWalk W;
        walk_init(gs, dg, c_begin, W);
        for (int m = 0; m < nchunks; ++m) {
            for (int s = 0; s < kStageK; ++s) {
                const int k = (c_begin + m) * kStageK + s - j0;
                if (k >= 0 && k < n && k < max_samples)
                    for (int a = 0; a < 3; ++a)
                        cells[3 * k + a] = W.cb[a] + (((W.qb[a] >> (kBaseBits - kFracBits)) + s * dq[a]) >> kFracBits) - 1;
            }
            walk_advance(W);
        }
    } else {
        const int CH = P.chunk;
        for (int kc = (wmin / CH) * CH; kc < wmax; kc += CH) {
            const int s0 = max(wmin - kc, 0);
            const int cnt = min(wmax - kc, CH) - s0;
            const ChunkBase b = chunk_base(gs, dg, kc + s0);
            const int bc[3] = {b.cx, b.cy, b.cz}, bq[3] = {b.qx, b.qy, b.qz};
            for (int s = 0; s < cnt; ++s) {
                const int k = kc + s0 + s - j0;
                if (k >= 0 && k < n && k < max_samples)
                    for (int a = 0; a < 3; ++a) cells[3 * k + a] = bc[a] + ((bq[a] + s * dq[a]) >> kFracBits) - 1;
            }
        }
    }
}

cudaError_t launch_debug_ray_cells(const ProjectParams& p, int i, int j, int staged, int32_t* cells, int max_samples,
                                   int32_t* count, cudaStream_t s) {
    gdrr_debug_ray_cells_kernel<<<1, kThreads, 0, s>>>(p, i, j, staged, cells, max_samples, count);
    return cudaGetLastError();
}

}  // namespace gdrr
