// Steps a1-a7 fused, PACKED-QUAD layout, quads STAGED THROUGH SHARED MEMORY BY TMA.
//
// Why.  The gather kernel (project_packed.cu) saturates the L1 data pipe: a 16-byte warp-wide
// load costs 6.7 wavefronts instead of 4, because 1.3 of its sectors miss L1 (every quad is
// first touched once per CTA beam, and each missed sector is served by a wavefront of its own)
// and because of bank-group conflicts (profiles/r01_packed_kernel_ncu.md).  Here the quads a
// CTA's 16 x 16 beam crosses during kStageK consecutive interval indices are fetched ONCE, as
// one box of the device volume, by a bulk tensor copy (cp.async.bulk.tensor, TMA) straight
// into shared memory, double buffered; the sampler then reads shared memory, where a load
// never misses and the only cost above 4 wavefronts is bank conflicts.
//
// The box.  Intervals are laid from the source, so all rays of the CTA are at the same
// interval index k and a chunk of kStageK indices is a thin curved slab of the beam.  Per
// chunk every thread contributes the cells of its first and last sample of the chunk (the
// cells in between are bracketed by them: positions are linear in k) to a CTA-wide bounding
// box (one redux per warp, its lane 0 posts it with shared atomics and counts the warp in); the
// warp that posts LAST requests the box for chunk c + 1 while chunk c is sampled -- no CTA barrier in
// the loop: a warp that has posted has finished chunk c - 1, whose stage the new box overwrites, and
// goes on to chunk c; it waits only for its own chunk's box (mbarrier).  The box
// has a fixed shape (kBX x kBY x kBZ quads: a tensor map fixes its box); a chunk whose
// bounding box does not fit (other geometries) is sampled from global memory by the gather
// path's own routine, so the result never depends on the staging.
// Row pitch kBX = 14 = 6 (mod 8) and slab pitch kBX kBY = 196 = 4 (mod 8): neighbouring quads
// fall in different 16-byte bank groups in every direction (profiles/r01_l1_model.md).
#include <cuda.h>

#include "packed_sampler.cuh"

namespace gdrr {

constexpr int kStageK = 16;                       // interval indices per staged chunk
constexpr int kBoxElems = kBX * kBY * kBZ;        // 2156 quads = 34,496 B
constexpr int kStageElems = (kBoxElems + 7) / 8 * 8;  // stage pitch: a multiple of 128 B
constexpr unsigned kBoxBytes = kBoxElems * 16u;
constexpr int kBaseBits = 27;                     // fraction bits of a chunk's base position (5.27 fixed point)

__device__ __forceinline__ unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_addr(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_addr(bar)) : "memory");
}
// box of the 3-D tensor (words along x, rows, slabs) at (c0, c1, c2) -> shared memory, completes on `bar`
__device__ __forceinline__ void tma_load_box(void* dst, const CUtensorMap* map, int c0, int c1, int c2,
                                             unsigned long long* bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
        ::"r"(smem_addr(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(smem_addr(bar)) : "memory");
}

// The quads of the staged boxes (2 stages), then the spectrum tables.
extern __shared__ __align__(128) uint4 s_box[];

// `cnt` consecutive samples of a chunk out of the staged box: as run_chunk (packed_sampler.cuh),
// the element index is relative to the box and both slabs of a cell are read with one address.
template <int VW, bool PRED>
__device__ __forceinline__ void run_chunk_staged(const Sampler& S, int qx, int qy, int qz, int idx0, int cnt,
                                                 unsigned rel, unsigned un, RayAcc<VW>& A) {
    uint4 a0 = make_uint4(0, 0, 0, 0), c0 = a0, a1 = a0, c1 = a0;
    bool act0 = !PRED || rel < un;
    if (act0) {
        const int idx = sample_index(idx0, qx, qy, qz, kBX, kBX * kBY);
        a0 = s_box[idx];
        c0 = s_box[idx + kBX * kBY];
    }
    for (int s = 0; s < cnt; s += 2) {
        float fx = frac_float(qx, S.fmask, S.fone);
        float fy = frac_float(qy, S.fmask, S.fone);
        float fz = frac_float(qz, S.fmask, S.fone);
        qx += S.dqx; qy += S.dqy; qz += S.dqz;
        const bool more = !PRED || s + 1 < cnt;
        const bool act1 = more && (!PRED || rel + 1u < un);
        if (act1) {
            const int idx = sample_index(idx0, qx, qy, qz, kBX, kBX * kBY);
            a1 = s_box[idx];
            c1 = s_box[idx + kBX * kBY];
        }
        if (act0) blend_sample<VW, !PRED>(a0, c0, fx, fy, fz, A.cur, A.curm4, A.part);
        if (more) {
            fx = frac_float(qx, S.fmask, S.fone);
            fy = frac_float(qy, S.fmask, S.fone);
            fz = frac_float(qz, S.fmask, S.fone);
            qx += S.dqx; qy += S.dqy; qz += S.dqz;
            rel += 2u;
            act0 = (s + 2 < cnt) && (!PRED || rel < un);
            if (act0) {
                const int idx = sample_index(idx0, qx, qy, qz, kBX, kBX * kBY);
                a0 = s_box[idx];
                c0 = s_box[idx + kBX * kBY];
            }
            if (act1) blend_sample<VW, !PRED>(a1, c1, fx, fy, fz, A.cur, A.curm4, A.part);
        }
    }
}

// The common case (every lane owns all kStageK samples): samples are taken in PAIRS -- both cells are read,
// then one vote decides for the pair whether every lane is in pure cells of its running material (two
// blends added to the running sum, in sample order) or the pair goes sample by sample through
// blend_sample.  Same arithmetic and order as run_chunk_staged, one vote and branch per two samples.
template <int VW>
__device__ __forceinline__ void run_chunk_staged_pairs(const Sampler& S, int qx, int qy, int qz, int idx0,
                                                       RayAcc<VW>& A) {
#pragma unroll 2          // measured: 1, 2, 4 within 0.3%; 8 (and the general path out of line) -1%
    for (int s = 0; s < kStageK; s += 2) {
        const int i0 = sample_index(idx0, qx, qy, qz, kBX, kBX * kBY);
        const unsigned bx0 = frac_bits(qx, S.fmask, S.fone), by0 = frac_bits(qy, S.fmask, S.fone),
                       bz0 = frac_bits(qz, S.fmask, S.fone);
        qx += S.dqx; qy += S.dqy; qz += S.dqz;
        const int i1 = sample_index(idx0, qx, qy, qz, kBX, kBX * kBY);
        const uint4 a0 = s_box[i0], c0 = s_box[i0 + kBX * kBY];
        const uint4 a1 = s_box[i1], c1 = s_box[i1 + kBX * kBY];
        const unsigned bx1 = frac_bits(qx, S.fmask, S.fone), by1 = frac_bits(qy, S.fmask, S.fone),
                       bz1 = frac_bits(qz, S.fmask, S.fone);
        qx += S.dqx; qy += S.dqy; qz += S.dqz;
        // [1, 2) -> [0, 1) for both samples of the pair at once (FADD2)
        float fx0, fx1, fy0, fy1, fz0, fz1;
        sub_one2(bx0, bx1, fx0, fx1);
        sub_one2(by0, by1, fy0, fy1);
        sub_one2(bz0, bz1, fz0, fz1);
        bool fast = true;
        if (VW > 1) fast = __all_sync(0xffffffffu, ((((a0.x ^ A.curm4) | (a1.x ^ A.curm4)) & 7u) == 0u));
        if (fast) {
            A.cur += blend_cell(a0, c0, fx0, fy0, fz0);
            A.cur += blend_cell(a1, c1, fx1, fy1, fz1);
        } else {
            blend_sample<VW, false>(a0, c0, fx0, fy0, fz0, A.cur, A.curm4, A.part);
            blend_sample<VW, false>(a1, c1, fx1, fy1, fz1, A.cur, A.curm4, A.part);
        }
    }
}

// CTA-shared bookkeeping of the staging pipeline
struct StageCtl {
    unsigned long long bar[2];     // "box of stage s has landed"
    int bb[3][6];                  // bounding box of chunk m in bb[m % 3]: min x, y, z, max x, y, z (cells)
    int lin[2];                    // stage s: element of cell (cx, cy, cz) = lin + (cz kBY + cy) kBX + cx
    int fit[2];                    // stage s holds the box of its chunk (else: gather from global memory)
    int krange[2];                 // smallest first / largest last+1 interval index of the CTA's rays
    int arrived[3];                // warps that have put their share into bb[slot]
};

template <int VW>
__global__ void __launch_bounds__(kStageThreads, GDRR_STAGE_CTAS)
gdrr_project_staged_kernel(const ProjectParams P, const __grid_constant__ CUtensorMap tmap) {
    __shared__ StageCtl ctl;
    float4* s_mu = reinterpret_cast<float4*>(s_box + 2 * kStageElems);
    float2* s_src = reinterpret_cast<float2*>(s_mu + P.n_energy);
    for (int e = threadIdx.x; e < P.n_energy; e += kStageThreads) {
        s_mu[e] = P.mu_tab[e];
        s_src[e] = P.src_tab[e];
    }
    if (threadIdx.x == 0) {
        mbar_init(&ctl.bar[0], 1);
        mbar_init(&ctl.bar[1], 1);
        for (int m = 0; m < 3; ++m)
            for (int a = 0; a < 3; ++a) { ctl.bb[m][a] = 0x7fffffff; ctl.bb[m][3 + a] = (int)0x80000000; }
        ctl.krange[0] = 0x7fffffff;
        ctl.krange[1] = (int)0x80000000;
        ctl.arrived[0] = ctl.arrived[1] = ctl.arrived[2] = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    // a warp is 4 (u) x 8 (v) pixels (thread_pixel_map), the CTA's tile kTileU x kStageTileV
    const int lane = threadIdx.x & 31;
    const int i = blockIdx.x * kTileU + ((threadIdx.x >> 5) & 3) * 4 + (lane & 3);
    const int j = blockIdx.y * kStageTileV + (threadIdx.x >> 7) * 8 + (lane >> 2);
    const int pl = blockIdx.z;
    const bool valid = i < P.g.nu && j < P.g.nv;

    // ---- a1: ray setup (fp64) ------------------------------------------------
    int j0, n;
    Sampler S;
    double gs[3], dg[3];
    {
        Ray r;
        ray_setup(P.g, P.g.proj_begin + pl, min(i, P.g.nu - 1), min(j, P.g.nv - 1), r);
        if (!valid) r.n = 0;
        if (valid && P.ray_table) {
            const size_t pix = ((size_t)pl * P.g.nv + j) * P.g.nu + i;
            reinterpret_cast<int2*>(P.ray_table)[pix] = make_int2(r.j0, r.n);
        }
        index_line(P.g, r, gs, dg);
        j0 = r.j0;
        n = r.n;
    }
    S.dqx = __double2int_rn(dg[0] * 8388608.0);
    S.dqy = __double2int_rn(dg[1] * 8388608.0);
    S.dqz = __double2int_rn(dg[2] * 8388608.0);
    S.sy = P.v.stride_y;
    S.sz = P.v.stride_z;
    S.vol0 = reinterpret_cast<const uint4*>(P.v.vox);
    S.vol1 = reinterpret_cast<const uint4*>(P.v.vox1);
    S.fmask = P.frac_mask;
    S.fone = P.one_bits;
    const unsigned un = (unsigned)n;

    // interval range of the whole CTA: all its rays walk the same chunks of kStageK indices
    {
        const int wmin = __reduce_min_sync(0xffffffffu, n > 0 ? j0 : 0x7fffffff);
        const int wmax = __reduce_max_sync(0xffffffffu, n > 0 ? j0 + n : (int)0x80000000);
        if (lane == 0 && wmin < wmax) {
            atomicMin(&ctl.krange[0], wmin);
            atomicMax(&ctl.krange[1], wmax);
        }
    }
    __syncthreads();
    const int kmin = ctl.krange[0], kmax = ctl.krange[1];

    float acc[VW];
#pragma unroll
    for (int m = 0; m < VW; ++m) acc[m] = 0.f;
    RayAcc<VW> A;
    A.cur = 0.f;
    A.curm4 = 4u;

    if (kmin < kmax) {
        const int c_begin = kmin / kStageK;
        const int nchunks = (kmax - 1) / kStageK - c_begin + 1;

        // Chunk bases.  The position of a chunk's first sample is (cell cb, fraction qb in 2^-27 voxel); the
        // next chunk's is that plus D = round(kStageK dg 2^27), in integers.  The fp64 line of the ray is used
        // once, for chunk 0: the base then drifts by <= 2^-28 voxel per chunk (2^-19 over the 500 chunks of
        // the longest ray a 180 GB volume allows), and 12 registers of doubles do not live through the loop.
        // Inside a chunk the samples step by dq = round(dg 2^23) from the base's 23-bit fraction.
        int cb[3], qb[3], D[3];
        {
            const double tk = (double)(c_begin * kStageK) + 0.5;
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const double x = fma(tk, dg[a], gs[a]);
                const double f = floor(x);
                cb[a] = (int)f;
                qb[a] = (int)((x - f) * (double)(1 << kBaseBits));
                D[a] = __double2int_rn(dg[a] * (double)kStageK * (double)(1 << kBaseBits));
            }
        }
        // this ray's share of the bounding box of the chunk whose base is (cb, qb), first index kc -> ctl.bb[slot]
        auto contribute = [&](int kc, int slot) {
            const int lo = max(j0 - kc, 0), hi = min(j0 + n - kc, kStageK);
            int mn[3] = {0x7fffffff, 0x7fffffff, 0x7fffffff};
            int mx[3] = {(int)0x80000000, (int)0x80000000, (int)0x80000000};
            if (hi > lo) {                       // cells of the first and the last sample, exactly as the loop forms them
                const int dq[3] = {S.dqx, S.dqy, S.dqz};
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    const int q23 = qb[a] >> (kBaseBits - kFracBits);
                    const int c_lo = cb[a] + ((q23 + lo * dq[a]) >> kFracBits);
                    const int c_hi = cb[a] + ((q23 + (hi - 1) * dq[a]) >> kFracBits);
                    mn[a] = min(c_lo, c_hi);
                    mx[a] = max(c_lo, c_hi);
                }
            }
            // the warp's share, posted by lane 0; the warp that arrives last (its lane 0) gets `true`
            bool last = false;
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                mn[a] = __reduce_min_sync(0xffffffffu, mn[a]);
                mx[a] = __reduce_max_sync(0xffffffffu, mx[a]);
            }
            if (lane == 0) {
                // (PTX reductions: the compiler would wrap atomicMin / atomicMax in a second warp reduction; the
                // acq_rel counter orders the six before it and, in the warp that arrives last, the others' before its reads)
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    asm volatile("red.relaxed.cta.shared::cta.min.s32 [%0], %1;" ::"r"(smem_addr(&ctl.bb[slot][a])), "r"(mn[a]) : "memory");
                    asm volatile("red.relaxed.cta.shared::cta.max.s32 [%0], %1;" ::"r"(smem_addr(&ctl.bb[slot][3 + a])), "r"(mx[a]) : "memory");
                }
                unsigned before;
                asm volatile("atom.acq_rel.cta.shared::cta.add.u32 %0, [%1], 1;" : "=r"(before) : "r"(smem_addr(&ctl.arrived[slot])) : "memory");
                last = before == (unsigned)(kThreads / 32 - 1);
            }
            return last;
        };
        // thread 0: request the box of chunk m into stage m & 1 if it fits
        auto issue = [&](int m, int slot) {
            int* bb = ctl.bb[slot];
            const int st = m & 1;
            const int b0 = bb[0], b1 = bb[1], b2 = bb[2];
            const bool fit = b0 <= bb[3] && bb[3] - b0 + 1 <= kBX && bb[4] - b1 + 1 <= kBY && bb[5] - b2 + 2 <= kBZ;
            // the slot is free for the chunk three ahead (no warp reaches that one before the box requested here
            // and the next one have been waited for)
            for (int a = 0; a < 3; ++a) { bb[a] = 0x7fffffff; bb[3 + a] = (int)0x80000000; }
            ctl.arrived[slot] = 0;
            ctl.fit[st] = fit;
            // element of cell (cx, cy, cz) in the stage: lin + (cz kBY + cy) kBX + cx
            ctl.lin[st] = st * kStageElems - ((b2 * kBY + b1) * kBX + b0);
            // the phase of bar[st] completes either way and orders fit / lin before their readers
            if (fit) {
                mbar_arrive_expect_tx(&ctl.bar[st], kBoxBytes);
                tma_load_box(s_box + st * kStageElems, &tmap, 4 * b0, b1, b2, &ctl.bar[st]);
            } else {
                mbar_arrive(&ctl.bar[st]);
            }
        };

        // No CTA barrier in the loop: a warp posts its share of the next chunk's box (it has then finished the
        // chunk before, whose stage the new box overwrites) and goes on; whichever warp posts last requests the box.
        if (contribute(c_begin * kStageK, 0)) issue(0, 0);
        unsigned phases = 0u;                    // bit st: parity of the next completion of bar[st]
        int slot1 = 1;                           // bounding-box slot of chunk m + 1 (m % 3 rotation)

        for (int m = 0; m < nchunks; ++m) {
            const int st = m & 1;
            // chunk m: working copy of its base; then the base moves on to chunk m + 1
            const int kc = (c_begin + m) * kStageK;
            const int wqx = qb[0] >> (kBaseBits - kFracBits), wqy = qb[1] >> (kBaseBits - kFracBits),
                      wqz = qb[2] >> (kBaseBits - kFracBits);
            const int rel_cell = (cb[2] * kBY + cb[1]) * kBX + cb[0];
            int dc[3] = {0, 0, 0};               // cells the base advanced by (the gather fallback wants chunk m's cell)
            if (m + 1 < nchunks) {
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    const int q = qb[a] + D[a];
                    dc[a] = q >> kBaseBits;
                    cb[a] += dc[a];
                    qb[a] = q & ((1 << kBaseBits) - 1);
                }
                if (contribute(kc + kStageK, slot1)) issue(m + 1, slot1);
            }
            slot1 = slot1 == 2 ? 0 : slot1 + 1;

            const unsigned rel = (unsigned)(kc - j0);
            const bool mine = rel < un && rel + (unsigned)kStageK <= un;     // this lane owns the whole chunk
            const bool all_mine = __all_sync(0xffffffffu, mine);
#pragma unroll
            for (int k = 0; k < VW; ++k) A.part[k] = 0.f;

            mbar_wait(&ctl.bar[st], (phases >> st) & 1u);      // box landed (or: chunk does not fit); fit / lin valid
            phases ^= 1u << st;
            if (ctl.fit[st]) {
                const int idx0 = rel_cell + ctl.lin[st];
                if (all_mine) run_chunk_staged_pairs<VW>(S, wqx, wqy, wqz, idx0, A);
                else run_chunk_staged<VW, true>(S, wqx, wqy, wqz, idx0, kStageK, rel, un, A);
            } else {
                ChunkBase b;
                b.cx = cb[0] - dc[0]; b.cy = cb[1] - dc[1]; b.cz = cb[2] - dc[2];
                b.qx = wqx; b.qy = wqy; b.qz = wqz;
                if (all_mine) run_chunk<VW, false>(S, b, kStageK, rel, un, A);
                else run_chunk<VW, true>(S, b, kStageK, rel, un, A);
            }
            add_routed<VW>(A.part, (int)(A.curm4 & 3u), A.cur);
            A.cur = 0.f;
#pragma unroll
            for (int k = 0; k < VW; ++k) acc[k] += A.part[k];
        }
    }

    if (valid) finish_pixel<VW>(P, s_mu, s_src, acc, P.g.step, pl, i, j);
}

template <int VW>
static cudaError_t launch_staged_t(const ProjectParams& p, const CUtensorMap& map, cudaStream_t s) {
    dim3 grid((p.g.nu + kTileU - 1) / kTileU, (p.g.nv + kStageTileV - 1) / kStageTileV, p.g.proj_count);
    const size_t smem = 2 * (size_t)kStageElems * 16 + (size_t)p.n_energy * (sizeof(float4) + sizeof(float2));
    // per device and cheap: set at every launch (the boxes alone exceed the 48 KB default)
    cudaError_t e = cudaFuncSetAttribute(gdrr_project_staged_kernel<VW>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         2 * kStageElems * 16 + 512 * 24 /* GDRR_MAX_ENERGIES bins */);
    if (e != cudaSuccess) return e;
    gdrr_project_staged_kernel<VW><<<grid, kStageThreads, smem, s>>>(p, map);
    return cudaGetLastError();
}

cudaError_t launch_project_staged(const ProjectParams& p, int vw, const void* tensor_map, cudaStream_t s) {
    const CUtensorMap& map = *reinterpret_cast<const CUtensorMap*>(tensor_map);
    if (vw == 1) return launch_staged_t<1>(p, map, s);
    if (vw == 2) return launch_staged_t<2>(p, map, s);
    return launch_staged_t<4>(p, map, s);
}

}  // namespace gdrr
