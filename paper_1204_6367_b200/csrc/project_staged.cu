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
// Roles.  A CTA is 8 CONSUMER warps (one ray per thread, 4 x 8 pixels per warp) and one PRODUCER
// warp.  Intervals are laid from the source, so all rays of the CTA are at the same interval
// index k and a chunk of kStageK indices is a thin curved slab of the beam.  The producer
// walks the chunks ahead of the consumers: it bounds the slab of chunk m by the positions of the
// tile's four CORNER rays at the chunk's first and last index (positions are linear in k, and
// the rays of a tile deviate from the bilinear blend of its corner rays by less than
// ProjectParams::hull_margin voxel: gdrr_api.cu derives the bound), waits until the stage
// is free (mbarrier `empty`, one arrival per consumer warp), and requests the box with ONE
// cp.async.bulk.tensor.3d whose completion flips mbarrier `full`.  A consumer warp waits for
// `full` of its chunk, samples it out of shared memory, and arrives on `empty`: the classic
// two-barrier ring, nothing else is shared between the warps inside the loop.
//
// The box has a fixed shape (kBX x kBY x kBZ quads: a tensor map fixes its box); a chunk whose
// bounds do not fit (other geometries) is sampled from global memory by the gather path's own
// routine, so the result never depends on the staging.  Quads of the box that lie outside the
// volume are zero-filled by the copy and never read by a ray that owns its sample.
// Row pitch kBX = 14 = 6 (mod 8) and slab pitch kBX kBY = 196 = 4 (mod 8): neighbouring quads
// fall in different 16-byte bank groups in every direction (profiles/r01_l1_model.md).
#include <cuda.h>

#include "packed_sampler.cuh"

namespace gdrr {

constexpr int kBoxElems = kBX * kBY * kBZ;        // 2156 quads = 34,496 B
constexpr int kStageElems = (kBoxElems + 7) / 8 * 8;  // stage pitch: a multiple of 128 B
constexpr unsigned kBoxBytes = kBoxElems * 16u;
constexpr int kConsumerWarps = kStageThreads / 32;
constexpr int kStageCtaThreads = kStageThreads + 32;  // + the producer warp
static_assert(kStageThreads % 128 == 0, "the lane -> pixel map below is 4 warps wide");

__device__ __forceinline__ unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

// mbarrier operations on the 32-bit shared-window address of the barrier (formed once per kernel: taking it anew at
// every use costs six instructions)
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// (try_wait has acquire semantics, arrive has release semantics, both at CTA scope: the PTX defaults)
__device__ __forceinline__ bool mbar_try_wait(unsigned bar, unsigned parity) {
    unsigned ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0u;
}
// A try_wait that fails returns after ~40 cycles (measured: the producer polled 88 times per wait), and a polling warp
// takes issue slots from the sampling warps: sleep between polls.  SLEEP_NS = 0: poll.
#ifndef GDRR_PRODUCER_SLEEP_NS
#define GDRR_PRODUCER_SLEEP_NS 128
#define GDRR_CONSUMER_SLEEP_NS 0
#endif
template <unsigned SLEEP_NS>
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    while (!mbar_try_wait(bar, parity)) {
        if (SLEEP_NS) __nanosleep(SLEEP_NS);
    }
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// box of the 3-D tensor (words along x, rows, slabs) at (c0, c1, c2) -> shared memory, completes on `bar`
__device__ __forceinline__ void tma_load_box(void* dst, const CUtensorMap* map, int c0, int c1, int c2, unsigned bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
        ::"r"(smem_addr(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(bar) : "memory");
}

// The quads of the staged boxes (2 stages), the rays' per-material sums (RayAcc), then the spectrum tables.
extern __shared__ __align__(128) uint4 s_box[];
constexpr int kAccBytes = 4 * kAccStride * (int)sizeof(float);

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
        if (act0) blend_sample<VW, !PRED>(a0, c0, fx, fy, fz, A);
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
            if (act1) blend_sample<VW, !PRED>(a1, c1, fx, fy, fz, A);
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
            blend_sample<VW, false>(a0, c0, fx0, fy0, fz0, A);
            blend_sample<VW, false>(a1, c1, fx1, fy1, fz1, A);
        }
    }
}

// CTA-shared bookkeeping of the staging ring
struct StageCtl {
    unsigned long long full[2];    // "the box of stage s has landed" (or: its chunk does not fit); 1 arrival + the copy's bytes
    unsigned long long empty[2];   // "every consumer warp has finished the chunk in stage s"; kConsumerWarps arrivals
    int lin[2];                    // stage s: element of cell (cx, cy, cz) = lin + (cz kBY + cy) kBX + cx
    int fit[2];                    // stage s holds the box of its chunk (else: gather from global memory)
    int krange[2];                 // smallest first / largest last+1 interval index of the CTA's rays
};

// SKEW (tests only, gdrr_debug_set_skew): warps are delayed by amounts keyed on their number and the chunk, so that the
// order in which they reach the barriers is forced through many interleavings; the result must not change by a bit.
template <bool SKEW>
__device__ __forceinline__ void skew_delay(unsigned key, unsigned mode) {
    if (SKEW) {
        const unsigned h = (key * 2654435761u) >> 27;                   // 0..31
        if (mode == 1u) __nanosleep(64u * h);                           // pseudo-random
        else if (mode == 2u) __nanosleep(400u * (key & 7u));            // the same warp always last
        else if (mode == 3u) __nanosleep((key & 8u) ? 3000u : 0u);      // the producer (key bit 3) late, consumers early
    }
}

template <int VW, bool SKEW>
__global__ void __launch_bounds__(kStageCtaThreads, GDRR_STAGE_CTAS)
gdrr_project_staged_kernel(const ProjectParams P, const __grid_constant__ CUtensorMap tmap) {
    __shared__ StageCtl ctl;
    float* s_acc = reinterpret_cast<float*>(s_box + 2 * kStageElems);
    float4* s_mu = reinterpret_cast<float4*>(s_box + 2 * kStageElems + kAccBytes / 16);
    float2* s_src = reinterpret_cast<float2*>(s_mu + P.n_energy);
    const unsigned bar_full = smem_addr(&ctl.full[0]), bar_empty = smem_addr(&ctl.empty[0]);     // [st]: + 8 st
    for (int e = threadIdx.x; e < P.n_energy; e += kStageCtaThreads) {
        s_mu[e] = P.mu_tab[e];
        s_src[e] = P.src_tab[e];
    }
    if (threadIdx.x == 0) {
        mbar_init(bar_full, 1);
        mbar_init(bar_full + 8u, 1);
        mbar_init(bar_empty, kConsumerWarps);
        mbar_init(bar_empty + 8u, kConsumerWarps);
        ctl.krange[0] = 0x7fffffff;
        ctl.krange[1] = (int)0x80000000;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    // (the warp number through a shuffle: the compiler then knows that the role branches below are warp-uniform)
    const int lane = threadIdx.x & 31, warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const bool producer = warp == kConsumerWarps;
    const int pl = blockIdx.z;
    // consumer: a warp is 4 (u) x 8 (v) pixels (thread_pixel_map), the CTA's tile kTileU x kStageTileV.
    // producer: lane -> (corner of the tile, axis, first / last index of a chunk); lanes 24..31 repeat lanes 12..19
    int i = blockIdx.x * kTileU + (warp & 3) * 4 + (lane & 3);
    int j = blockIdx.y * kStageTileV + (warp >> 2) * 8 + (lane >> 2);
    const int p_axis = (lane >> 2) % 3, p_last = lane >= 12 ? kStageK - 1 : 0;
    if (producer) {
        i = blockIdx.x * kTileU + ((lane & 1) ? kTileU - 1 : 0);
        j = blockIdx.y * kStageTileV + ((lane & 2) ? kStageTileV - 1 : 0);
    }
    const bool valid = !producer && i < P.g.nu && j < P.g.nv;

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
    const int c_begin = kmin < kmax ? kmin / kStageK : 0;
    const int nchunks = kmin < kmax ? (kmax - 1) / kStageK - c_begin + 1 : 0;

    if (producer) {
        // ---- the producer warp: bounds of chunk m from the corner rays, then the box request ----------------
        const double my_gs = p_axis == 0 ? gs[0] : p_axis == 1 ? gs[1] : gs[2];
        const double my_dg = p_axis == 0 ? dg[0] : p_axis == 1 ? dg[1] : dg[2];
        const double marg = p_axis == 0 ? P.hull_margin[0] : p_axis == 1 ? P.hull_margin[1] : P.hull_margin[2];
        for (int m = 0; m < nchunks; ++m) {
            const int st = m & 1;
            const double tk = (double)((c_begin + m) * kStageK + p_last) + 0.5;
            const double pos = fma(tk, my_dg, my_gs);
            const int lo = (int)floor(pos - marg), hi = (int)floor(pos + marg);
            int mn[3], mx[3];
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                mn[a] = __reduce_min_sync(0xffffffffu, p_axis == a ? lo : 0x7fffffff);
                mx[a] = __reduce_max_sync(0xffffffffu, p_axis == a ? hi : (int)0x80000000);
            }
            const bool fit = mx[0] - mn[0] + 1 <= kBX && mx[1] - mn[1] + 1 <= kBY && mx[2] - mn[2] + 2 <= kBZ;
            skew_delay<SKEW>(8u + (unsigned)m, P.debug_skew);
            // stage st is free once every consumer warp has finished chunk m - 2
            if (m >= 2) mbar_wait<GDRR_PRODUCER_SLEEP_NS>(bar_empty + 8u * st, (unsigned)((m >> 1) - 1) & 1u);
            if (lane == 0) {
                ctl.fit[st] = fit;
                // element of cell (cx, cy, cz) in the stage: lin + (cz kBY + cy) kBX + cx
                ctl.lin[st] = st * kStageElems - ((mn[2] * kBY + mn[1]) * kBX + mn[0]);
                // the phase of full[st] completes either way; its release / acquire orders fit and lin before their readers
                if (fit) {
                    mbar_arrive_expect_tx(bar_full + 8u * st, kBoxBytes);
                    tma_load_box(s_box + st * kStageElems, &tmap, 4 * mn[0], mn[1], mn[2], bar_full + 8u * st);
                } else {
                    mbar_arrive(bar_full + 8u * st);
                }
            }
            __syncwarp();
        }
        return;
    }

    // ---- the consumer warps ---------------------------------------------------------------------------------
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

    float acc[VW];
    RayAcc<VW> A;
    init_ray<VW>(A, s_acc + threadIdx.x);

    if (nchunks > 0) {
        ChunkWalk W;                                 // base position of the current chunk (packed_sampler.cuh)
        walk_init(gs, dg, c_begin, W);
        // chunks [m_lo, m_hi) are owned entirely by every lane of this warp (warp-uniform)
        const int first_full = (j0 + kStageK - 1) / kStageK, end_full = (j0 + n) / kStageK;
        const int m_lo = __reduce_max_sync(0xffffffffu, first_full) - c_begin;
        const int m_hi = __reduce_min_sync(0xffffffffu, end_full) - c_begin;

        for (int m = 0; m < nchunks; ++m) {
            const int st = m & 1;
            // chunk m: working copy of its base; then the base moves on to chunk m + 1
            const int wqx = W.qb[0] >> (kBaseBits - kFracBits), wqy = W.qb[1] >> (kBaseBits - kFracBits),
                      wqz = W.qb[2] >> (kBaseBits - kFracBits);
            const int bcx = W.cb[0], bcy = W.cb[1], bcz = W.cb[2];
            walk_advance(W);
            skew_delay<SKEW>((unsigned)(warp + 3 * m), P.debug_skew);
            mbar_wait<GDRR_CONSUMER_SLEEP_NS>(bar_full + 8u * st, (unsigned)(m >> 1) & 1u);      // box landed (or: chunk does not fit); fit / lin valid
            const bool all_mine = m >= m_lo && m < m_hi;
            const int r = (c_begin + m) * kStageK - j0;         // the chunk's first index in this ray's own count
            const unsigned rel = (unsigned)r;
            if (ctl.fit[st]) {
                const int idx0 = (bcz * kBY + bcy) * kBX + bcx + ctl.lin[st];
                if (all_mine) {
                    run_chunk_staged_pairs<VW>(S, wqx, wqy, wqz, idx0, A);
                } else if (__any_sync(0xffffffffu, r + kStageK > 0 && r < n)) {      // some lane has a sample in this chunk
                    run_chunk_staged<VW, true>(S, wqx, wqy, wqz, idx0, kStageK, rel, un, A);
                }
            } else {
                ChunkBase b;
                b.cx = bcx; b.cy = bcy; b.cz = bcz;
                b.qx = wqx; b.qy = wqy; b.qz = wqz;
                if (all_mine) run_chunk<VW, false>(S, b, kStageK, rel, un, A);
                else run_chunk<VW, true>(S, b, kStageK, rel, un, A);
            }
            // this warp is done with stage st
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_empty + 8u * st);
            flush_chunk<VW>(A);
        }
    }
    finish_ray<VW>(A, acc);

    if (valid) finish_pixel<VW>(P, s_mu, s_src, acc, P.g.step, pl, i, j);
}

template <int VW, bool SKEW>
static cudaError_t launch_staged_t(const ProjectParams& p, const CUtensorMap& map, cudaStream_t s) {
    dim3 grid((p.g.nu + kTileU - 1) / kTileU, (p.g.nv + kStageTileV - 1) / kStageTileV, p.g.proj_count);
    const size_t smem = 2 * (size_t)kStageElems * 16 + kAccBytes + (size_t)p.n_energy * (sizeof(float4) + sizeof(float2));
    // per device and cheap: set at every launch (the boxes alone exceed the 48 KB default)
    cudaError_t e = cudaFuncSetAttribute(gdrr_project_staged_kernel<VW, SKEW>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         2 * kStageElems * 16 + kAccBytes + 512 * 24 /* GDRR_MAX_ENERGIES bins */);
    if (e != cudaSuccess) return e;
    gdrr_project_staged_kernel<VW, SKEW><<<grid, kStageCtaThreads, smem, s>>>(p, map);
    return cudaGetLastError();
}

cudaError_t launch_project_staged(const ProjectParams& p, int vw, const void* tensor_map, cudaStream_t s) {
    const CUtensorMap& map = *reinterpret_cast<const CUtensorMap*>(tensor_map);
    if (p.debug_skew) {                         // tests only: forced warp orders
        if (vw == 1) return launch_staged_t<1, true>(p, map, s);
        if (vw == 2) return launch_staged_t<2, true>(p, map, s);
        return launch_staged_t<4, true>(p, map, s);
    }
    if (vw == 1) return launch_staged_t<1, false>(p, map, s);
    if (vw == 2) return launch_staged_t<2, false>(p, map, s);
    return launch_staged_t<4, false>(p, map, s);
}

}  // namespace gdrr
