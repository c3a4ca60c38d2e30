// Device pieces of the packed-quad sampler shared by its two kernels: project_packed.cu (quads
// gathered from global memory through L1) and project_staged.cu (quads staged through shared memory
// by TMA).  Layout, tags and the measured L1 model: see the header of project_packed.cu.
#pragma once
#include "project_common.cuh"

namespace gdrr {


template <int VW>
__device__ __forceinline__ void add_routed(float (&part)[VW], int m, float v) {
#pragma unroll
    for (int k = 0; k < VW; ++k) part[k] += (m == k) ? v : 0.f;
}

__device__ __forceinline__ float lerp(float a, float b, float t) { return fmaf(t, b - a, a); }

// Packed fp32 pairs (sm_100 FADD2 / FFMA2: two fp32 lanes per instruction, same rounding as the
// scalar forms; .ftz as the rest of the library).
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(unsigned lo, unsigned hi) {
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "r"(lo), "r"(hi));
    return r;
}
__device__ __forceinline__ f32x2 bcast2(float v) {
    f32x2 r;
    asm("mov.b64 %0, {%1, %1};" : "=l"(r) : "f"(v));
    return r;
}
__device__ __forceinline__ f32x2 lerp2(f32x2 a, f32x2 b, f32x2 t) {       // a + t (b - a), per lane
    f32x2 d, r;
    asm("sub.ftz.f32x2 %0, %1, %2;" : "=l"(d) : "l"(b), "l"(a));
    asm("fma.rn.ftz.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(t), "l"(d), "l"(a));
    return r;
}
// Tri-linear blend of one cell.  Words of a quad: (x0y0, x0y1, x1y0, x1y1), so that the two
// x-lerps of a slab are one packed lerp between its register pairs, the two z-lerps another.
__device__ __forceinline__ float blend_cell(const uint4& a, const uint4& c, float fx, float fy, float fz) {
    const f32x2 tx = bcast2(fx), tz = bcast2(fz);
    const f32x2 va = lerp2(pack2(a.x, a.y), pack2(a.z, a.w), tx);       // slab iz:     (y0, y1) at x
    const f32x2 vc = lerp2(pack2(c.x, c.y), pack2(c.z, c.w), tx);       // slab iz + 1
    const f32x2 v = lerp2(va, vc, tz);                                  // (y0, y1) at (x, z)
    float y0, y1;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(y0), "=f"(y1) : "l"(v));
    return lerp(y0, y1, fy);
}

// (q & mask) | one in a single LOP3; mask and one arrive as kernel parameters so
// that they live in registers instead of being split into two immediate ops.
__device__ __forceinline__ float frac_float(int q, unsigned mask, unsigned one) {
    unsigned o;
    asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(o) : "r"(q), "r"(mask), "r"(one));
    return __uint_as_float(o) - 1.f;
}

// The same in two steps, for the pair loop of the staged sampler: bits of 1 + fraction, then
// (1 + f0, 1 + f1) - (1, 1) as one packed add.
__device__ __forceinline__ unsigned frac_bits(int q, unsigned mask, unsigned one) {
    unsigned o;
    asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(o) : "r"(q), "r"(mask), "r"(one));
    return o;
}
__device__ __forceinline__ void sub_one2(unsigned b0, unsigned b1, float& f0, float& f1) {
    f32x2 r;
    asm("add.ftz.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pack2(b0, b1)), "l"(pack2(0xBF800000u, 0xBF800000u)));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(f0), "=f"(f1) : "l"(r));
}

// thread -> pixel: a warp is 4 (u) x 8 (v) pixels, so that a load phase (8 consecutive lanes) is a
// compact 4 x 2 patch of rays; the CTA's 16 x 16 tile is 4 x 2 warps.
__device__ __forceinline__ void thread_pixel_map(int& i, int& j) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    i = blockIdx.x * kTileU + (warp & 3) * 4 + (lane & 3);
    j = blockIdx.y * kTileV + (warp >> 2) * 8 + (lane >> 2);
}

// Element index of cell (cx, cy, cz): linear, strides sy = 3 and sz = 4 (mod 8).
__device__ __forceinline__ int elem_index(int cx, int cy, int cz, int sy, int sz) {
    return cz * sz + cy * sy + cx;
}

// State of one ray while it is sampled.  Three levels of sums keep the fp32 accumulation short and the registers few:
// `cur` (this chunk's pure cells of the running material), `run` (the ray's total for the running material since it
// last changed), and the ray's per-material totals of everything else (mixed cells, closed runs) in SHARED memory:
// slot[m * kAccStride] is this thread's sum for material m (its own bank; only this thread touches it).
constexpr int kAccStride = kThreads;
template <int VW>
struct RayAcc {
    float cur;          // this chunk's sum of pure cells of material curm4 & 3
    float run;          // the same over the earlier chunks since the running material last changed
    unsigned curm4;     // 4 | running material
    float* slot;        // shared memory: slot[m * kAccStride] += values routed to material m
};

template <int VW>
__device__ __forceinline__ void route(RayAcc<VW>& A, unsigned m, float v) {
    A.slot[m * kAccStride] += v;
}

// The running sum moves to material m4 (4 | material): what it held goes to its old material.
template <int VW>
__device__ __forceinline__ void switch_material(RayAcc<VW>& A, unsigned m4) {
    route<VW>(A, A.curm4 & 3u, A.cur + A.run);
    A.cur = 0.f;
    A.run = 0.f;
    A.curm4 = m4;
}

// A cell that is not a pure cell of the running material; v = blend_cell(a, c, fx, fy, fz) of all 8 words.
// Tags of the first element a (volume_layout.cu): a.x bit 2 "all 8 corners have the material of a.x"; a.y bit 2 "the 8
// corners have exactly two materials", the second one in (a.w bit 2, a.z bit 2).
template <int VW>
__device__ __forceinline__ void blend_general(const uint4& a, const uint4& c, float fx, float fy, float fz, float v,
                                              RayAcc<VW>& A) {
    // (the two-material test comes first: in a noisy volume it is what most lanes that get here need, and the arms
    // of this chain are short enough for ptxas to predicate, so a later arm costs every lane of an earlier one nothing)
    const unsigned p = a.x & 3u;
    if (a.y & 4u) {
        // two materials p and q: one more blend of the corners of material p alone (the others as 0), the rest is q's
        uint4 ma, mc;
        ma.x = a.x;
        ma.y = ((a.y ^ p) & 3u) ? 0u : a.y;
        ma.z = ((a.z ^ p) & 3u) ? 0u : a.z;
        ma.w = ((a.w ^ p) & 3u) ? 0u : a.w;
        mc.x = ((c.x ^ p) & 3u) ? 0u : c.x;
        mc.y = ((c.y ^ p) & 3u) ? 0u : c.y;
        mc.z = ((c.z ^ p) & 3u) ? 0u : c.z;
        mc.w = ((c.w ^ p) & 3u) ? 0u : c.w;
        const float vp = blend_cell(ma, mc, fx, fy, fz);
        const unsigned q = ((a.z >> 2) & 1u) | ((a.w >> 1) & 2u);
        route<VW>(A, p, vp);
        route<VW>(A, q, v - vp);
    } else if (a.x & 4u) {
        // pure cell of another material: the running sum moves there
        switch_material<VW>(A, a.x & 7u);
        A.cur = v;
    } else {
        // three or four materials: route every weighted corner
        const float gx = 1.f - fx, gy = 1.f - fy, gz = 1.f - fz;
        const float w00 = gy * gz, w10 = fy * gz, w01 = gy * fz, w11 = fy * fz;
        // w<y><z>; words (x0y0, x0y1, x1y0, x1y1)
        route<VW>(A, a.x & 3u, gx * w00 * __uint_as_float(a.x));
        route<VW>(A, a.y & 3u, gx * w10 * __uint_as_float(a.y));
        route<VW>(A, a.z & 3u, fx * w00 * __uint_as_float(a.z));
        route<VW>(A, a.w & 3u, fx * w10 * __uint_as_float(a.w));
        route<VW>(A, c.x & 3u, gx * w01 * __uint_as_float(c.x));
        route<VW>(A, c.y & 3u, gx * w11 * __uint_as_float(c.y));
        route<VW>(A, c.z & 3u, fx * w01 * __uint_as_float(c.z));
        route<VW>(A, c.w & 3u, fx * w11 * __uint_as_float(c.w));
    }
    // (the running material changes only at a PURE cell of another material: following the corners of mixed cells makes
    // it flip at every sample of a noisy volume, and every flip is a routed sum and a slow next sample)
}

// One sample.  UNI: every lane of the warp is here (unpredicated chunk): vote, so that the common case "all lanes
// in a pure cell of their running material" is a warp-uniform branch without reconvergence overhead.
template <int VW, bool UNI>
__device__ __forceinline__ void blend_sample(const uint4& a, const uint4& c, float fx, float fy, float fz,
                                             RayAcc<VW>& A) {
    const float v = blend_cell(a, c, fx, fy, fz);
    if (VW == 1) {
        A.cur += v;
        return;
    }
    const bool fast = (a.x & 7u) == A.curm4;        // pure cell of the running material
    if (UNI) {
        if (__all_sync(0xffffffffu, fast)) {
            A.cur += v;
            return;
        }
    }
    if (fast) A.cur += v;
    else blend_general<VW>(a, c, fx, fy, fz, v, A);
}

// End of a chunk: the chunk's sum moves up one level (see RayAcc).
template <int VW>
__device__ __forceinline__ void flush_chunk(RayAcc<VW>& A) {
    A.run += A.cur;
    A.cur = 0.f;
}

// `slot`: this thread's first slot of a [4][kAccStride] float array in shared memory (not needed for one material).
template <int VW>
__device__ __forceinline__ void init_ray(RayAcc<VW>& A, float* slot) {
    A.cur = 0.f;
    A.run = 0.f;
    A.curm4 = 4u;
    A.slot = slot;
    if (VW > 1) {
#pragma unroll
        for (int k = 0; k < 4; ++k) slot[k * kAccStride] = 0.f;
    }
}

// End of the ray: the per-material totals, with the running material's total added to its own.
template <int VW>
__device__ __forceinline__ void finish_ray(RayAcc<VW>& A, float (&acc)[VW]) {
    if (VW == 1) {
        acc[0] = A.run;
        return;
    }
    route<VW>(A, A.curm4 & 3u, A.run);
#pragma unroll
    for (int k = 0; k < VW; ++k) acc[k] = A.slot[k * kAccStride];
}

// element of the sample at in-chunk fixed-point position q (idx0 = element of the chunk's base cell)
__device__ __forceinline__ int sample_index(int idx0, int qx, int qy, int qz, int sy, int sz) {
    return idx0 + (qz >> kFracBits) * sz + (qy >> kFracBits) * sy + (qx >> kFracBits);
}

struct Sampler {
    const uint4* __restrict__ vol0;     // slab iz
    const uint4* __restrict__ vol1;     // slab iz + 1
    int sy, sz;
    int dqx, dqy, dqz;
    unsigned fmask, fone;
};

// `cnt` consecutive samples of a chunk.  PRED = false: every lane of the warp owns all of
// them and cnt is even (the common case); PRED = true: sample s is this ray's iff
// rel + s < un (first and last chunk of the warp).  Two register buffers: the loads of
// sample s + 1 are in flight while sample s is blended.
template <int VW, bool PRED>
__device__ __forceinline__ void run_chunk(const Sampler& S, const ChunkBase& b, int cnt, unsigned rel, unsigned un,
                                          RayAcc<VW>& A) {
    int qx = b.qx, qy = b.qy, qz = b.qz;
    const int idx0 = elem_index(b.cx, b.cy, b.cz, S.sy, S.sz);
    uint4 a0 = make_uint4(0, 0, 0, 0), c0 = a0, a1 = a0, c1 = a0;
    bool act0 = !PRED || rel < un;
    if (act0) {
        const int idx = sample_index(idx0, qx, qy, qz, S.sy, S.sz);
        a0 = __ldg(S.vol0 + idx);
        c0 = __ldg(S.vol1 + idx);
    }
    for (int s = 0; s < cnt; s += 2) {
        float fx = frac_float(qx, S.fmask, S.fone);
        float fy = frac_float(qy, S.fmask, S.fone);
        float fz = frac_float(qz, S.fmask, S.fone);
        qx += S.dqx; qy += S.dqy; qz += S.dqz;
        const bool more = !PRED || s + 1 < cnt;                  // warp-uniform
        const bool act1 = more && (!PRED || rel + 1u < un);
        if (act1) {
            const int idx = sample_index(idx0, qx, qy, qz, S.sy, S.sz);
            a1 = __ldg(S.vol0 + idx);
            c1 = __ldg(S.vol1 + idx);
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
                const int idx = sample_index(idx0, qx, qy, qz, S.sy, S.sz);
                a0 = __ldg(S.vol0 + idx);
                c0 = __ldg(S.vol1 + idx);
            }
            if (act1) blend_sample<VW, !PRED>(a1, c1, fx, fy, fz, A);
        }
    }
}

// Chunk bases of the staged sampler.  The position of a chunk's first sample is (cell cb, fraction qb in 2^-27 voxel);
// the next chunk's is that plus D = round(kStageK dg 2^27), in integers.  The fp64 line of the ray is used once, for the
// CTA's first chunk: the base then drifts by <= 2^-28 voxel per chunk (2^-19 over the 500 chunks of the longest ray a
// 180 GB volume allows), and 12 registers of doubles do not live through the loop.  Inside a chunk the samples step by
// dq = round(dg 2^23) from the base's 23-bit fraction.
constexpr int kStageK = 16;                       // interval indices per staged chunk
constexpr int kBaseBits = 27;                     // fraction bits of a chunk's base position (5.27 fixed point)
struct ChunkWalk {
    int cb[3], qb[3], D[3];
};
__device__ __forceinline__ void walk_init(const double (&gs)[3], const double (&dg)[3], int first_chunk, ChunkWalk& W) {
    const double tk = (double)(first_chunk * kStageK) + 0.5;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double x = fma(tk, dg[a], gs[a]);
        const double f = floor(x);
        W.cb[a] = (int)f;
        W.qb[a] = (int)((x - f) * (double)(1 << kBaseBits));
        W.D[a] = __double2int_rn(dg[a] * (double)kStageK * (double)(1 << kBaseBits));
    }
}
__device__ __forceinline__ void walk_advance(ChunkWalk& W) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const int q = W.qb[a] + W.D[a];
        W.cb[a] += q >> kBaseBits;
        W.qb[a] = q & ((1 << kBaseBits) - 1);
    }
}

// The unpredicated chunk in PAIRS (as the staged sampler's pair loop): both cells of two consecutive samples are
// requested, one vote decides for the pair, the fractions come from packed subtractions.
template <int VW>
__device__ __forceinline__ void run_chunk_pairs(const Sampler& S, const ChunkBase& b, int cnt, RayAcc<VW>& A) {
    int qx = b.qx, qy = b.qy, qz = b.qz;
    const int idx0 = elem_index(b.cx, b.cy, b.cz, S.sy, S.sz);
#pragma unroll 2
    for (int s = 0; s < cnt; s += 2) {
        const int i0 = sample_index(idx0, qx, qy, qz, S.sy, S.sz);
        const unsigned bx0 = frac_bits(qx, S.fmask, S.fone), by0 = frac_bits(qy, S.fmask, S.fone),
                       bz0 = frac_bits(qz, S.fmask, S.fone);
        qx += S.dqx; qy += S.dqy; qz += S.dqz;
        const int i1 = sample_index(idx0, qx, qy, qz, S.sy, S.sz);
        const uint4 a0 = __ldg(S.vol0 + i0), c0 = __ldg(S.vol1 + i0);
        const uint4 a1 = __ldg(S.vol0 + i1), c1 = __ldg(S.vol1 + i1);
        const unsigned bx1 = frac_bits(qx, S.fmask, S.fone), by1 = frac_bits(qy, S.fmask, S.fone),
                       bz1 = frac_bits(qz, S.fmask, S.fone);
        qx += S.dqx; qy += S.dqy; qz += S.dqz;
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

}  // namespace gdrr
