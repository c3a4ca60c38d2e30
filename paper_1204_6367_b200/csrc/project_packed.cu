// Steps a1-a7 fused, PACKED-QUAD layout (GDRR_LAYOUT_PACKED_QUAD): the fast path.
//
// Layout.  A voxel is ONE 32-bit word: fp32 rho whose three lowest mantissa
// bits carry tags (n_materials > 1): bits 0-1 the material index, bit 2 (first
// word of an element only) "all 8 corners of this cell have this material".
// Element (ix, iy, iz) of the device volume is the 2x2 quad of words
// {(ix,iy), (ix,iy+1), (ix+1,iy), (ix+1,iy+1)} of slab iz, stored for EVERY
// (ix, iy) (quads overlap, 16 B per voxel).  A sample needs two 16-byte loads
// (slabs iz and iz+1).
//
// What bounds the gather (profiles/r01_l1_model.md, measured on B200): a 16-byte
// warp-wide load is served in 4 phases of 8 lanes; inside a phase, distinct
// elements whose index is equal mod 8 (same 16-byte bank group of the L1 data
// RAM) serialise, whatever line they are in; the tag stage takes 4 lines per
// cycle.  So (1) the lanes of a warp must sample the SAME interval index k at
// the same time (intervals are laid from the source, so equal k is a sphere
// around the source and the warp's footprint stays a compact 2-D patch; starting
// every ray at its own j0 spreads the warp over up to 8 steps of depth), and
// (2) neighbouring elements must differ mod 8 in every direction: elements are
// stored linearly with the row stride = 3 and the slab stride = 4 (mod 8).
//
// Material routing.  In a segmented volume almost every cell is pure (98.8% of
// C3's cells), so the common path is one scalar tri-linear blend added to a
// running sum that is routed to its material only when the material changes;
// cells with mixed corners take a slower branch that routes each weighted
// corner.  Both give the same value.
//
// The words are used as floats as they are (|stored - rho| <= 11 ulp, DESIGN.md
// Q24); the library is compiled with -ftz=true so that rho = 0 tagged with a
// material (a denormal bit pattern) contributes exactly 0.
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

// UNI: every lane of the warp is here (unpredicated chunk): vote, so that the common case "all lanes
// in a pure cell of their running material" is a warp-uniform branch without reconvergence overhead.
template <int VW, bool UNI>
__device__ __forceinline__ void blend_sample(const uint4& a, const uint4& c, float fx, float fy, float fz,
                                             float& cur, unsigned& curm4, float (&part)[VW]) {
    bool fast = true;
    if (VW > 1) fast = (a.x & 7u) == curm4;        // pure cell of the running material
    if (VW > 1 && UNI) {
        if (__all_sync(0xffffffffu, fast)) {
            cur += blend_cell(a, c, fx, fy, fz);
            return;
        }
    }
    if (fast) {
        cur += blend_cell(a, c, fx, fy, fz);
    } else {
        // mixed cell, or a pure cell of another material: route every weighted corner
        const float gx = 1.f - fx, gy = 1.f - fy, gz = 1.f - fz;
        const float w00 = gy * gz, w10 = fy * gz, w01 = gy * fz, w11 = fy * fz;
        // w<y><z>; words (x0y0, x0y1, x1y0, x1y1)
        add_routed<VW>(part, (int)(a.x & 3u), gx * w00 * __uint_as_float(a.x));
        add_routed<VW>(part, (int)(a.y & 3u), gx * w10 * __uint_as_float(a.y));
        add_routed<VW>(part, (int)(a.z & 3u), fx * w00 * __uint_as_float(a.z));
        add_routed<VW>(part, (int)(a.w & 3u), fx * w10 * __uint_as_float(a.w));
        add_routed<VW>(part, (int)(c.x & 3u), gx * w01 * __uint_as_float(c.x));
        add_routed<VW>(part, (int)(c.y & 3u), gx * w11 * __uint_as_float(c.y));
        add_routed<VW>(part, (int)(c.z & 3u), fx * w01 * __uint_as_float(c.z));
        add_routed<VW>(part, (int)(c.w & 3u), fx * w11 * __uint_as_float(c.w));
        // the running sum follows the material the ray is now in
        const unsigned m4 = (c.w & 3u) | 4u;
        if (m4 != curm4) {
            add_routed<VW>(part, (int)(curm4 & 3u), cur);
            cur = 0.f;
            curm4 = m4;
        }
    }
}

// element of the sample at in-chunk fixed-point position q (idx0 = element of the chunk's base cell)
__device__ __forceinline__ int sample_index(int idx0, int qx, int qy, int qz, int sy, int sz) {
    return idx0 + (qz >> kFracBits) * sz + (qy >> kFracBits) * sy + (qx >> kFracBits);
}

// State of one ray while it is sampled.
template <int VW>
struct RayAcc {
    float part[VW];     // per-material partial sums of the current chunk
    float cur;          // running sum of pure cells of material curm4 & 3
    unsigned curm4;     // 4 | material
};

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
        if (act0) blend_sample<VW, !PRED>(a0, c0, fx, fy, fz, A.cur, A.curm4, A.part);
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
            if (act1) blend_sample<VW, !PRED>(a1, c1, fx, fy, fz, A.cur, A.curm4, A.part);
        }
    }
}

template <int VW>
__global__ void __launch_bounds__(kThreads, 4)
gdrr_project_packed_kernel(const ProjectParams P) {
    // the ray's line in index space (6 doubles) is needed once per chunk only: keep it in
    // shared memory, not in 12 registers of the sampling loop
    __shared__ double s_line[6][kThreads];
    float4* s_mu;
    float2* s_src;
    load_tables(P, s_mu, s_src);

    int i, j;
    thread_pixel_map(i, j);
    const int pl = blockIdx.z;
    // lanes outside the detector stay in the warp (the loop below is warp-synchronous) with n = 0
    const bool valid = i < P.g.nu && j < P.g.nv;

    // ---- a1: ray setup (fp64) ------------------------------------------------
    int j0, n;
    Sampler S;
    {
        Ray r;
        ray_setup(P.g, P.g.proj_begin + pl, min(i, P.g.nu - 1), min(j, P.g.nv - 1), r);
        if (!valid) r.n = 0;
        if (valid && P.ray_table) {
            const size_t pix = ((size_t)pl * P.g.nv + j) * P.g.nu + i;
            reinterpret_cast<int2*>(P.ray_table)[pix] = make_int2(r.j0, r.n);
        }
        double gs[3], dg[3];
        index_line(P.g, r, gs, dg);
        S.dqx = __double2int_rn(dg[0] * 8388608.0);
        S.dqy = __double2int_rn(dg[1] * 8388608.0);
        S.dqz = __double2int_rn(dg[2] * 8388608.0);
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            s_line[a][threadIdx.x] = gs[a];
            s_line[3 + a][threadIdx.x] = dg[a];
        }
        j0 = r.j0;
        n = r.n;
    }
    S.sy = P.v.stride_y;
    S.sz = P.v.stride_z;
    S.vol0 = reinterpret_cast<const uint4*>(P.v.vox);
    S.vol1 = reinterpret_cast<const uint4*>(P.v.vox1);
    S.fmask = P.frac_mask;
    S.fone = P.one_bits;

    // Interval indices k are counted from the source (reading Q9), so all lanes of the
    // warp walk the same k: the warp's samples lie on a sphere around the source.
    const int kmin = __reduce_min_sync(0xffffffffu, n > 0 ? j0 : 0x7fffffff);
    const int kmax = __reduce_max_sync(0xffffffffu, n > 0 ? j0 + n : (int)0x80000000);
    const unsigned un = (unsigned)n;
    const int CH = P.chunk;

    // ---- a2-a4: sampling -------------------------------------------------------
    float acc[VW];
#pragma unroll
    for (int m = 0; m < VW; ++m) acc[m] = 0.f;
    RayAcc<VW> A;
    A.cur = 0.f;
    A.curm4 = 4u;

    for (int kc = (kmin / CH) * CH; kc < kmax; kc += CH) {
        const int s0 = max(kmin - kc, 0);
        const int cnt = min(kmax - kc, CH) - s0;
        double gs[3], dg[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            gs[a] = s_line[a][threadIdx.x];
            dg[a] = s_line[3 + a][threadIdx.x];
        }
        const ChunkBase b = chunk_base(gs, dg, kc + s0);
        const unsigned rel = (unsigned)(kc + s0 - j0);
#pragma unroll
        for (int m = 0; m < VW; ++m) A.part[m] = 0.f;

        const bool mine = rel < un && rel + (unsigned)cnt <= un;         // this lane owns the whole chunk
        if (__all_sync(0xffffffffu, mine) && !(cnt & 1))
            run_chunk<VW, false>(S, b, cnt, rel, un, A);
        else
            run_chunk<VW, true>(S, b, cnt, rel, un, A);

        add_routed<VW>(A.part, (int)(A.curm4 & 3u), A.cur);
        A.cur = 0.f;
#pragma unroll
        for (int m = 0; m < VW; ++m) acc[m] += A.part[m];
    }

    if (valid) finish_pixel<VW>(P, s_mu, s_src, acc, P.g.step, pl, i, j);
}

template <int VW>
static cudaError_t launch_packed_t(const ProjectParams& p, cudaStream_t s) {
    dim3 grid((p.g.nu + kTileU - 1) / kTileU, (p.g.nv + kTileV - 1) / kTileV, p.g.proj_count);
    const size_t smem = (size_t)p.n_energy * (sizeof(float4) + sizeof(float2));
    gdrr_project_packed_kernel<VW><<<grid, kThreads, smem, s>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_project_packed(const ProjectParams& p, int vw, cudaStream_t s) {
    if (vw == 1) return launch_packed_t<1>(p, s);
    if (vw == 2) return launch_packed_t<2>(p, s);
    return launch_packed_t<4>(p, s);
}

}  // namespace gdrr
