// Steps a1-a7 fused, PACKED-QUAD layout (GDRR_LAYOUT_PACKED_QUAD): the fast path.
//
// Why this layout.  ncu on the one-hot float4 kernel (profiles/r01_v1_onehot.md):
// l1tex data-pipe wavefronts at 95% of peak, 10.2 wavefronts per 16-byte
// warp-wide load and 8 such loads per sample -- the kernel is bound by L1
// wavefronts, not by bytes, DRAM or issue slots.  So the lever is wavefronts
// per sample.  Here a voxel is ONE 32-bit word: fp32 rho whose two lowest
// mantissa bits carry the material index (n_materials > 1), and element
// (ix, iy, iz) of the device volume is the 2x2 quad of words
// {(ix,iy), (ix+1,iy), (ix,iy+1), (ix+1,iy+1)} of slab iz, stored for EVERY
// (ix, iy) (quads overlap, 16 B per voxel like the float4 layout).  A sample
// then needs two 16-byte loads (slabs iz and iz+1) instead of eight.
//
// Material routing.  In a segmented volume almost every cell is pure (all 8
// corners of one material: 98.8% of C3's cells), so the common path is one
// scalar tri-linear blend added to a running sum that is routed to its
// material only when the material changes; cells with mixed corners take a
// slower branch that routes each weighted corner.  Both give the same value.
//
// The words are used as floats as they are (the material bits are part of the
// stored value: |stored - rho| <= 5 ulp, 3e-7 relative; DESIGN.md "Packed
// words"); the library is compiled with -ftz=true so that rho = 0 tagged with a
// material (a denormal bit pattern) contributes exactly 0.
#include "project_common.cuh"

namespace gdrr {

template <int VW>
__device__ __forceinline__ void add_routed(float (&part)[VW], int m, float v) {
#pragma unroll
    for (int k = 0; k < VW; ++k) part[k] += (m == k) ? v : 0.f;
}

__device__ __forceinline__ float lerp(float a, float b, float t) { return fmaf(t, b - a, a); }

// (q & mask) | one in a single LOP3; mask and one arrive as kernel parameters so
// that they live in registers instead of being split into two immediate ops.
__device__ __forceinline__ float frac_float(int q, unsigned mask, unsigned one) {
    unsigned o;
    asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(o) : "r"(q), "r"(mask), "r"(one));
    return __uint_as_float(o) - 1.f;
}

// element index: slabs linear, 4 (x) x 2 (y) tiles of 8 quads = 128 B inside a slab
__device__ __forceinline__ int quad_index(int ix, int iy, int iz, int sy, int sz) {
    return iz * sz + (iy >> 1) * sy + ((iy & 1) << 2) + ix + (ix & ~3);
}

template <int VW, int MINB, int UNROLL>
__global__ void __launch_bounds__(kThreads, MINB)
gdrr_project_packed_kernel(const ProjectParams P) {
    float4* s_mu;
    float2* s_src;
    load_tables(P, s_mu, s_src);

    int i, j;
    thread_pixel(i, j);
    const int pl = blockIdx.z;
    if (i >= P.g.nu || j >= P.g.nv) return;

    // ---- a1: ray setup (fp64) ------------------------------------------------
    Ray r;
    ray_setup(P.g, P.g.proj_begin + pl, i, j, r);
    if (P.ray_table) {
        const size_t pix = ((size_t)pl * P.g.nv + j) * P.g.nu + i;
        reinterpret_cast<int2*>(P.ray_table)[pix] = make_int2(r.j0, r.n);
    }
    double gs[3], dg[3];
    index_line(P.g, r, gs, dg);
    const int dqx = __double2int_rn(dg[0] * 8388608.0);
    const int dqy = __double2int_rn(dg[1] * 8388608.0);
    const int dqz = __double2int_rn(dg[2] * 8388608.0);

    const int sy = P.v.stride_y, sz = P.v.stride_z;
    const uint4* __restrict__ vol0 = reinterpret_cast<const uint4*>(P.v.vox);   // slab iz
    const uint4* __restrict__ vol1 = vol0 + sz;                                  // slab iz + 1
    const unsigned fmask = P.frac_mask, fone = P.one_bits;

    // ---- a2-a4: sampling -------------------------------------------------------
    float acc[VW];
#pragma unroll
    for (int m = 0; m < VW; ++m) acc[m] = 0.f;
    unsigned curm = 0;         // material of the running sum of pure cells
    float cur = 0.f;

    for (int kc = 0; kc < r.n; kc += P.chunk) {
        const ChunkBase b = chunk_base(gs, dg, r.j0 + kc);
        int qx = b.qx, qy = b.qy, qz = b.qz;
        const int cnt = min(P.chunk, r.n - kc);

        float part[VW];
#pragma unroll
        for (int m = 0; m < VW; ++m) part[m] = 0.f;

        // software pipeline: the two loads of sample s + 1 are in flight while sample s is blended
        int idx = quad_index(b.cx, b.cy, b.cz, sy, sz);
        uint4 a = __ldg(vol0 + idx);            // slab iz:     (x0y0, x1y0, x0y1, x1y1)
        uint4 c = __ldg(vol1 + idx);            // slab iz + 1

#pragma unroll UNROLL
        for (int s = 0; s < cnt; ++s) {
            const float fx = frac_float(qx, fmask, fone);
            const float fy = frac_float(qy, fmask, fone);
            const float fz = frac_float(qz, fmask, fone);
            qx += dqx;
            qy += dqy;
            qz += dqz;
            uint4 an = a, cn = c;
            if (s + 1 < cnt) {
                idx = quad_index(b.cx + (qx >> kFracBits), b.cy + (qy >> kFracBits),
                                 b.cz + (qz >> kFracBits), sy, sz);
                an = __ldg(vol0 + idx);
                cn = __ldg(vol1 + idx);
            }

            bool fast = true;
            if (VW > 1) {
                // all 8 corners of the current material?  (two lowest bits of every word)
                const unsigned d = (a.x ^ a.y) | (a.x ^ a.z) | (a.x ^ a.w) | (a.x ^ c.x) | (a.x ^ c.y) |
                                   (a.x ^ c.z) | (a.x ^ c.w) | (a.x ^ curm);
                fast = (d & 3u) == 0u;
            }
            if (fast) {
                const float v0 = lerp(lerp(__uint_as_float(a.x), __uint_as_float(a.y), fx),
                                      lerp(__uint_as_float(a.z), __uint_as_float(a.w), fx), fy);
                const float v1 = lerp(lerp(__uint_as_float(c.x), __uint_as_float(c.y), fx),
                                      lerp(__uint_as_float(c.z), __uint_as_float(c.w), fx), fy);
                cur += lerp(v0, v1, fz);
            } else {
                // mixed cell, or a pure cell of another material: route every weighted corner
                const float gx = 1.f - fx, gy = 1.f - fy, gz = 1.f - fz;
                const float w00 = gy * gz, w10 = fy * gz, w01 = gy * fz, w11 = fy * fz;
                add_routed<VW>(part, (int)(a.x & 3u), gx * w00 * __uint_as_float(a.x));
                add_routed<VW>(part, (int)(a.y & 3u), fx * w00 * __uint_as_float(a.y));
                add_routed<VW>(part, (int)(a.z & 3u), gx * w10 * __uint_as_float(a.z));
                add_routed<VW>(part, (int)(a.w & 3u), fx * w10 * __uint_as_float(a.w));
                add_routed<VW>(part, (int)(c.x & 3u), gx * w01 * __uint_as_float(c.x));
                add_routed<VW>(part, (int)(c.y & 3u), fx * w01 * __uint_as_float(c.y));
                add_routed<VW>(part, (int)(c.z & 3u), gx * w11 * __uint_as_float(c.z));
                add_routed<VW>(part, (int)(c.w & 3u), fx * w11 * __uint_as_float(c.w));
                // the running sum follows the material the ray is now in
                const unsigned m = c.w & 3u;
                if (m != curm) {
                    add_routed<VW>(part, (int)curm, cur);
                    cur = 0.f;
                    curm = m;
                }
            }
            a = an;
            c = cn;
        }
        add_routed<VW>(part, (int)curm, cur);
        cur = 0.f;
#pragma unroll
        for (int m = 0; m < VW; ++m) acc[m] += part[m];
    }

    finish_pixel<VW>(P, s_mu, s_src, acc, pl, i, j);
}

template <int VW, int MINB, int UNROLL>
static cudaError_t launch_packed_t(const ProjectParams& p, cudaStream_t s) {
    dim3 grid((p.g.nu + kTileU - 1) / kTileU, (p.g.nv + kTileV - 1) / kTileV, p.g.proj_count);
    const size_t smem = (size_t)p.n_energy * (sizeof(float4) + sizeof(float2));
    gdrr_project_packed_kernel<VW, MINB, UNROLL><<<grid, kThreads, smem, s>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_project_packed(const ProjectParams& p, int vw, int variant, cudaStream_t s) {
    if (vw == 1) return launch_packed_t<1, 4, 2>(p, s);
    if (vw == 2) return launch_packed_t<2, 4, 2>(p, s);
    switch (variant) {
        case 1: return launch_packed_t<4, 3, 2>(p, s);
        case 2: return launch_packed_t<4, 5, 2>(p, s);
        case 3: return launch_packed_t<4, 6, 2>(p, s);
        case 4: return launch_packed_t<4, 4, 1>(p, s);
        case 5: return launch_packed_t<4, 5, 1>(p, s);
        case 6: return launch_packed_t<4, 6, 1>(p, s);
        case 7: return launch_packed_t<4, 4, 4>(p, s);
        case 8: return launch_packed_t<4, 3, 4>(p, s);
        default: return launch_packed_t<4, 4, 2>(p, s);
    }
}

}  // namespace gdrr
