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

template <int VW>
__global__ void __launch_bounds__(kThreads)
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

    const uint4* __restrict__ vol = reinterpret_cast<const uint4*>(P.v.vox);
    const int sy = P.v.stride_y, sz = P.v.stride_z;

    // ---- a2-a4: sampling -------------------------------------------------------
    float acc[VW];
#pragma unroll
    for (int m = 0; m < VW; ++m) acc[m] = 0.f;

    for (int kc = 0; kc < r.n; kc += P.chunk) {
        const ChunkBase b = chunk_base(gs, dg, r.j0 + kc);
        int qx = b.qx, qy = b.qy, qz = b.qz;
        const int cnt = min(P.chunk, r.n - kc);

        float part[VW];
#pragma unroll
        for (int m = 0; m < VW; ++m) part[m] = 0.f;
        int curm = 0;          // material of the running sum of pure cells
        float cur = 0.f;

#pragma unroll 2
        for (int s = 0; s < cnt; ++s) {
            const int ix = b.cx + (qx >> kFracBits);
            const int iy = b.cy + (qy >> kFracBits);
            const int iz = b.cz + (qz >> kFracBits);
            const float fx = __int_as_float((qx & 0x7FFFFF) | 0x3F800000) - 1.f;
            const float fy = __int_as_float((qy & 0x7FFFFF) | 0x3F800000) - 1.f;
            const float fz = __int_as_float((qz & 0x7FFFFF) | 0x3F800000) - 1.f;
            // element index: slabs linear, 4 (x) x 2 (y) tiles of 8 quads = 128 B inside a slab
            const int idx = iz * sz + (iy >> 1) * sy + ((iy & 1) << 2) + ix + (ix & ~3);
            const uint4 a = __ldg(vol + idx);           // slab iz:     (x0y0, x1y0, x0y1, x1y1)
            const uint4 c = __ldg(vol + idx + sz);      // slab iz + 1

            bool pure = true;
            if (VW > 1) {
                const unsigned d = (a.x ^ a.y) | (a.x ^ a.z) | (a.x ^ a.w) | (a.x ^ c.x) | (a.x ^ c.y) |
                                   (a.x ^ c.z) | (a.x ^ c.w);
                pure = (d & 3u) == 0u;
            }
            if (pure) {
                const float v0 = lerp(lerp(__uint_as_float(a.x), __uint_as_float(a.y), fx),
                                      lerp(__uint_as_float(a.z), __uint_as_float(a.w), fx), fy);
                const float v1 = lerp(lerp(__uint_as_float(c.x), __uint_as_float(c.y), fx),
                                      lerp(__uint_as_float(c.z), __uint_as_float(c.w), fx), fy);
                const float v = lerp(v0, v1, fz);
                if (VW > 1) {
                    const int m = (int)(a.x & 3u);
                    if (m != curm) {
                        add_routed<VW>(part, curm, cur);
                        cur = 0.f;
                        curm = m;
                    }
                }
                cur += v;
            } else {
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
            }
            qx += dqx;
            qy += dqy;
            qz += dqz;
        }
        add_routed<VW>(part, curm, cur);
#pragma unroll
        for (int m = 0; m < VW; ++m) acc[m] += part[m];
    }

    finish_pixel<VW>(P, s_mu, s_src, acc, pl, i, j);
}

cudaError_t launch_project_packed(const ProjectParams& p, int vw, cudaStream_t s) {
    dim3 grid((p.g.nu + kTileU - 1) / kTileU, (p.g.nv + kTileV - 1) / kTileV, p.g.proj_count);
    const size_t smem = (size_t)p.n_energy * (sizeof(float4) + sizeof(float2));
    if (vw == 1) gdrr_project_packed_kernel<1><<<grid, kThreads, smem, s>>>(p);
    else if (vw == 2) gdrr_project_packed_kernel<2><<<grid, kThreads, smem, s>>>(p);
    else gdrr_project_packed_kernel<4><<<grid, kThreads, smem, s>>>(p);
    return cudaGetLastError();
}

}  // namespace gdrr
