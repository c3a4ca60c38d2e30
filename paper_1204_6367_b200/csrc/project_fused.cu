// Steps a1-a7 fused, EXACT layouts (GDRR_LAYOUT_BRICK / GDRR_LAYOUT_LINEAR):
// ray setup, fixed-step tri-linear sampling of the per-material density planes,
// and the energy sum.
//
// One thread per detector pixel.  The volume stores, per voxel, VW floats (one
// per material: rho at the voxel's material, 0 elsewhere), so one vector load
// per corner serves all materials and the 8 tri-linear weights are shared by
// them.  rho is kept bit-exact.  This is the reference layout of the library;
// the packed-quad layout (project_packed.cu) is the fast one.
#include "project_common.cuh"

namespace gdrr {

template <int VW> struct Vox;
template <> struct Vox<1> { using T = float; };
template <> struct Vox<2> { using T = float2; };
template <> struct Vox<4> { using T = float4; };

template <int VW>
__device__ __forceinline__ void fma_vox(float (&acc)[VW], float w, const typename Vox<VW>::T& v);
template <>
__device__ __forceinline__ void fma_vox<1>(float (&acc)[1], float w, const float& v) {
    acc[0] = fmaf(w, v, acc[0]);
}
template <>
__device__ __forceinline__ void fma_vox<2>(float (&acc)[2], float w, const float2& v) {
    acc[0] = fmaf(w, v.x, acc[0]);
    acc[1] = fmaf(w, v.y, acc[1]);
}
template <>
__device__ __forceinline__ void fma_vox<4>(float (&acc)[4], float w, const float4& v) {
    acc[0] = fmaf(w, v.x, acc[0]);
    acc[1] = fmaf(w, v.y, acc[1]);
    acc[2] = fmaf(w, v.z, acc[2]);
    acc[3] = fmaf(w, v.w, acc[3]);
}

// Element offset contributed by padded index i along one axis.
// BRICK: 2x2x2 bricks of 8 elements; x -> bit 0, y -> bit 1, z -> bit 2 inside a
// brick; bricks x fastest.  stride = 8 (x), 8 * bricks_per_row (y), 8 * bricks_per_slab (z).
template <int LAYOUT, int AXIS>
__device__ __forceinline__ int axis_offset(int i, int stride) {
    if (LAYOUT == 0) return (i >> 1) * stride + ((i & 1) << AXIS);
    return i * stride;
}

template <int VW, int LAYOUT>
__global__ void __launch_bounds__(kThreads)
gdrr_project_kernel(const ProjectParams P) {
    using V = typename Vox<VW>::T;
    float4* s_mu;
    float2* s_src;
    load_tables(P, s_mu, s_src);

    int i, j;
    thread_pixel(i, j);
    const int pl = blockIdx.z;                                 // projection inside this call
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

    const V* __restrict__ vox = reinterpret_cast<const V*>(P.v.vox);
    const int sy = P.v.stride_y, sz = P.v.stride_z;
    constexpr int sx = (LAYOUT == 0) ? 8 : 1;

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

#pragma unroll 2
        for (int s = 0; s < cnt; ++s) {
            const int ix = b.cx + (qx >> kFracBits);
            const int iy = b.cy + (qy >> kFracBits);
            const int iz = b.cz + (qz >> kFracBits);
            const float Fx = __int_as_float((qx & 0x7FFFFF) | 0x3F800000);   // 1 + frac
            const float Fy = __int_as_float((qy & 0x7FFFFF) | 0x3F800000);
            const float Fz = __int_as_float((qz & 0x7FFFFF) | 0x3F800000);
            const float wx1 = Fx - 1.f, wx0 = 2.f - Fx;
            const float wy1 = Fy - 1.f, wy0 = 2.f - Fy;
            const float wz1 = Fz - 1.f, wz0 = 2.f - Fz;

            const int x0 = axis_offset<LAYOUT, 0>(ix, sx), x1 = axis_offset<LAYOUT, 0>(ix + 1, sx);
            const int y0 = axis_offset<LAYOUT, 1>(iy, sy), y1 = axis_offset<LAYOUT, 1>(iy + 1, sy);
            const int z0 = axis_offset<LAYOUT, 2>(iz, sz), z1 = axis_offset<LAYOUT, 2>(iz + 1, sz);
            const int o00 = y0 + z0, o10 = y1 + z0, o01 = y0 + z1, o11 = y1 + z1;

            const V v000 = __ldg(vox + (o00 + x0));
            const V v100 = __ldg(vox + (o00 + x1));
            const V v010 = __ldg(vox + (o10 + x0));
            const V v110 = __ldg(vox + (o10 + x1));
            const V v001 = __ldg(vox + (o01 + x0));
            const V v101 = __ldg(vox + (o01 + x1));
            const V v011 = __ldg(vox + (o11 + x0));
            const V v111 = __ldg(vox + (o11 + x1));

            const float w00 = wy0 * wz0, w10 = wy1 * wz0, w01 = wy0 * wz1, w11 = wy1 * wz1;
            fma_vox<VW>(part, wx0 * w00, v000);
            fma_vox<VW>(part, wx1 * w00, v100);
            fma_vox<VW>(part, wx0 * w10, v010);
            fma_vox<VW>(part, wx1 * w10, v110);
            fma_vox<VW>(part, wx0 * w01, v001);
            fma_vox<VW>(part, wx1 * w01, v101);
            fma_vox<VW>(part, wx0 * w11, v011);
            fma_vox<VW>(part, wx1 * w11, v111);

            qx += dqx;
            qy += dqy;
            qz += dqz;
        }
#pragma unroll
        for (int m = 0; m < VW; ++m) acc[m] += part[m];
    }

    finish_pixel<VW>(P, s_mu, s_src, acc, P.g.step, pl, i, j);
}

// Ray setup alone: the integer ray table and/or the sample count sum(n).
__global__ void __launch_bounds__(kThreads)
gdrr_ray_setup_kernel(const GeomParams g, int32_t* __restrict__ ray_table,
                      unsigned long long* __restrict__ n_samples) {
    int i, j;
    thread_pixel(i, j);
    const int pl = blockIdx.z;
    int n = 0;
    if (i < g.nu && j < g.nv) {
        Ray r;
        ray_setup(g, g.proj_begin + pl, i, j, r);
        n = r.n;
        if (ray_table) {
            const size_t pix = ((size_t)pl * g.nv + j) * g.nu + i;
            reinterpret_cast<int2*>(ray_table)[pix] = make_int2(r.j0, r.n);
        }
    }
    if (n_samples) {
        unsigned int tot = __reduce_add_sync(0xffffffffu, (unsigned int)n);
        if ((threadIdx.x & 31) == 0 && tot) atomicAdd(n_samples, (unsigned long long)tot);
    }
}

template <int VW, int LAYOUT>
static cudaError_t launch_project_t(const ProjectParams& p, cudaStream_t s) {
    dim3 grid((p.g.nu + kTileU - 1) / kTileU, (p.g.nv + kTileV - 1) / kTileV, p.g.proj_count);
    const size_t smem = (size_t)p.n_energy * (sizeof(float4) + sizeof(float2));
    gdrr_project_kernel<VW, LAYOUT><<<grid, kThreads, smem, s>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_project_exact(const ProjectParams& p, int vw, int layout, cudaStream_t s) {
    if (layout == 0) {
        if (vw == 1) return launch_project_t<1, 0>(p, s);
        if (vw == 2) return launch_project_t<2, 0>(p, s);
        return launch_project_t<4, 0>(p, s);
    }
    if (vw == 1) return launch_project_t<1, 1>(p, s);
    if (vw == 2) return launch_project_t<2, 1>(p, s);
    return launch_project_t<4, 1>(p, s);
}

cudaError_t launch_ray_setup(const GeomParams& g, int32_t* ray_table,
                             unsigned long long* n_samples, cudaStream_t s) {
    dim3 grid((g.nu + kTileU - 1) / kTileU, (g.nv + kTileV - 1) / kTileV, g.proj_count);
    gdrr_ray_setup_kernel<<<grid, kThreads, 0, s>>>(g, ray_table, n_samples);
    return cudaGetLastError();
}

}  // namespace gdrr
