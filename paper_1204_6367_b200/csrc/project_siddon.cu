// GDRR_METHOD_SIDDON: Siddon's exact radiological path fused with the
// energy sum.  The voxels are homogeneous boxes [lo + i d, lo + (i + 1) d); the line
// integral of material m is the sum over voxels of rho [mat = m] |ray /\ voxel|.
//
// One thread per detector pixel.  Ray setup in fp64 (ray_setup.cuh, the same clip of the
// source->pixel segment to the volume box as the tri-linear method).  The traversal is the
// incremental form of Siddon's merge: per axis the parameter of the next lattice plane the
// ray meets, the smallest of the three ends the current voxel's segment.  Parameters are
// kept in fp32 RELATIVE TO THE ENTRY POINT (range 0 .. chord, <= a few hundred mm) and are
// formed as fma(plane counter, dt, t0) from integer counters, never by repeated addition, so a
// crossing is placed within one ulp of the chord (3e-5 mm at 500 mm) however long the ray;
// a boundary misplaced by that much changes LI by 3e-5 mm x the density jump (~1e-7 relative).
// Segments of zero or negative length (ties at lattice edges, rounding) contribute nothing.
//
// Works on every device layout: the exact ones hold VW floats per voxel (one per material),
// PACKED_QUAD is read through the first word of each quad (rho with its material tag).
// fp32 accumulation is chunked like the tri-linear sampler's (32 segments per partial sum).
#include "project_common.cuh"

namespace gdrr {

template <int VW> struct SVox;
template <> struct SVox<1> { using T = float; };
template <> struct SVox<2> { using T = float2; };
template <> struct SVox<4> { using T = float4; };

__device__ __forceinline__ void add_len(float (&a)[1], float len, const float& v) { a[0] = fmaf(len, v, a[0]); }
__device__ __forceinline__ void add_len(float (&a)[2], float len, const float2& v) {
    a[0] = fmaf(len, v.x, a[0]);
    a[1] = fmaf(len, v.y, a[1]);
}
__device__ __forceinline__ void add_len(float (&a)[4], float len, const float4& v) {
    a[0] = fmaf(len, v.x, a[0]);
    a[1] = fmaf(len, v.y, a[1]);
    a[2] = fmaf(len, v.z, a[2]);
    a[3] = fmaf(len, v.w, a[3]);
}

template <int VW>
__device__ __forceinline__ void add_routed_s(float (&part)[VW], int m, float v) {
#pragma unroll
    for (int k = 0; k < VW; ++k) part[k] += (m == k) ? v : 0.f;
}

// element offset of padded voxel index i along one axis (project_fused.cu has the same map)
template <int LAYOUT, int AXIS>
__device__ __forceinline__ int siddon_axis_offset(int i, int stride) {
    if (LAYOUT == 0) return (i >> 1) * stride + ((i & 1) << AXIS);
    return i * stride;
}

// LAYOUT: 0 brick, 1 linear (exact, VW floats per voxel), 2 packed quad (first word of a quad)
template <int VW, int LAYOUT>
__global__ void __launch_bounds__(kThreads)
gdrr_project_siddon_kernel(const ProjectParams P) {
    using V = typename SVox<VW>::T;
    float4* s_mu;
    float2* s_src;
    load_tables(P, s_mu, s_src);

    int i, j;
    thread_pixel(i, j);
    const int pl = blockIdx.z;
    if (i >= P.g.nu || j >= P.g.nv) return;
    const size_t pix = ((size_t)pl * P.g.nv + j) * P.g.nu + i;

    Ray r;
    ray_setup(P.g, P.g.proj_begin + pl, i, j, r);
    if (P.ray_table) reinterpret_cast<int2*>(P.ray_table)[pix] = make_int2(r.j0, r.n);

    float acc[VW];
#pragma unroll
    for (int m = 0; m < VW; ++m) acc[m] = 0.f;
    int n_seg = 0;

    const double chord = r.t_out - r.t_in;
    if (r.hit) {
        // ---- set-up of the traversal (fp64): voxel at the entry point, plane counters, parameters
        int idx[3], stp[3], left[3];     // voxel index, +-1, planes still to cross before leaving the box
        float t0[3], dt[3];              // parameter (relative to t_in) of the next plane, and per plane
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const int N = P.v.nvox[a];
            const double x = fma(r.t_in, r.dir[a], r.S[a]);
            int v = (int)floor((x - P.g.lo[a]) / P.g.d[a]);
            v = min(max(v, 0), N - 1);
            idx[a] = v;
            if (r.dir[a] > 0.0) {
                stp[a] = 1;
                left[a] = N - v;
                t0[a] = (float)((P.g.lo[a] + (double)(v + 1) * P.g.d[a] - r.S[a]) / r.dir[a] - r.t_in);
                dt[a] = (float)(P.g.d[a] / r.dir[a]);
            } else if (r.dir[a] < 0.0) {
                stp[a] = -1;
                left[a] = v + 1;
                t0[a] = (float)((P.g.lo[a] + (double)v * P.g.d[a] - r.S[a]) / r.dir[a] - r.t_in);
                dt[a] = (float)(-P.g.d[a] / r.dir[a]);
            } else {
                stp[a] = 0;
                left[a] = 0x7fffffff;
                t0[a] = 3.0e38f;
                dt[a] = 0.f;
            }
        }
        const float t_end = (float)chord;
        constexpr int sx = (LAYOUT == 0) ? 8 : 1;
        const int sy = P.v.stride_y, sz = P.v.stride_z;
        // element offsets of the padded voxel (idx + 1)
        int ox = siddon_axis_offset<LAYOUT, 0>(idx[0] + 1, sx);
        int oy = siddon_axis_offset<LAYOUT, 1>(idx[1] + 1, sy);
        int oz = siddon_axis_offset<LAYOUT, 2>(idx[2] + 1, sz);
        int kx = 0, ky = 0, kz = 0;                      // planes crossed so far per axis
        float tx = t0[0], ty = t0[1], tz = t0[2];
        float t = 0.f;
        unsigned curm = 0;
        float cur = 0.f;
        bool inside = true;

        while (inside) {
            float part[VW];
#pragma unroll
            for (int m = 0; m < VW; ++m) part[m] = 0.f;
            for (int s = 0; s < kMaxChunk && inside; ++s) {
                // the voxel the ray is in, and where it leaves it
                const float tn = fminf(fminf(tx, ty), fminf(tz, t_end));
                const float len = tn - t;
                if (LAYOUT == 2) {
                    const unsigned w = __ldg(reinterpret_cast<const unsigned*>(P.v.vox) + 4 * (size_t)(oz + oy + ox));
                    if (len > 0.f) {
                        ++n_seg;
                        if (VW == 1) {
                            cur = fmaf(len, __uint_as_float(w), cur);
                        } else {
                            const unsigned m = w & 3u;
                            if (m != curm) {
                                add_routed_s<VW>(part, (int)curm, cur);
                                cur = 0.f;
                                curm = m;
                            }
                            cur = fmaf(len, __uint_as_float(w), cur);
                        }
                    }
                } else {
                    const V v = __ldg(reinterpret_cast<const V*>(P.v.vox) + (oz + oy + ox));
                    if (len > 0.f) {
                        ++n_seg;
                        add_len(part, len, v);
                    }
                }
                t = fmaxf(tn, t);
                // step into the next voxel across the plane that was met (x before y before z at ties)
                if (tn >= t_end) {
                    inside = false;
                } else if (tx <= ty && tx <= tz) {
                    ++kx;
                    idx[0] += stp[0];
                    ox = siddon_axis_offset<LAYOUT, 0>(idx[0] + 1, sx);
                    tx = fmaf((float)kx, dt[0], t0[0]);
                    inside = kx < left[0];
                } else if (ty <= tz) {
                    ++ky;
                    idx[1] += stp[1];
                    oy = siddon_axis_offset<LAYOUT, 1>(idx[1] + 1, sy);
                    ty = fmaf((float)ky, dt[1], t0[1]);
                    inside = ky < left[1];
                } else {
                    ++kz;
                    idx[2] += stp[2];
                    oz = siddon_axis_offset<LAYOUT, 2>(idx[2] + 1, sz);
                    tz = fmaf((float)kz, dt[2], t0[2]);
                    inside = kz < left[2];
                }
            }
            if (LAYOUT == 2) {
                add_routed_s<VW>(part, (int)curm, cur);
                cur = 0.f;
            }
#pragma unroll
            for (int m = 0; m < VW; ++m) acc[m] += part[m];
        }
    }

    if (P.seg_table) P.seg_table[pix] = n_seg;
    if (P.signal) finish_pixel<VW>(P, s_mu, s_src, acc, 1.0, pl, i, j);
}

template <int VW, int LAYOUT>
static cudaError_t launch_siddon_t(const ProjectParams& p, cudaStream_t s) {
    dim3 grid((p.g.nu + kTileU - 1) / kTileU, (p.g.nv + kTileV - 1) / kTileV, p.g.proj_count);
    const size_t smem = (size_t)p.n_energy * (sizeof(float4) + sizeof(float2));
    gdrr_project_siddon_kernel<VW, LAYOUT><<<grid, kThreads, smem, s>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_project_siddon(const ProjectParams& p, int vw, int layout, cudaStream_t s) {
    if (layout == 2) {
        if (vw == 1) return launch_siddon_t<1, 2>(p, s);
        if (vw == 2) return launch_siddon_t<2, 2>(p, s);
        return launch_siddon_t<4, 2>(p, s);
    }
    if (layout == 0) {
        if (vw == 1) return launch_siddon_t<1, 0>(p, s);
        if (vw == 2) return launch_siddon_t<2, 0>(p, s);
        return launch_siddon_t<4, 0>(p, s);
    }
    if (vw == 1) return launch_siddon_t<1, 1>(p, s);
    if (vw == 2) return launch_siddon_t<2, 1>(p, s);
    return launch_siddon_t<4, 1>(p, s);
}

}  // namespace gdrr
