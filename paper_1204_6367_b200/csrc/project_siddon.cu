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
// a PACKED_QUAD volume carries a second, compact copy for this walk: the same tagged word per
// voxel, rows in groups of four (4 B per voxel instead of 16; a 128-byte line is 8 x 4 voxels).
// fp32 accumulation is chunked like the tri-linear sampler's (32 segments per partial sum).
#include "packed_sampler.cuh"

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

// Element offset contributed by voxel index i along one axis.  LAYOUT 0: padded 2x2x2 bricks of the exact
// BRICK layout (project_fused.cu has the same map); 1: padded linear; 2: the packed volume's compact copy,
// unpadded, rows in groups of four: iz SZ + (iy >> 2) SY + 4 ix + (iy & 3) (volume_layout.cu).
template <int LAYOUT, int AXIS>
__device__ __forceinline__ int siddon_axis_offset(int i, int stride) {
    if (LAYOUT == 0) return ((i + 1) >> 1) * stride + (((i + 1) & 1) << AXIS);
    if (LAYOUT == 1) return (i + 1) * stride;
    if (AXIS == 0) return 4 * i;
    if (AXIS == 1) return (i >> 2) * stride + (i & 3);
    return i * stride;
}

// The material of the walk changes (a few times per ray): the closed run goes to its material's slot.  Out of line, so
// that the walk's loop keeps a plain branch around it instead of ten predicated instructions in every step.
__device__ __noinline__ void route_out_of_line(float* slot, unsigned m, float v) { slot[m * kAccStride] += v; }

// One voxel value: the exact layouts hold VW floats, the packed layout one tagged word.
template <int VW, int LAYOUT> struct SiddonVoxel { using T = typename SVox<VW>::T; };
template <int VW> struct SiddonVoxel<VW, 2> { using T = unsigned; };

template <int VW, int LAYOUT>
__device__ __forceinline__ typename SiddonVoxel<VW, LAYOUT>::T load_voxel(const void* vox, int off) {
    using T = typename SiddonVoxel<VW, LAYOUT>::T;
    return __ldg(reinterpret_cast<const T*>(vox) + off);
}

// LAYOUT: 0 brick, 1 linear (exact, VW floats per voxel), 2 packed volume's compact copy (one word per voxel)
// COUNT: also count the segments of positive length (gdrr_siddon_segments)
template <int VW, int LAYOUT, bool COUNT>
__global__ void __launch_bounds__(kThreads)
gdrr_project_siddon_kernel(const ProjectParams P) {
    using VT = typename SiddonVoxel<VW, LAYOUT>::T;
    __shared__ float s_acc[LAYOUT == 2 ? 4 : 1][LAYOUT == 2 ? kAccStride : 1];      // per-material sums of a packed walk
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

    if (r.hit) {
        // ---- set-up of the traversal (fp64): voxel at the entry point, parameters of the next planes
        int idx[3], stp[3];
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
                t0[a] = (float)((P.g.lo[a] + (double)(v + 1) * P.g.d[a] - r.S[a]) / r.dir[a] - r.t_in);
                dt[a] = (float)(P.g.d[a] / r.dir[a]);
            } else if (r.dir[a] < 0.0) {
                stp[a] = -1;
                t0[a] = (float)((P.g.lo[a] + (double)v * P.g.d[a] - r.S[a]) / r.dir[a] - r.t_in);
                dt[a] = (float)(-P.g.d[a] / r.dir[a]);
            } else {
                stp[a] = 0;
                t0[a] = 3.0e38f;
                dt[a] = 0.f;
            }
        }
        const float t_end = (float)(r.t_out - r.t_in);
        // The plane through which the ray leaves the box has the parameter t_end up to ~3 ulp (t0, dt and
        // t_end are rounded separately): a crossing within 16 ulp of the end IS the end, so the walk never
        // steps out of the lattice; the sliver it may drop is < 5e-4 mm of the last voxel.
        const float t_stop = t_end * (1.f - 16.f * 5.96e-8f);
        constexpr int sx = (LAYOUT == 0) ? 8 : 1;
        const int sy = LAYOUT == 2 ? P.v.cstride_y : P.v.stride_y, sz = LAYOUT == 2 ? P.v.cstride_z : P.v.stride_z;
        const void* vox = LAYOUT == 2 ? P.v.compact : P.v.vox;
        int off = siddon_axis_offset<LAYOUT, 0>(idx[0], sx) + siddon_axis_offset<LAYOUT, 1>(idx[1], sy) +
                  siddon_axis_offset<LAYOUT, 2>(idx[2], sz);
        // linear element orders: stepping one voxel along an axis adds a constant to the element offset
        const int dox = stp[0] * (LAYOUT == 2 ? 4 : sx), doy = stp[1] * sy, doz = stp[2] * sz;
        const int y_edge = stp[1] > 0 ? 3 : 0, doy_cross = stp[1] * (sy - 3);       // LAYOUT 2 only
        // 1 / dt for the re-base (0 for an axis the ray does not move along: its parameter stays 3e38)
        const float idt[3] = {dt[0] > 0.f ? 1.f / dt[0] : 0.f, dt[1] > 0.f ? 1.f / dt[1] : 0.f,
                              dt[2] > 0.f ? 1.f / dt[2] : 0.f};
        // Inside a chunk of kMaxChunk steps the parameters are LOCAL: relative to the point where the chunk's first voxel
        // was entered (tg, a parameter relative to the ray's entry), so that they stay below ~50 mm and the one addition
        // of dt per step costs 32 x half an ulp of THAT (6e-5 mm) instead of the chord's (5e-4 mm at 500 mm: measured
        // as 1.2e-3 of LI error behind a density jump on C2).  At a chunk's start the three global parameters are formed
        // anew as fma(planes crossed, dt, t0) -- the count is what the drifted value still gives when rounded -- so
        // nothing accumulates from chunk to chunk.
        float tg = 0.f;
        float tx = t0[0], ty = t0[1], tz = t0[2];
        float te = t_end, ts = t_stop;
        RayAcc<VW> A;                                    // LAYOUT 2: running sum of the current material (packed_sampler.cuh)
        if (LAYOUT == 2) init_ray<VW>(A, &s_acc[0][threadIdx.x]);

        // the walk moves a pointer; the voxel of segment s + 1 is requested before segment s is accumulated.
        // (compact copy: its base is 256-byte aligned and SY, SZ are multiples of 4 words, so bits 2-3 of the
        // address are the row's place in its group of four)
        const VT* ptr = reinterpret_cast<const VT*>(vox) + off;
        const unsigned y_edge_bits = 4u * (unsigned)y_edge;
        // (kept in registers: left alone, ptxas re-forms these from their inputs in every step of the walk)
        int doy_cross_r = doy_cross, step_y_r = stp[1];
        asm volatile("" : "+r"(doy_cross_r), "+r"(step_y_r));
        VT v = __ldg(ptr);
        bool more = true;
        while (more) {
            float part[VW];
#pragma unroll
            for (int m = 0; m < VW; ++m) part[m] = 0.f;
            {
                const float gx = fmaf(rintf((tg + tx - t0[0]) * idt[0]), dt[0], t0[0]);
                const float gy = fmaf(rintf((tg + ty - t0[1]) * idt[1]), dt[1], t0[1]);
                const float gz = fmaf(rintf((tg + tz - t0[2]) * idt[2]), dt[2], t0[2]);
                // the current voxel was entered at the last plane crossed (an axis the ray does not move along has none)
                tg = fmaxf(fmaxf(dt[0] > 0.f ? gx - dt[0] : 0.f, dt[1] > 0.f ? gy - dt[1] : 0.f),
                           fmaxf(dt[2] > 0.f ? gz - dt[2] : 0.f, 0.f));
                tx = gx - tg; ty = gy - tg; tz = gz - tg;
                te = t_end - tg; ts = t_stop - tg;
            }
            float t = 0.f;
#pragma unroll 2
            for (int s = 0; s < kMaxChunk && more; ++s) {
                const float tn = fminf(fminf(tx, ty), fminf(tz, te));       // where the ray leaves this voxel
                const float tnew = fmaxf(tn, t);
                const float len = tnew - t;                                 // >= 0
                t = tnew;
                more = tn < ts;
                // cross the plane that was met (x before y before z at ties)
                const bool bx = tx == tn;
                const bool by = !bx && ty == tn;
                if (LAYOUT == 0) {
                    idx[0] += bx ? stp[0] : 0;
                    idx[1] += by ? stp[1] : 0;
                    idx[2] += (bx || by) ? 0 : stp[2];
                    ptr = reinterpret_cast<const VT*>(vox) + (siddon_axis_offset<LAYOUT, 0>(idx[0], sx) +
                          siddon_axis_offset<LAYOUT, 1>(idx[1], sy) + siddon_axis_offset<LAYOUT, 2>(idx[2], sz));
                } else if (LAYOUT == 2) {
                    // rows in groups of 4: a step in y moves by one word inside a group, by a row of groups across its edge
                    const int dy_now = (((unsigned)(uintptr_t)ptr & 12u) == y_edge_bits) ? doy_cross_r : step_y_r;
                    ptr += bx ? dox : (by ? dy_now : doz);
                } else {
                    ptr += bx ? dox : (by ? doy : doz);
                }
                if (bx) tx += dt[0];
                if (by) ty += dt[1];
                if (!bx && !by) tz += dt[2];
                const VT cv = v;
                if (more) v = __ldg(ptr);                                   // (past the end the walk has left the lattice)
                if (COUNT) n_seg += len > 0.f ? 1 : 0;
                if constexpr (LAYOUT == 2) {
                    if (VW > 1) {
                        const unsigned m4 = (cv & 3u) | 4u;
                        if (m4 != A.curm4) {
                            route_out_of_line(A.slot, A.curm4 & 3u, A.cur + A.run);
                            A.cur = 0.f;
                            A.run = 0.f;
                            A.curm4 = m4;
                        }
                    }
                    A.cur = fmaf(len, __uint_as_float(cv), A.cur);
                } else {
                    add_len(part, len, cv);
                }
            }
            if (LAYOUT == 2) {
                flush_chunk<VW>(A);
            } else {
#pragma unroll
                for (int m = 0; m < VW; ++m) acc[m] += part[m];
            }
        }
        if (LAYOUT == 2) finish_ray<VW>(A, acc);
    }

    if (COUNT && P.seg_table) P.seg_table[pix] = n_seg;
    if (P.signal) finish_pixel<VW>(P, s_mu, s_src, acc, 1.0, pl, i, j);
}

template <int VW, int LAYOUT, bool COUNT>
static cudaError_t launch_siddon_c(const ProjectParams& p, cudaStream_t s) {
    dim3 grid((p.g.nu + kTileU - 1) / kTileU, (p.g.nv + kTileV - 1) / kTileV, p.g.proj_count);
    const size_t smem = (size_t)p.n_energy * (sizeof(float4) + sizeof(float2));
    gdrr_project_siddon_kernel<VW, LAYOUT, COUNT><<<grid, kThreads, smem, s>>>(p);
    return cudaGetLastError();
}

template <int VW, int LAYOUT>
static cudaError_t launch_siddon_t(const ProjectParams& p, cudaStream_t s) {
    if (p.seg_table) return launch_siddon_c<VW, LAYOUT, true>(p, s);
    return launch_siddon_c<VW, LAYOUT, false>(p, s);
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
