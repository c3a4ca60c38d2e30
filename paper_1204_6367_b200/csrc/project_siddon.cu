// GDRR_METHOD_SIDDON: Siddon's exact radiological path fused with the
// energy sum.  The voxels are homogeneous boxes [lo + i d, lo + (i + 1) d); the line
// integral of material m is the sum over voxels of rho [mat = m] |ray /\ voxel|.
//
// One thread per detector pixel.  Ray setup in fp64 (ray_setup.cuh, the same clip of the
// source->pixel segment to the volume box as the tri-linear method).  The traversal is the
// incremental form of Siddon's merge: per axis the parameter of the next lattice plane the
// ray meets, the smallest of the three ends the current voxel's segment.  The walk runs in
// chunks of 32 steps on fp32 parameters LOCAL to the chunk (relative to a point near the entry
// of its first voxel, so below ~50 mm); at every chunk start they are formed anew IN FP64
// from the count of planes crossed, count x dt + t0 minus that point, with the ray's fp64
// constants read back from shared memory.  A crossing is then placed within the 32 fp32
// additions of one chunk (<= 6e-5 mm, typically 5e-6) however long the ray.  (Round 2's first
// form rounded count x dt + t0 to fp32 at the chord's magnitude: 3e-5 mm per plane plus the
// rounding of dt times the count, 1.2e-4 mm between two axes; behind a bone / air jump that
// is 4e-4 mm g/cm^3, which the whole-scan parity run met once in 48 projections of C3.)
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

// fp64 -> fp32 as one F2F (under -ftz the plain cast adds a compare and a multiply to flush denormals, which never occur here)
__device__ __forceinline__ float to_float(double x) {
    float f;
    asm("cvt.rn.f32.f64 %0, %1;" : "=f"(f) : "d"(x));
    return f;
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
__global__ void __launch_bounds__(kThreads, 5)           // 48 registers: 5 CTAs per SM (4 at the 54 ptxas takes if left alone)
gdrr_project_siddon_kernel(const ProjectParams P) {
    using VT = typename SiddonVoxel<VW, LAYOUT>::T;
    __shared__ float s_acc[LAYOUT == 2 ? 4 : 1][LAYOUT == 2 ? kAccStride : 1];      // per-material sums of a packed walk
    __shared__ double s_ray[7][kThreads];           // this thread's t0[3], dt[3], t_end in fp64 (read at chunk starts only)
    __shared__ float s_idt[3][kThreads];            // ... 1 / dt (0 for an axis the ray does not move along)
    __shared__ float s_t0[3][kThreads];             // ... and t0 rounded to fp32, for the plane counts
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
            double t0d = 3.0e38, dtd = 0.0;
            if (r.dir[a] > 0.0) {
                stp[a] = 1;
                t0d = (P.g.lo[a] + (double)(v + 1) * P.g.d[a] - r.S[a]) / r.dir[a] - r.t_in;
                dtd = P.g.d[a] / r.dir[a];
            } else if (r.dir[a] < 0.0) {
                stp[a] = -1;
                t0d = (P.g.lo[a] + (double)v * P.g.d[a] - r.S[a]) / r.dir[a] - r.t_in;
                dtd = -P.g.d[a] / r.dir[a];
            } else {
                stp[a] = 0;
            }
            t0[a] = (float)t0d;
            dt[a] = (float)dtd;
            s_ray[a][threadIdx.x] = t0d;
            s_ray[3 + a][threadIdx.x] = dtd;
            s_t0[a][threadIdx.x] = t0[a];
            s_idt[a][threadIdx.x] = dt[a] > 0.f ? 1.f / dt[a] : 0.f;     // (0: that axis' parameter stays 3e38)
        }
        s_ray[6][threadIdx.x] = r.t_out - r.t_in;
        // The plane through which the ray leaves the box has the chunk-local parameter te up to the fp32 additions of
        // one chunk (<= 32 x half an ulp of te): a crossing within 64 ulp of the end IS the end, so the walk never
        // steps out of the lattice; the sliver it may drop is < 4e-6 of the last chunk's length (2e-4 mm at 50 mm).
        constexpr int sx = (LAYOUT == 0) ? 8 : 1;
        const int sy = LAYOUT == 2 ? P.v.cstride_y : P.v.stride_y, sz = LAYOUT == 2 ? P.v.cstride_z : P.v.stride_z;
        const void* vox = LAYOUT == 2 ? P.v.compact : P.v.vox;
        int off = siddon_axis_offset<LAYOUT, 0>(idx[0], sx) + siddon_axis_offset<LAYOUT, 1>(idx[1], sy) +
                  siddon_axis_offset<LAYOUT, 2>(idx[2], sz);
        // linear element orders: stepping one voxel along an axis adds a constant to the element offset
        const int dox = stp[0] * (LAYOUT == 2 ? 4 : sx), doy = stp[1] * sy, doz = stp[2] * sz;
        const int y_edge = stp[1] > 0 ? 3 : 0, doy_cross = stp[1] * (sy - 3);       // LAYOUT 2 only
        // Inside a chunk of kMaxChunk steps the parameters are LOCAL: relative to the point where the chunk's first voxel
        // was entered (tg, a parameter relative to the ray's entry), so that they stay below ~50 mm and the one addition
        // of dt per step costs 32 x half an ulp of THAT (6e-5 mm) instead of the chord's (5e-4 mm at 500 mm: measured
        // as 1.2e-3 of LI error behind a density jump on C2).  At a chunk's start the three global parameters are formed
        // anew in fp64 as fma(planes crossed, dt, t0) -- the count is what the drifted fp32 value still gives when
        // rounded -- and the frame's origin is taken off in fp64 too, so nothing accumulates from chunk to chunk and
        // nothing is rounded at the chord's magnitude.
        float tg = 0.f, t = 0.f;
        float tx = t0[0], ty = t0[1], tz = t0[2];
        float te = 0.f, ts = 0.f;
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
                // origin of the chunk's frame: the fp32 sum below, taken as exact (any point near the entry of the
                // current voxel serves; what matters is that every parameter is taken relative to the SAME number)
                const float ref = tg + t;
                const double refd = (double)ref;
                const double gx = fma((double)rintf((tg + tx - s_t0[0][threadIdx.x]) * s_idt[0][threadIdx.x]),
                                      s_ray[3][threadIdx.x], s_ray[0][threadIdx.x]);
                const double gy = fma((double)rintf((tg + ty - s_t0[1][threadIdx.x]) * s_idt[1][threadIdx.x]),
                                      s_ray[4][threadIdx.x], s_ray[1][threadIdx.x]);
                const double gz = fma((double)rintf((tg + tz - s_t0[2][threadIdx.x]) * s_idt[2][threadIdx.x]),
                                      s_ray[5][threadIdx.x], s_ray[2][threadIdx.x]);
                tx = to_float(gx - refd); ty = to_float(gy - refd); tz = to_float(gz - refd);
                te = to_float(s_ray[6][threadIdx.x] - refd);
                ts = te * (1.f - 64.f * 5.96e-8f);
                tg = ref;
                // the current voxel was entered at the last plane crossed (an axis the ray does not move along has none;
                // the ray's own entry is 0 - ref): local magnitudes, so fp32 places it within 1e-6 mm
                t = fmaxf(fmaxf(dt[0] > 0.f ? tx - dt[0] : -ref, dt[1] > 0.f ? ty - dt[1] : -ref),
                          fmaxf(dt[2] > 0.f ? tz - dt[2] : -ref, -ref));
            }
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
