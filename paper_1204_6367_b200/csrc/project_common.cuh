// Pieces shared by the sampling kernels: thread -> pixel mapping, the spectrum
// tables in shared memory, the in-chunk fixed-point position, the energy sum.
#pragma once
#include "gdrr_internal.h"
#include "ray_setup.cuh"

namespace gdrr {

// thread -> pixel: warp w covers an 8 (u) x 4 (v) block of the CTA's 16 x 16 tile
__device__ __forceinline__ void thread_pixel(int& i, int& j) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    i = blockIdx.x * kTileU + (warp & 1) * 8 + (lane & 7);
    j = blockIdx.y * kTileV + (warp >> 1) * 4 + (lane >> 3);
}

// Spectrum tables -> shared memory (all threads of the CTA must call this).
__device__ __forceinline__ void load_tables(const ProjectParams& P, float4*& s_mu, float2*& s_src) {
    extern __shared__ float4 smem_f4[];
    s_mu = smem_f4;                                               // [n_energy]
    s_src = reinterpret_cast<float2*>(s_mu + P.n_energy);         // [n_energy]
    for (int e = threadIdx.x; e < P.n_energy; e += kThreads) {
        s_mu[e] = P.mu_tab[e];
        s_src[e] = P.src_tab[e];
    }
    __syncthreads();
}

// Position of sample j0 + kc in fp64, split per axis into the integer cell
// (padded index coordinates) and a 23-bit fixed-point fraction.
struct ChunkBase {
    int cx, cy, cz;     // cell of the first sample of the chunk
    int qx, qy, qz;     // fraction * 2^23, in [0, 2^23)
};

__device__ __forceinline__ ChunkBase chunk_base(const double (&gs)[3], const double (&dg)[3], int k) {
    const double tk = (double)k + 0.5;
    const double bx = fma(tk, dg[0], gs[0]);
    const double by = fma(tk, dg[1], gs[1]);
    const double bz = fma(tk, dg[2], gs[2]);
    const double fx = floor(bx), fy = floor(by), fz = floor(bz);
    ChunkBase b;
    b.cx = (int)fx; b.cy = (int)fy; b.cz = (int)fz;
    b.qx = (int)((bx - fx) * 8388608.0);
    b.qy = (int)((by - fy) * 8388608.0);
    b.qz = (int)((bz - fz) * 8388608.0);
    return b;
}

// padded index coordinate of the point at parameter t:  q_a(t) = gs_a + (t / dl) * dg_a
__device__ __forceinline__ void index_line(const GeomParams& g, const Ray& r, double (&gs)[3],
                                           double (&dg)[3]) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        // (not part of the bit-exact ray table: reciprocals instead of six fp64 divisions per ray)
        gs[a] = (r.S[a] - g.c[a]) * g.inv_d[a] + g.ofs[a];
        dg[a] = g.step * r.dir[a] * g.inv_d[a];
    }
}

// Steps a5-a7: scale the sums (by dl for the midpoint rule, by 1 for Siddon's lengths), optional LI output, energy sum with the tables in
// shared memory (exp as ex2 of pre-scaled arguments), store.
template <int VW>
__device__ __forceinline__ void finish_pixel(const ProjectParams& P, const float4* s_mu,
                                             const float2* s_src, const float (&acc)[VW],
                                             double scale, int pl, int i, int j) {
    float li[VW];
#pragma unroll
    for (int m = 0; m < VW; ++m) li[m] = (float)((double)acc[m] * scale);
    if (P.li) {
        const size_t plane = (size_t)P.g.nv * P.g.nu;
        float* o = P.li + ((size_t)pl * P.li_mat_total + P.li_mat0) * plane + (size_t)j * P.g.nu + i;
#pragma unroll
        for (int m = 0; m < VW; ++m)
            if (m < P.n_mat) o[m * plane] = li[m];
    }
    if (P.li_only) return;          // one group of more than four materials: gdrr_energy_sum_kernel forms the signal
    // exp(-tau) as ex2 of the NEGATED optical depth, formed directly: the signs go into the line integrals once
    const float ntb = P.bt_thick ? -P.bt_thick[i] : 0.f;
    float nli[VW];
#pragma unroll
    for (int m = 0; m < VW; ++m) nli[m] = -li[m];
    float sig = 0.f;
    auto bin = [&](int e, float weight) {
        const float4 mu = s_mu[e];
        float ntau = s_src[e].y * ntb;
        ntau = fmaf(mu.x, nli[0], ntau);
        if (VW > 1) ntau = fmaf(mu.y, nli[VW > 1 ? 1 : 0], ntau);
        if (VW > 2) {
            ntau = fmaf(mu.z, nli[VW > 2 ? 2 : 0], ntau);
            ntau = fmaf(mu.w, nli[VW > 2 ? 3 : 0], ntau);
        }
        sig = fmaf(weight, exp2f(ntau), sig);
    };
    if (P.gain) {
        // pixel-dependent detector response r(E, u) = r(E) g(E, u) (reading Q32): g streams in from global
        // memory, energy-major, so that the pixels of a warp read neighbouring words.  (Its own loop: predicated off, the
        // loads and their address arithmetic would still issue in every bin of the common case.)
        const size_t gain_plane = (size_t)P.g.nv * P.g.nu;
        const float* gain = P.gain + (size_t)j * P.g.nu + i;
#pragma unroll 1        // (the rare path: kept small, so that it does not raise the kernels' register counts)
        for (int e = 0; e < P.n_energy; ++e) bin(e, s_src[e].x * __ldg(gain + (size_t)e * gain_plane));
    } else {
        for (int e = 0; e < P.n_energy; ++e) bin(e, s_src[e].x);
    }
    if (P.fluence) sig *= P.fluence[(size_t)j * P.g.nu + i];
    P.signal[((size_t)pl * P.g.nv + j) * P.g.nu + i] = sig;
}

}  // namespace gdrr
