// Steps a6-a7 on their own, for volumes of MORE THAN FOUR materials (PAPER.md:97 puts no bound on the material index).
// Such a volume is kept as groups of four materials, each a complete device volume in which the voxels of the other
// groups are empty (gdrr_api.cu); the sampling kernels run once per group and write only their group's line integrals
// into the caller's [proj][n_materials][nv][nu] array.  This kernel then forms
//   P = w(u) sum_E phi_E R_E g(E, u) exp(-mu_bt,E t_bt(i)) exp(-sum_m mu_hat[m][E] LI_m)
// from all of them: one thread per pixel, the table [n_energy][n_materials] of log2(e) mu_hat in shared memory.
#include "project_common.cuh"

namespace gdrr {

constexpr int kMaxMat = 16;     // GDRR_MAX_MATERIALS

__global__ void __launch_bounds__(kThreads)
gdrr_energy_sum_kernel(const ProjectParams P) {
    extern __shared__ float s_tab[];                     // [n_energy][M] mu, then [n_energy] float2 (phi R, log2e mu_bt)
    const int M = P.li_mat_total;
    float2* s_src = reinterpret_cast<float2*>(s_tab + (((size_t)P.n_energy * M + 1) & ~(size_t)1));      // 8-byte aligned
    for (int k = threadIdx.x; k < P.n_energy * M; k += kThreads) s_tab[k] = P.mu_all[k];
    for (int e = threadIdx.x; e < P.n_energy; e += kThreads) s_src[e] = P.src_tab[e];
    __syncthreads();
    int i, j;
    thread_pixel(i, j);
    const int pl = blockIdx.z;
    if (i >= P.g.nu || j >= P.g.nv) return;
    const size_t plane = (size_t)P.g.nv * P.g.nu, pix = (size_t)j * P.g.nu + i;
    float li[kMaxMat];
#pragma unroll
    for (int m = 0; m < kMaxMat; ++m) li[m] = m < M ? P.li[((size_t)pl * M + m) * plane + pix] : 0.f;
    const float tb = P.bt_thick ? P.bt_thick[i] : 0.f;
    const float* gain = P.gain ? P.gain + pix : nullptr;
    float sig = 0.f;
    for (int e = 0; e < P.n_energy; ++e) {
        float2 sc = s_src[e];
        if (gain) sc.x *= __ldg(gain + (size_t)e * plane);
        float tau = sc.y * tb;
#pragma unroll
        for (int m = 0; m < kMaxMat; ++m)
            if (m < M) tau = fmaf(s_tab[e * M + m], li[m], tau);
        sig = fmaf(sc.x, exp2f(-tau), sig);
    }
    if (P.fluence) sig *= P.fluence[pix];
    P.signal[(size_t)pl * plane + pix] = sig;
}

cudaError_t launch_energy_sum(const ProjectParams& p, cudaStream_t s) {
    dim3 grid((p.g.nu + kTileU - 1) / kTileU, (p.g.nv + kTileV - 1) / kTileV, p.g.proj_count);
    const size_t smem = (((size_t)p.n_energy * p.li_mat_total + 1) & ~(size_t)1) * sizeof(float) + (size_t)p.n_energy * sizeof(float2);
    cudaError_t e = cudaFuncSetAttribute(gdrr_energy_sum_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         512 * (kMaxMat * 4 + 8));
    if (e != cudaSuccess) return e;
    gdrr_energy_sum_kernel<<<grid, kThreads, smem, s>>>(p);
    return cudaGetLastError();
}

}  // namespace gdrr
