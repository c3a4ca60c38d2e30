// L1 data-pipe micro-benchmark (profiles/r01_l1_model.md): what a warp-wide 16-byte load costs
// when some of its sectors miss L1.  Read the counters with
//   ncu --metrics l1tex__data_pipe_lsu_wavefronts.sum,l1tex__t_requests_pipe_lsu_mem_global_op_ld.sum ./l1_partial_miss
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o l1_partial_miss l1_partial_miss.cu
// Partial misses: in every 8-lane phase, `nmiss` lanes stream through fresh lines (slot = lane&7 kept), the rest hit a resident line.
#include <cuda_runtime.h>
#include <cstdio>
__global__ void __launch_bounds__(256) k(const char* hot, const char* cold, int iters, unsigned* out, int nmiss) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const size_t wid = (size_t)blockIdx.x * 8 + warp;
    const int kk = lane & 7, ph = lane >> 3;
    const bool miss = kk < nmiss;
    // hot: one line per phase per warp, lane slot kk;  cold: per (warp, lane) a private run of lines, slot kk
    const char* p = miss ? cold + ((wid * 32 + lane) * (size_t)iters) * 128 + kk * 16
                         : hot + (wid * 4 + ph) * 128 + kk * 16;
    const size_t step = miss ? 128 : 0;
    unsigned acc = 0;
    for (int it = 0; it < iters; ++it) {
        uint4 v;
        asm volatile("ld.global.nc.v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
        acc ^= v.x ^ v.y ^ v.z ^ v.w;
        p += step;
    }
    out[wid * 32 + lane] = acc;
}
int main() {
    const int ctas = 148 * 2, iters = 128;
    size_t warps = (size_t)ctas * 8;
    char *hot, *cold; unsigned* out;
    cudaMalloc(&hot, warps * 4 * 128 + 4096); cudaMalloc(&cold, warps * 32 * (size_t)iters * 128 + 4096);
    cudaMemset(hot, 1, warps * 4 * 128); cudaMemset(cold, 1, warps * 32 * (size_t)iters * 128);
    cudaMalloc(&out, warps * 32 * 4);
    for (int nm = 0; nm <= 8; nm = nm ? nm * 2 : 1) k<<<ctas, 256>>>(hot, cold, iters, out, nm);
    printf("%s\n", cudaGetErrorString(cudaDeviceSynchronize()));
    return 0;
}
