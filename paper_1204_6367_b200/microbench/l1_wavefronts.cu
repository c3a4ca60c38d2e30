// L1 data-pipe micro-benchmark: cycles per warp-wide global load for lane address patterns
// (all L1 hits).  It measured the model the packed sampler's layout is built on
// (profiles/r01_l1_model.md).  Not part of the library; build and run by hand on a B200:
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 -o l1_wavefronts l1_wavefronts.cu
//   ./l1_wavefronts [patterns.txt]      (patterns.txt: lines of `name width off0 ... off31`)
#include <cuda_runtime.h>
#include <cstdio>
#include <cstdlib>
#include <vector>
#include <string>

template <int W>  // W = bytes per lane: 4, 8, 16, 32
__device__ __forceinline__ unsigned ld(const char* p) {
    unsigned a, b, c, d, e, f, g, h;
    if (W == 4) { asm volatile("ld.global.nc.b32 %0, [%1];" : "=r"(a) : "l"(p)); return a; }
    if (W == 8) { asm volatile("ld.global.nc.v2.b32 {%0,%1}, [%2];" : "=r"(a), "=r"(b) : "l"(p)); return a ^ b; }
    if (W == 16) { asm volatile("ld.global.nc.v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(a), "=r"(b), "=r"(c), "=r"(d) : "l"(p)); return a ^ b ^ c ^ d; }
    asm volatile("ld.global.nc.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(a), "=r"(b), "=r"(c), "=r"(d), "=r"(e), "=r"(f), "=r"(g), "=r"(h) : "l"(p));
    return a ^ b ^ c ^ d ^ e ^ f ^ g ^ h;
}

template <int W>
__global__ void __launch_bounds__(256) kern(const char* base, const int* offs, int iters, unsigned* out, long long* cyc) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int off = offs[lane];
    // each warp has its own 4 KB window inside a 32 KB per-CTA region (L1 resident)
    const char* p = base + (size_t)blockIdx.x * 65536 + warp * 8192 + off;
    unsigned acc = 0;
    // warm the L1
    for (int k = 0; k < 4; ++k) acc ^= ld<W>(p);
    __syncthreads();
    long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) acc ^= ld<W>(p + u * 128 + (it & 3) * 1024);
    }
    long long t1 = clock64();
    __syncthreads();
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
    if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}

struct Pat { std::string name; int w; int off[32]; };

int main(int argc, char** argv) {
    std::vector<Pat> pats;
    auto add = [&](const char* n, int w, auto f) { Pat p; p.name = n; p.w = w; for (int l = 0; l < 32; ++l) p.off[l] = f(l); pats.push_back(p); };
    for (int w : {4, 8, 16, 32}) {
        add("coalesced", w, [=](int l) { return l * w; });
        add("broadcast", w, [=](int l) { return 0; });
    }
    // ---- 16-byte loads, quarter-warp = 8 lanes
    add("q: 8 lanes -> 2 lines, same elem slot", 16, [](int l) { return (l >> 3) * 256 + ((l & 7) >> 2) * 128; });
    add("q: 8 lanes -> 2 lines, disjoint banks (A0-3,B4-7)", 16, [](int l) { int q = l >> 3, k = l & 7; return q * 256 + (k >> 2) * 128 + k * 16; });
    add("q: 8 lanes -> 4 lines, disjoint banks", 16, [](int l) { int q = l >> 3, k = l & 7; return q * 512 + (k >> 1) * 128 + k * 16; });
    add("q: 8 lanes -> 8 lines, disjoint banks", 16, [](int l) { int q = l >> 3, k = l & 7; return q * 1024 + k * 128 + k * 16; });
    add("q: 8 lanes -> 8 lines, same bank", 16, [](int l) { int q = l >> 3, k = l & 7; return q * 1024 + k * 128; });
    add("q: 8 lanes -> 1 line, 3 distinct elems", 16, [](int l) { int q = l >> 3, k = l & 7; return q * 128 + (k % 3) * 16; });
    add("q: 8 lanes -> 1 line, 8 elems permuted", 16, [](int l) { int q = l >> 3, k = l & 7; return q * 128 + ((k * 5) & 7) * 16; });
    add("all 32 lanes -> 1 line (8 elems x4)", 16, [](int l) { return (l & 7) * 16; });
    add("all 32 lanes -> 2 lines interleaved", 16, [](int l) { return (l & 1) * 128 + ((l >> 1) & 7) * 16; });
    add("warp: 13 distinct elems in 4 lines, by quarter 1 line", 16, [](int l) { int q = l >> 3, k = l & 7; return q * 128 + (k % 3 + (q & 1)) * 16; });
    add("lanes pairs across quarters same line (l&3 lines)", 16, [](int l) { return (l & 3) * 128 + (l >> 2) * 16; });
    // ---- 32-byte loads, eighth-warp = 4 lanes?
    add("o: 4 lanes -> 1 line permuted", 32, [](int l) { int o = l >> 2, k = l & 3; return o * 128 + ((k * 3) & 3) * 32; });
    add("o: 4 lanes -> 2 lines same slot", 32, [](int l) { int o = l >> 2, k = l & 3; return o * 256 + (k >> 1) * 128; });
    add("o: 4 lanes -> 2 lines disjoint", 32, [](int l) { int o = l >> 2, k = l & 3; return o * 256 + (k >> 1) * 128 + k * 32; });
    add("o: 4 lanes -> 4 lines disjoint", 32, [](int l) { int o = l >> 2, k = l & 3; return o * 512 + k * 128 + k * 32; });
    add("o: 4 lanes -> 4 lines same slot", 32, [](int l) { int o = l >> 2, k = l & 3; return o * 512 + k * 128; });
    add("8 lanes -> 1 line (4 elems x2) ", 32, [](int l) { int q = l >> 3, k = l & 7; return q * 128 + (k & 3) * 32; });
    add("all lanes 2 distinct sectors one line", 32, [](int l) { return (l & 1) * 32; });
    add("all lanes 4 sectors, 4 lines", 32, [](int l) { return (l & 3) * 128; });
    // ---- 4-byte loads, whole warp one phase
    add("w: 32 lanes -> 2 lines disjoint banks", 4, [](int l) { return (l >> 4) * 128 + l * 4; });
    add("w: 32 lanes -> 4 lines disjoint banks", 4, [](int l) { return (l >> 3) * 128 + l * 4; });
    add("w: 32 lanes -> 4 lines same bank", 4, [](int l) { return (l & 3) * 128; });
    add("w: 32 lanes -> 8 lines disjoint banks", 4, [](int l) { return (l >> 2) * 128 + l * 4; });
    add("w: 32 lanes -> 32 lines", 4, [](int l) { return l * 128; });
    // ---- 8-byte
    add("h: 16 lanes -> 2 lines disjoint", 8, [](int l) { int h = l >> 4, k = l & 15; return h * 256 + (k >> 3) * 128 + k * 8; });
    add("h: 16 lanes -> 4 lines disjoint", 8, [](int l) { int h = l >> 4, k = l & 15; return h * 512 + (k >> 2) * 128 + k * 8; });

    if (argc > 1) {
        pats.clear();
        FILE* fp = fopen(argv[1], "r");
        char nm[256]; int w;
        while (fp && fscanf(fp, "%255s %d", nm, &w) == 2) {
            Pat p; p.name = nm; p.w = w;
            for (int l = 0; l < 32; ++l) if (fscanf(fp, "%d", &p.off[l]) != 1) return 2;
            pats.push_back(p);
        }
    }
    const int ctas = 148 * 2, threads = 256, iters = 512;
    char* base; int* offs; unsigned* out; long long* cyc;
    cudaMalloc(&base, (size_t)ctas * 65536 + 65536);
    cudaMemset(base, 1, (size_t)ctas * 65536 + 65536);
    cudaMalloc(&offs, 128); cudaMalloc(&out, ctas * threads * 4); cudaMalloc(&cyc, ctas * 8);
    std::vector<long long> h(ctas);
    printf("%-58s %3s %10s %10s\n", "pattern", "W", "cyc/ld/SM", "ms");
    for (auto& p : pats) {
        cudaMemcpy(offs, p.off, 128, cudaMemcpyHostToDevice);
        cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
        for (int rep = 0; rep < 2; ++rep) {
            cudaEventRecord(e0);
            if (p.w == 4) kern<4><<<ctas, threads>>>(base, offs, iters, out, cyc);
            if (p.w == 8) kern<8><<<ctas, threads>>>(base, offs, iters, out, cyc);
            if (p.w == 16) kern<16><<<ctas, threads>>>(base, offs, iters, out, cyc);
            if (p.w == 32) kern<32><<<ctas, threads>>>(base, offs, iters, out, cyc);
            cudaEventRecord(e1);
            cudaError_t e = cudaDeviceSynchronize();
            if (e != cudaSuccess) { printf("CUDA error %s\n", cudaGetErrorString(e)); return 1; }
        }
        float ms; cudaEventElapsedTime(&ms, e0, e1);
        cudaMemcpy(h.data(), cyc, ctas * 8, cudaMemcpyDeviceToHost);
        double mean = 0; for (auto c : h) mean += c; mean /= ctas;
        // 2 CTAs per SM x 8 warps x iters x 8 loads per SM during `mean` cycles
        double per = mean / (2.0 * 8 * iters * 8);
        printf("%-58s %3d %10.2f %10.3f\n", p.name.c_str(), p.w, per, ms);
    }
    return 0;
}
