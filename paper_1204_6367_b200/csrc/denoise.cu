// Scatter denoising: relaxed Jacobi sweeps of the paper's Eq. (5),
//   S(k+1) = (1 - w) S(k) + w/4 [ Sum S(k) - 1/beta (1 - S_hat / S(k)) ],   S(0) = S_hat,
// with replicated edges [Q28] and a positive floor [Q29].  A detector image is small
// (512 x 384) and a sweep is 12 bytes of traffic per pixel, so one launch per sweep would be bound
// by launch latency (one image) or HBM (a scan of images).  Here a CTA loads a tile of S and S_hat
// with a halo of kSweeps pixels into shared memory and performs up to kSweeps sweeps on it: cells
// next to a tile edge that is not an image edge go stale one ring per sweep, and after t sweeps
// the cells at least t away from such edges are exact; those include the CTA's output tile.
// At an image edge the tile ends with the image and clamping the neighbour index to the tile IS
// the replicated edge.  fp32 arithmetic; S_hat / S by reciprocal and multiply (2 ulp, far inside the tolerance).
#include <mutex>

#include "denoise_static.h"
#include "gdrr_internal.h"

namespace gdrr {

constexpr int kDnTileW = 128, kDnTileH = 32, kSweeps = 4;
constexpr int kDnW = kDnTileW + 2 * kSweeps, kDnH = kDnTileH + 2 * kSweeps;     // 136 x 40 cells

struct DenoiseParams {
    const float* s_hat;     // [n_images][nv][nu]
    const float* src;       // S(k) (== s_hat for the first launch: S(0) = max(S_hat, floor))
    float* dst;             // S(k + sweeps)
    int nu, nv;
    int sweeps;             // 1 .. kSweeps
    float one_minus_w, w4, inv_beta, floor_value;
};

constexpr int kDnRows = 4;                        // threads: kDnW columns x kDnRows; a thread owns kDnH / kDnRows cells of a column
constexpr int kDnPer = kDnH / kDnRows;

__global__ void __launch_bounds__(kDnW * kDnRows)
gdrr_denoise_kernel(const DenoiseParams P) {
    __shared__ float s_a[kDnH][kDnW], s_b[kDnH][kDnW];
    const size_t img = (size_t)blockIdx.z * P.nu * P.nv;
    const int x0 = blockIdx.x * kDnTileW, y0 = blockIdx.y * kDnTileH;
    // the tile's cells that exist: [xa, xb) x [ya, yb) in image coordinates
    const int xa = max(x0 - kSweeps, 0), xb = min(x0 + kDnTileW + kSweeps, P.nu);
    const int ya = max(y0 - kSweeps, 0), yb = min(y0 + kDnTileH + kSweeps, P.nv);
    const int w = xb - xa, h = yb - ya;
    const int lx = threadIdx.x, ty = threadIdx.y;
    const bool col = lx < w;
    const int lxp = min(lx + 1, w - 1), lxm = max(lx - 1, 0);
    float hat[kDnPer];                             // S_hat of this thread's cells stays in registers
#pragma unroll
    for (int r = 0; r < kDnPer; ++r) {
        const int ly = ty + r * kDnRows;
        hat[r] = 0.f;
        if (col && ly < h) {
            const size_t g = img + (size_t)(ya + ly) * P.nu + (xa + lx);
            s_a[ly][lx] = fmaxf(P.src[g], P.floor_value);
            hat[r] = P.s_hat[g];
        }
    }
    __syncthreads();
    float (*cur)[kDnW] = s_a;
    float (*nxt)[kDnW] = s_b;
    for (int t = 0; t < P.sweeps; ++t) {
#pragma unroll
        for (int r = 0; r < kDnPer; ++r) {
            const int ly = ty + r * kDnRows;
            if (col && ly < h) {
                const float s = cur[ly][lx];
                const float sum = cur[ly][lxp] + cur[min(ly + 1, h - 1)][lx] + cur[ly][lxm] + cur[max(ly - 1, 0)][lx];
                const float v = P.one_minus_w * s + P.w4 * (sum - P.inv_beta * (1.f - __fdividef(hat[r], s)));
                nxt[ly][lx] = fmaxf(v, P.floor_value);
            }
        }
        __syncthreads();
        float (*tmp)[kDnW] = cur; cur = nxt; nxt = tmp;
    }
    // the output tile
    const int ox = x0 - xa, oy = y0 - ya;
    const int tw = min(kDnTileW, P.nu - x0), th = min(kDnTileH, P.nv - y0);
#pragma unroll
    for (int r = 0; r < kDnPer; ++r) {
        const int ly = ty + r * kDnRows;
        if (lx >= ox && lx < ox + tw && ly >= oy && ly < oy + th)
            P.dst[img + (size_t)(ya + ly) * P.nu + (xa + lx)] = cur[ly][lx];
    }
}

// n_iter sweeps of every image; the result ends in s_dev.  Returns the number of launches through *launches.
cudaError_t launch_denoise(const float* s_hat, float* s_dev, float* scratch, int nu, int nv, int n_images,
                           double beta, double omega, int n_iter, double floor_value, cudaStream_t st, int* launches) {
    *launches = 0;
    DenoiseParams p;
    p.s_hat = s_hat; p.nu = nu; p.nv = nv;
    p.one_minus_w = (float)(1.0 - omega); p.w4 = (float)(omega / 4.0); p.inv_beta = (float)(1.0 / beta);
    p.floor_value = (float)floor_value;
    dim3 grid((nu + kDnTileW - 1) / kDnTileW, (nv + kDnTileH - 1) / kDnTileH, n_images);
    const int n_launch = n_iter > 0 ? (n_iter + kSweeps - 1) / kSweeps : 1;
    // ping-pong so that the last launch writes s_dev
    float* bufs[2] = {s_dev, scratch};
    int which = (n_launch & 1) ? 0 : 1;         // destination of the first launch
    const float* src = s_hat;
    int left = n_iter;
    for (int l = 0; l < n_launch; ++l) {
        p.src = src;
        p.dst = bufs[which];
        p.sweeps = left < kSweeps ? left : kSweeps;      // 0 when n_iter == 0: S = max(S_hat, floor)
        gdrr_denoise_kernel<<<grid, dim3(kDnW, kDnRows), 0, st>>>(p);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        ++*launches;
        left -= p.sweeps;
        src = bufs[which];
        which ^= 1;
    }
    return cudaSuccess;
}

// ---- gdrr_denoise_scatter_static: the same sweeps for callers that cannot allocate (include/gdrr.h) ----------------
// The ping-pong scratch image is this file-scope array instead of a caller's buffer.  Every GPU that loads the library
// holds its kDenoiseStaticFloats x 4 B (16 MiB) from the first use of the module until the process exits.
// In HOST code the name `g_denoise_scratch` is a host-side stand-in, not a device address: the address the kernel gets
// is the one cudaGetSymbolAddress returns on the current device, resolved here once per device.
// Nothing in it has to start at zero: a launch writes every pixel of its destination image before any later launch
// reads it, and the call's result ends in the caller's s_dev, so the contents a previous call left are never read.
// All calls share the one array: two calls that overlap on a GPU (different streams, or graphs replayed concurrently) race.
static __device__ __align__(256) float g_denoise_scratch[kDenoiseStaticFloats];

constexpr int kMaxDevices = 64;

cudaError_t launch_denoise_static(const float* s_hat, float* s_dev, int nu, int nv, int n_images, double beta, double omega,
                                  int n_iter, double floor_value, cudaStream_t st, int* launches) {
    static std::mutex mu;
    static float* addr[kMaxDevices] = {};           // device address of g_denoise_scratch, per device ordinal
    *launches = 0;
    if ((size_t)nu * (size_t)nv * (size_t)n_images > kDenoiseStaticFloats) return cudaErrorInvalidValue;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    float* scratch = nullptr;
    {
        std::lock_guard<std::mutex> lock(mu);
        if (!addr[dev]) {                            // set-up, once per device, with that device current
            float* p = nullptr;
            e = cudaGetSymbolAddress((void**)&p, g_denoise_scratch);
            if (e != cudaSuccess) return e;
            addr[dev] = p;
        }
        scratch = addr[dev];
    }
    return launch_denoise(s_hat, s_dev, scratch, nu, nv, n_images, beta, omega, n_iter, floor_value, st, launches);
}

}  // namespace gdrr
