// Step a0: volume ingest ("material type and density at each voxel").
//
// Turns (rho fp32, material u8) [nz][ny][nx] into the layout the sampler reads:
// per voxel VW floats (rho in the slot of the voxel's material, 0 elsewhere),
// with a one-voxel replicated-edge pad (so clamp-to-edge, reading Q7, needs no
// instruction in the sampler), stored either as 2x2x2 bricks or linearly.
// One thread per stored voxel, stores coalesced in storage order.
#include "gdrr_internal.h"

namespace gdrr {

template <int VW> struct VoxT;
template <> struct VoxT<1> { using T = float; };
template <> struct VoxT<2> { using T = float2; };
template <> struct VoxT<4> { using T = float4; };

template <int VW>
__device__ __forceinline__ typename VoxT<VW>::T one_hot(float rho, int m);
template <> __device__ __forceinline__ float one_hot<1>(float rho, int) { return rho; }
template <> __device__ __forceinline__ float2 one_hot<2>(float rho, int m) {
    return make_float2(m == 0 ? rho : 0.f, m == 1 ? rho : 0.f);
}
template <> __device__ __forceinline__ float4 one_hot<4>(float rho, int m) {
    return make_float4(m == 0 ? rho : 0.f, m == 1 ? rho : 0.f, m == 2 ? rho : 0.f,
                       m == 3 ? rho : 0.f);
}

template <int VW, int LAYOUT>
__global__ void __launch_bounds__(256)
gdrr_ingest_kernel(const IngestParams P) {
    using V = typename VoxT<VW>::T;
    // stored slabs [ez0, ez0 + ezn) of the padded volume (LINEAR), or everything (BRICK: ez0 = 0, ezn = pz)
    const size_t first = (size_t)P.px * P.py * P.ez0, total = (size_t)P.px * P.py * (P.ez0 + P.ezn);
    const size_t o = first + (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (o >= total) return;
    int sx_, sy_, sz_;      // stored (padded) coordinates of element o
    if (LAYOUT == 0) {
        const int e = (int)(o & 7);
        size_t b = o >> 3;
        const int nbx = P.px >> 1, nby = P.py >> 1;
        const int bx = (int)(b % nbx);
        b /= nbx;
        const int by = (int)(b % nby);
        const int bz = (int)(b / nby);
        sx_ = 2 * bx + (e & 1);
        sy_ = 2 * by + ((e >> 1) & 1);
        sz_ = 2 * bz + (e >> 2);
    } else {
        size_t t = o;
        sx_ = (int)(t % P.px);
        t /= P.px;
        sy_ = (int)(t % P.py);
        sz_ = (int)(t / P.py);
    }
    // stored index s <-> voxel s - 1, clamped to the lattice (replicated edge)
    const int ix = min(max(sx_ - 1, 0), P.nx - 1);
    const int iy = min(max(sy_ - 1, 0), P.ny - 1);
    const int iz = min(max(sz_ - 1, 0), P.nz - 1);
    const size_t src = ((size_t)iz * P.ny + iy) * P.nx + ix;
    const int m = P.mat[src];
    if (m >= P.n_mat) *P.bad_flag = 1;
    // a voxel whose material belongs to another group of four is an empty voxel of this device volume
    const int local = m - P.mat_lo;
    const bool here = (unsigned)local < (unsigned)P.n_group;
    reinterpret_cast<V*>(P.vox)[o] = one_hot<VW>(here ? P.rho[src] : 0.f, here ? local : 0);
}

// PACKED_QUAD (project_packed.cu): element (ex, ey, ez) = the four words of stored
// voxels (ex, ey), (ex, ey+1), (ex+1, ey), (ex+1, ey+1) of slab ez.  With more than
// one material a word is rho rounded to a 21-bit mantissa with tags in the three
// freed bits: bits 0-1 the material index; bit 2 describes cell (ex, ey, ez), whose 8
// corners are this quad and the one above it in slab ez + 1: in the first word "all 8
// corners have this material"; in the second word "the 8 corners have exactly two
// materials", the one that is not the first word's then in bit 2 of the fourth (its
// bit 1) and third (its bit 0) words.  Elements are stored linearly with strides sy, sz.
// One thread per element slot; slots that are stride padding are zeroed.  Grid: x over a row's sy slots
// (+ the few pad slots between the last row and the slab pitch, taken by the blocks of the last row),
// y = row, z = slab: no division in the index arithmetic.
__global__ void __launch_bounds__(256)
gdrr_ingest_packed_kernel(const IngestParams P) {
    const int ez = P.ez0 + blockIdx.z, ey = blockIdx.y;
    int ex = blockIdx.x * blockDim.x + threadIdx.x;
    const int row_slots = (ey == P.py - 1) ? P.sz - ey * P.sy : P.sy;      // the last row also owns the slab's tail pad
    if (ex >= row_slots) return;
    const size_t o = (size_t)ez * P.sz + (size_t)ey * P.sy + ex;
    uint4 out = make_uint4(0u, 0u, 0u, 0u);
    if (ex < P.px && ey < P.py) {
        unsigned w[4];
        unsigned mixed = 0u, m0 = 0u, seen = 0u;        // seen: bit m set if a corner has material m
#pragma unroll
        for (int dz = 0; dz < 2; ++dz) {
            const int iz = min(max(ez + dz - 1, 0), P.nz - 1);
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const int ix = min(max(ex + (k >> 1) - 1, 0), P.nx - 1);
                const int iy = min(max(ey + (k & 1) - 1, 0), P.ny - 1);
                const size_t src = ((size_t)iz * P.ny + iy) * P.nx + ix;
                const unsigned mg = P.mat[src];
                if ((int)mg >= P.n_mat) *P.bad_flag = 1;
                // a voxel whose material belongs to another group of four is an empty voxel (tag 0) of this device volume
                const bool here = mg - (unsigned)P.mat_lo < (unsigned)P.n_group;
                const unsigned m = here ? mg - (unsigned)P.mat_lo : 0u;
                if (dz == 0 && k == 0) m0 = m;
                mixed |= m ^ m0;
                seen |= 1u << (m & 3u);
                if (dz == 0) {
                    unsigned bits = here ? __float_as_uint(P.rho[src]) : 0u;
                    if (P.tagged) bits = ((bits + 4u) & ~7u) | (m & 3u);
                    w[k] = bits;
                }
            }
        }
        if (P.tagged && mixed == 0u) w[0] |= 4u;
        if (P.tagged && __popc(seen) == 2) {
            const unsigned q = (unsigned)(__ffs((int)(seen & ~(1u << (m0 & 3u)))) - 1);     // the other material
            w[1] |= 4u;
            w[2] |= (q & 1u) << 2;
            w[3] |= (q & 2u) << 1;
        }
        out = make_uint4(w[0], w[1], w[2], w[3]);
    }
    reinterpret_cast<uint4*>(P.vox)[o] = out;
}

// The same, FOUR consecutive elements of a row per thread, for volumes whose rows are 4-voxel aligned (nx % 4 == 0,
// aligned input pointers: launch_ingest checks).  The four elements need voxel columns ex0 - 1 .. ex0 + 3 of two rows in
// two slabs; away from the volume's faces that is one aligned 4-byte word of materials plus one byte, and one float4 of
// densities plus one float, per row and slab: 12 loads for four elements where the kernel above issues 48.  Each
// voxel's material is mapped once (the kernel above: up to four times), the set of materials of a cell is the OR of two
// per-COLUMN sets (a column = the 2 x 2 voxels of one x), and the range check looks at the four voxels this thread
// alone owns (slab ez - 1, row ey - 1, columns ex0 .. ex0 + 3: every voxel has exactly one such owner, and at the
// faces a few more).  A block is 32 threads (x) by kIngestRows rows: neighbouring rows find each other's voxels in L1
// (measured on C3, ms per ingest: 2 rows 0.341, 4 rows 0.345, 8 rows 0.355; the round's first form of this kernel 0.529).
// Bit-identical output (tests/test_gpu_ingest.py).
// GROUPED: the device volume is one of a chain of material groups (mat_lo / n_group map the caller's index to a tag);
// else tag = material index.
constexpr int kIngestRows = 2;
template <bool GROUPED>
__global__ void __launch_bounds__(32 * kIngestRows)
gdrr_ingest_packed4_kernel(const IngestParams P) {
    const int ez = P.ez0 + blockIdx.z, ey = kIngestRows * blockIdx.y + threadIdx.y;
    const int ex0 = 4 * (blockIdx.x * 32 + threadIdx.x);
    if (ey >= P.py) return;
    const int row_slots = (ey == P.py - 1) ? P.sz - ey * P.sy : P.sy;      // the last row also owns the slab's tail pad
    if (ex0 >= row_slots) return;
    uint4 out[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) out[e] = make_uint4(0u, 0u, 0u, 0u);
    if (ex0 < P.px) {
        unsigned colset[5] = {0u, 0u, 0u, 0u, 0u};     // bit m: one of the column's four voxels has tag m
        unsigned tag0[5];                              // tag of (slab 0, row 0, column)
        unsigned bits[2][5];                           // [row][column]: word of slab 0 (rho, tagged)
        bool bad = false;
        // One path for every thread (no divergence at the ends of a row).  Column c is voxel ex0 - 1 + c, clamped to the
        // lattice.  nx % 4 == 0, so the aligned word [ex0, ex0 + 3] lies inside the row for every ex0 < nx.  The last
        // element column (ex0 == nx) stores element 0 only, whose columns 0 and 1 are both voxel nx - 1: column 1
        // repeats column 0 there, and columns 2 .. 4 (the row's last word, so that the load stays in bounds) go unused.
        // Column 0 is a load of its own at max(ex0 - 1, 0).  (Offsets in int: launch_ingest's caller has checked that
        // the padded volume fits int32 indexing.)
        const int x_left = max(ex0 - 1, 0), x_word = min(ex0, P.nx - 4);
        const bool past_end = ex0 >= P.nx;
#pragma unroll
        for (int dz = 0; dz < 2; ++dz) {
            const int iz = min(max(ez + dz - 1, 0), P.nz - 1);
#pragma unroll
            for (int row = 0; row < 2; ++row) {
                const int iy = min(max(ey + row - 1, 0), P.ny - 1);
                const int base = (iz * P.ny + iy) * P.nx;
                unsigned mg[5];
                float rh[5];
                mg[0] = P.mat[base + x_left];
                const unsigned wd = *reinterpret_cast<const unsigned*>(P.mat + (base + x_word));
                mg[1] = past_end ? mg[0] : (wd & 0xffu);
                mg[2] = (wd >> 8) & 0xffu;
                mg[3] = (wd >> 16) & 0xffu;
                mg[4] = wd >> 24;
                if (dz == 0) {
                    rh[0] = P.rho[base + x_left];
                    const float4 f = *reinterpret_cast<const float4*>(P.rho + (base + x_word));
                    rh[1] = past_end ? rh[0] : f.x;
                    rh[2] = f.y; rh[3] = f.z; rh[4] = f.w;
                }
#pragma unroll
                for (int c = 0; c < 5; ++c) {
                    if (dz == 0 && row == 0 && c > 0) bad = bad || (int)mg[c] >= P.n_mat;      // the voxels this thread owns
                    // a voxel whose material belongs to another group of four is an empty voxel (tag 0) of this device volume
                    const unsigned local = GROUPED ? mg[c] - (unsigned)P.mat_lo : mg[c];
                    const bool here = local < (unsigned)P.n_group;
                    const unsigned m = here ? local : 0u;
                    colset[c] |= 1u << m;
                    if (dz == 0) {
                        if (row == 0) tag0[c] = m;
                        unsigned b = here ? __float_as_uint(rh[c]) : 0u;
                        if (P.tagged) b = ((b + 4u) & ~7u) | m;
                        bits[row][c] = b;
                    }
                }
            }
        }
        if (bad) *P.bad_flag = 1;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            if (ex0 + e < P.px) {
                // element ex0 + e: words (x0y0, x0y1, x1y0, x1y1) = columns e, e + 1 of the two rows
                unsigned w[4] = {bits[0][e], bits[1][e], bits[0][e + 1], bits[1][e + 1]};
                if (P.tagged) {
                    const unsigned seen = colset[e] | colset[e + 1];
                    const int n_seen = __popc(seen);
                    if (n_seen == 1) w[0] |= 4u;
                    if (n_seen == 2) {
                        const unsigned q = (unsigned)(__ffs((int)(seen & ~(1u << tag0[e]))) - 1);     // the other material
                        w[1] |= 4u;
                        w[2] |= (q & 1u) << 2;
                        w[3] |= (q & 2u) << 1;
                    }
                }
                out[e] = make_uint4(w[0], w[1], w[2], w[3]);
            }
        }
    }
    uint4* dst = reinterpret_cast<uint4*>(P.vox) + ((size_t)ez * P.sz + (size_t)ey * P.sy + ex0);
#pragma unroll
    for (int e = 0; e < 4; ++e)
        if (ex0 + e < row_slots) dst[e] = out[e];
}

// PACKED_QUAD, second copy for the Siddon walk (project_siddon.cu), made from the quads the first time the
// Siddon method is used on a volume: the same tagged word per voxel (no pad, no purity flag), stored once, with the
// rows in groups of four: word (ix, iy, iz) sits at  iz * SZ + (iy >> 2) * SY + 4 ix + (iy & 3),  SY = 4 nx,
// SZ = SY * ceil(ny / 4).  A 128-byte line is 8 (x) x 4 (y) voxels: a walk along x or along y finds 8 or 4 of its
// voxels in a line, and a step along x or z adds a constant to the offset (a step along y: 1, or SY - 3 across a
// group's edge).  Measured against 4 x 4 x 2 bricks (offset recomputed from the indices): +14% over a scan,
// the same speed at every gantry angle; plain linear rows: +13% over a scan but -16% where the rays run along y.
// One thread per stored word.
__global__ void __launch_bounds__(256)
gdrr_ingest_compact_kernel(const IngestParams P) {
    // grid: x over the 4 nx words of a group of rows, y = group of rows, z = slab
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= 4 * P.nx) return;
    const int ix = t >> 2, iy = 4 * blockIdx.y + (t & 3), iz = blockIdx.z;
    unsigned bits = 0u;
    if (iy < P.ny) {
        // voxel (ix, iy, iz) is the first word of quad (ix + 1, iy + 1, iz + 1); drop its purity flag
        bits = reinterpret_cast<const unsigned*>(P.vox)[4 * ((size_t)(iz + 1) * P.sz + (size_t)(iy + 1) * P.sy + (ix + 1))];
        if (P.tagged) bits &= ~4u;
    }
    reinterpret_cast<unsigned*>(P.compact)[((size_t)iz * P.cby + blockIdx.y) * (4 * (size_t)P.nx) + t] = bits;
}

template <int VW, int LAYOUT>
static cudaError_t launch_ingest_t(const IngestParams& p, cudaStream_t s) {
    const size_t total = (size_t)p.px * p.py * p.ezn;
    const unsigned int blocks = (unsigned int)((total + 255) / 256);
    gdrr_ingest_kernel<VW, LAYOUT><<<blocks, 256, 0, s>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_compact_copy(const IngestParams& p, cudaStream_t s) {
    gdrr_ingest_compact_kernel<<<dim3((4 * p.nx + 255) / 256, p.cby, p.nz), 256, 0, s>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_ingest(const IngestParams& p, int vw, int layout, cudaStream_t s) {
    if (layout == 2) {
        // (py and pz, cby and nz stay far below the 65535 limit of grid.y / grid.z for any volume that fits int32 indexing)
        const int row_max = p.sy + 8;                                   // a row, or the last row plus the slab's tail pad
        if (p.nx % 4 == 0 && (uintptr_t)p.mat % 4 == 0 && (uintptr_t)p.rho % 16 == 0) {
            // four elements per thread, vector loads; 32 threads = 128 elements of a row per block (a C2 row is 257 + pad)
            const dim3 grid((row_max + 127) / 128, (p.py + kIngestRows - 1) / kIngestRows, p.ezn), block(32, kIngestRows);
            if (p.mat_lo == 0) gdrr_ingest_packed4_kernel<false><<<grid, block, 0, s>>>(p);
            else gdrr_ingest_packed4_kernel<true><<<grid, block, 0, s>>>(p);
            return cudaGetLastError();
        }
        // (64 threads per block: a row of 257 + pad slots, C2, wastes 17% of its threads instead of 48% with 256)
        gdrr_ingest_packed_kernel<<<dim3((row_max + 63) / 64, p.py, p.ezn), 64, 0, s>>>(p);
        return cudaGetLastError();
    }
    if (layout == 0) {
        if (vw == 1) return launch_ingest_t<1, 0>(p, s);
        if (vw == 2) return launch_ingest_t<2, 0>(p, s);
        return launch_ingest_t<4, 0>(p, s);
    }
    if (vw == 1) return launch_ingest_t<1, 1>(p, s);
    if (vw == 2) return launch_ingest_t<2, 1>(p, s);
    return launch_ingest_t<4, 1>(p, s);
}

}  // namespace gdrr
