// Internal declarations shared by the translation units of libgdrr_b200.so.
// Not part of the ABI (include/gdrr.h is).  Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gdrr {

// Tile of detector pixels one CTA owns: 16 x 16, eight warps (8 (u) x 4 (v) pixels
// each in the exact-layout kernels, 4 x 8 in the packed sampler).
constexpr int kTileU = 16;
constexpr int kTileV = 16;
constexpr int kThreads = kTileU * kTileV;
// staged sampler (project_staged.cu; the tensor map is made in gdrr_api.cu): the same 16 x 16 tile sampled by 8 consumer
// warps, plus one producer warp; two staged boxes of kBX x kBY x kBZ quads; 3 CTAs per SM
// (measured on C3: a 16 x 8 tile with a 14 x 14 x 7 box, 4 CTAs per SM: -8%)
#define GDRR_STAGE_CTAS 3
constexpr int kStageTileV = 16;
constexpr int kStageThreads = kTileU * kStageTileV;
constexpr int kBX = 14, kBY = 14, kBZ = 11;       // box, in quads
constexpr int kMaxChunk = 32;       // samples between two fp64 re-bases of the position
constexpr int kFracBits = 23;       // fixed-point fraction bits of the in-chunk position

// Everything the ray-setup arithmetic (step a1) needs.  All fp64; the order of
// operations in ray_setup.cuh is part of the definition of (j0, n).
struct GeomParams {
    double half_nu, half_nv;        // 0.5 * (nu - 1), 0.5 * (nv - 1)
    double du, dv, u_off, v_off;
    double step;                    // dl
    double lo[3], hi[3];            // volume box
    double c[3], d[3];              // box centre, voxel size
    double inv_d[3];                // 1 / d (host): the index-space line is formed with multiplications
    double ofs[3];                  // 0.5 * (N - 1) + 1: world -> padded index coordinates
    const double* poses;            // [n_proj][12] source S, detector origin P, u_hat, v_hat; device
    int nu, nv;
    int proj_begin, proj_count;
};

struct VolumeParams {
    const void* vox;                // device, layout below
    const void* vox1;               // PACKED_QUAD: vox + one slab (its own parameter: one IMAD.WIDE per load)
    int stride_y;                   // BRICK: 8 * bricks per row;   LINEAR: stored nx;      PACKED_QUAD: elements per row (= 3 mod 8)
    int nvox[3];                    // nx, ny, nz (Siddon traversal)
    const void* compact;            // PACKED_QUAD: one tagged word per voxel, rows in groups of four (Siddon walk)
    int cstride_y, cstride_z;       //   words per group of four rows (4 nx), per slab
    int stride_z;                   // BRICK: 8 * bricks per slab;  LINEAR: stored nx * ny; PACKED_QUAD: elements per slab (= 4 mod 8)
};

struct ProjectParams {
    GeomParams g;
    VolumeParams v;
    const float4* mu_tab;           // [n_energy] log2(e) * mu_hat[m = 0..3][E]
    const float2* src_tab;          // [n_energy] (phi_E * R_E, log2(e) * mu_bt[E])
    const float* bt_thick;          // [nu] or nullptr
    const float* fluence;           // [nv][nu] or nullptr
    const float* gain;              // [n_energy][nv][nu] pixel-dependent response gain g(E, u) or nullptr (reading Q32)
    int n_energy, n_mat;            // n_mat: materials of THIS device volume (<= 4; a group of the caller's materials)
    // more than four materials: the volume is kept as groups of four (gdrr_api.cu); a launch then only writes its
    // group's line integrals (li_only) at material offset li_mat0 of the caller's [proj][li_mat_total][nv][nu] array,
    // and gdrr_energy_sum_kernel forms the signal from all of them with mu_all
    int li_only, li_mat0, li_mat_total;
    const float* mu_all;            // [n_energy][li_mat_total] log2(e) * mu_hat, or nullptr (<= 4 materials)
    int chunk;                      // <= kMaxChunk
    unsigned frac_mask, one_bits;   // 0x007FFFFF, 0x3F800000: kept in registers by the samplers
    // staged sampler: bound, in voxels per axis, on how far a ray of a 16 x 16-pixel tile can lie outside the hull of
    // the tile's four corner rays at equal interval index (curvature of the equal-index surface plus the
    // fixed-point slack of the sampler's positions); gdrr_api.cu hull_margins()
    double hull_margin[3];
    unsigned debug_skew;            // tests only (gdrr_debug_set_skew): forced warp orders in the staged kernel, 0 = off
    float* signal;                  // [proj_count][nv][nu]
    float* li;                      // [proj_count][n_mat][nv][nu] or nullptr
    int32_t* ray_table;             // [proj_count][nv][nu][2] or nullptr
    int32_t* seg_table;             // Siddon only: [proj_count][nv][nu] segments of positive length, or nullptr
};

struct IngestParams {
    const float* rho;               // [nz][ny][nx]
    const uint8_t* mat;
    void* vox;
    int nx, ny, nz;
    int px, py, pz;                 // stored dims (voxels for BRICK / LINEAR, quads for PACKED_QUAD)
    int ez0, ezn;                   // stored slabs [ez0, ez0 + ezn) to write in this launch (BRICK: always all of them)
    int sy, sz;                     // PACKED_QUAD: element strides (VolumeParams)
    void* compact;                  // PACKED_QUAD: the one-word-per-voxel copy, rows in groups of four
    int cbx, cby;                   //   ceil(nx / 4), ceil(ny / 4) (cby: groups of four rows per slab)
    int n_mat;                      // the caller's material count: an index >= n_mat raises bad_flag
    int mat_lo, n_group;            // this device volume holds materials [mat_lo, mat_lo + n_group) as tags 0..n_group-1;
                                    // voxels of other materials are stored as rho = 0 (tag 0): they add nothing to any sum
    int tagged;                     // PACKED_QUAD: words carry tags (n_group > 1)
    int* bad_flag;                  // set to 1 if a material index >= n_mat is seen
};

// Host-callable launchers (each returns the cudaGetLastError() of its launch).
cudaError_t launch_ingest(const IngestParams& p, int vw, int layout, cudaStream_t s);
// PACKED_QUAD: fills p.compact (one word per voxel, rows in groups of four) from the quads in p.vox; needs nx..nz, sy, sz, cbx, cby, n_mat
cudaError_t launch_compact_copy(const IngestParams& p, cudaStream_t s);
cudaError_t launch_project_exact(const ProjectParams& p, int vw, int layout, cudaStream_t s);
cudaError_t launch_project_packed(const ProjectParams& p, int vw, cudaStream_t s);
// tensor_map: a CUtensorMap over the packed-quad volume (3-D: words along x, rows, slabs; box 4*14 x 14 x 11);
// launches kStageThreads + 32 threads per CTA (the consumer warps and the producer warp)
cudaError_t launch_project_staged(const ProjectParams& p, int vw, const void* tensor_map, cudaStream_t s);
cudaError_t launch_project_texture(const ProjectParams& p, int vw, unsigned long long tex_object, cudaStream_t s);
cudaError_t launch_project_siddon(const ProjectParams& p, int vw, int layout, cudaStream_t s);
// tests only: cells of every sample of ray (i, j) of projection p.g.proj_begin as the staged (or gather) kernel forms them
cudaError_t launch_debug_ray_cells(const ProjectParams& p, int i, int j, int staged, int32_t* cells, int max_samples,
                                   int32_t* count, cudaStream_t s);
cudaError_t launch_ray_setup(const GeomParams& g, int32_t* ray_table,
                             unsigned long long* n_samples, cudaStream_t s);

// more than four materials: signal from the line integrals of all groups (energy_sum.cu)
cudaError_t launch_energy_sum(const ProjectParams& p, cudaStream_t s);
cudaError_t launch_denoise(const float* s_hat, float* s_dev, float* scratch, int nu, int nv, int n_images,
                           double beta, double omega, int n_iter, double floor_value, cudaStream_t st, int* launches);

}  // namespace gdrr
