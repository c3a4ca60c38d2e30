/*
 * gdrr.h -- C ABI of the B200-native poly-energetic primary-signal projector
 * of gDRR (Jia et al., arXiv 1204.6367, section 2.3).
 *
 * What it computes (Eq. (1) at PAPER.md:147):
 *
 *     P(u) = sum_E  phi_E * w(u) * exp(-mu_bt(E) t_bt(u)) * R_E
 *                   * exp( - sum_m mu_hat_m(E) * LI_m(u) )
 *     LI_m(u) = dl * sum_k  trilinear(rho_m)(x_k),   rho_m = rho * [material == m]
 *
 * where x_k are the MIDPOINTS of intervals of equal length dl laid from the
 * point source along the straight path to the centre of detector pixel u
 * (PAPER.md:151), dl defaults to half the smallest voxel edge,
 * mu(x,E) = rho(x) * mu_hat(material(x), E), the energy integral
 * is a sum over channels, the source is a spectrum phi(E) and a
 * fluence map w(u), the detector is energy integrating with
 * response R(E), and the geometry is the cone-beam gantry of
 * PAPER.md:93-95.  Interpolating per-material density planes and applying
 * mu_hat afterwards is identical to the paper's per-energy interpolation of mu
 * by linearity of the interpolant (reading Q10).
 *
 * Everything runs in hand-written sm_100a CUDA kernels; there is no CPU
 * fallback and no other backend.  Every function returns a status code and
 * never throws or aborts across the ABI.  On error no output is written and
 * gdrr_last_error() describes it.
 *
 * Memory ownership: every "_dev" pointer is DEVICE memory owned by the caller
 * (e.g. a torch tensor) and must stay alive as documented; every other pointer
 * is HOST memory that is copied during the call.  The library itself allocates
 * only the small per-context tables (angles, spectrum, bowtie, fluence map,
 * an error flag).  "cuda_stream" is a cudaStream_t passed as void* (NULL = the
 * legacy default stream).  A context is not thread-safe; distinct contexts are
 * independent.
 *
 * Units: lengths mm, rho g/cm^3, mu_hat mm^-1 per g/cm^3, mu_bt mm^-1.
 * Conventions (readings Q1-Q9): source S = -SAD (cos phi, sin phi, 0);
 * detector origin P = (SDD-SAD)(cos(phi+theta), sin(phi+theta), 0);
 * u_hat = (-sin(phi+theta), cos(phi+theta), 0); v_hat = +z; pixel (i, j) centre
 * at u = (i-(nu-1)/2) du + u_off, v = (j-(nv-1)/2) dv + v_off; voxel (ix,iy,iz)
 * centre at centre + ((ix,iy,iz)-(N-1)/2) * spacing; clamp-to-edge inside the
 * volume box, nothing sampled outside it.
 */
#ifndef GDRR_H
#define GDRR_H

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define GDRR_API __attribute__((visibility("default")))
#else
#define GDRR_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gdrr_context gdrr_context; /* geometry, spectrum tables, last error */
typedef struct gdrr_volume gdrr_volume;   /* refers to a caller-owned device workspace */

enum {
    GDRR_OK = 0,
    GDRR_ERR_INVALID_ARG = -1,
    GDRR_ERR_NOT_READY = -2,   /* geometry or spectrum not set, or they disagree with the volume */
    GDRR_ERR_CUDA = -3,
    GDRR_ERR_WORKSPACE = -4,   /* caller's workspace too small or misaligned */
    GDRR_ERR_UNSUPPORTED = -5
};

/* Device layout of the volume the sampler reads (step a0 of DESIGN.md).  All
 * carry a one-voxel replicated-edge pad, so clamp-to-edge costs no instruction.
 * BRICK and LINEAR hold, per voxel, one fp32 per material (rho at the voxel's
 * own material, 0 elsewhere; vector width 1, 2 or 4 floats), rho bit-exact.
 * PACKED_QUAD (the fast one) holds one 32-bit word per voxel -- with more than
 * one material, fp32 rho rounded to a 21-bit mantissa with the material index
 * and a "pure cell" flag in the three freed bits (|stored - rho| <= 11 ulp =
 * 1.3e-6 relative) -- as overlapping 2x2 (x, y) quads, 16 bytes per voxel. */
enum {
    GDRR_LAYOUT_BRICK = 0,       /* 2x2x2-voxel bricks, x fastest inside a brick, bricks x fastest */
    GDRR_LAYOUT_LINEAR = 1,      /* plain [nz+2][ny+2][nx+2], x fastest */
    GDRR_LAYOUT_PACKED_QUAD = 2  /* quads of packed words, linear with bank-skewed strides */
};

/* How the line integrals of Eq. (1) are evaluated. */
enum {
    GDRR_METHOD_TRILINEAR = 0,   /* the paper's default: fixed-step midpoint rule on the tri-linear field */
    GDRR_METHOD_SIDDON = 1,      /* the paper's option: Siddon's exact radiological path through
                                    homogeneous voxels, LI_m = sum_voxels rho [mat = m] |ray /\ voxel| */
    GDRR_METHOD_TEXTURE = 2      /* the paper's own GPU design: the midpoint rule with the
                                    hardware's 9-bit-weight texture filtering; optional, reported separately,
                                    cannot meet the 1e-4 bar; needs gdrr_volume_attach_texture */
};

/* Which kernel samples a PACKED_QUAD volume with the tri-linear method.  Both give the same
 * numbers to rounding order (the staged one sums in chunks of 16 samples, the gather one of 32). */
enum {
    GDRR_SAMPLER_AUTO = 0,     /* STAGED when the volume's tensor map could be made and the beam of a 16 x 16-pixel
                                  CTA over 16 steps can fit the 14 x 14 x 11-quad box; else GATHER */
    GDRR_SAMPLER_GATHER = 1,   /* quads gathered from global memory through L1 */
    GDRR_SAMPLER_STAGED = 2    /* quads of a CTA's beam staged through shared memory by TMA (a chunk whose beam
                                  does not fit is gathered; GATHER is used if 16 steps exceed 15 voxels) */
};

/* Up to four materials a volume is ONE device volume and gdrr_project one kernel.  More (PAPER.md:97 puts no bound on
 * the material index): the volume is kept as ceil(n / 4) device volumes, one per group of four materials, in each of
 * which the voxels of the other groups are empty; gdrr_project then samples every group (one launch each, writing that
 * group's line integrals) and forms the signal from all line integrals in one more kernel.  Time and workspace grow
 * with the number of groups. */
#define GDRR_MAX_MATERIALS 16
#define GDRR_MAX_ENERGIES 512

/* ---- context ----------------------------------------------------------- */

/* Creates a context bound to CUDA device `cuda_device`.  *out is NULL on error
 * (gdrr_last_error(NULL) then returns the message). */
GDRR_API int gdrr_create_context(int cuda_device, gdrr_context** out);
GDRR_API int gdrr_destroy_context(gdrr_context* ctx);
/* Message of the last failing call on ctx (or of the last failing
 * gdrr_create_context when ctx is NULL).  Valid until the next call. */
GDRR_API const char* gdrr_last_error(const gdrr_context* ctx);

/* ---- volume: step a0, PAPER.md:97 -------------------------------------- */

/* Bytes of device workspace gdrr_create_volume needs for this shape (PACKED_QUAD: 16 B per quad with the
 * skewed strides, rounded to 256, plus 4 B per voxel, rows padded to groups of four, for the Siddon walk's compact copy). */
GDRR_API int gdrr_volume_workspace_bytes(int nx, int ny, int nz, int n_materials, int layout,
                                size_t* bytes);

/* Re-lays (rho, material) into the sampler's layout inside `workspace_dev` with a CUDA kernel on `cuda_stream`
 * and returns WITHOUT waiting for it: the volume can be used at once on any stream (the library orders its own
 * kernels behind the ingest).  The ingest checks material < n_materials on the device; the verdict is read, never
 * waited for, by every later call that takes the volume and finds the ingest finished, and by gdrr_volume_status,
 * which waits.  A volume with a bad material index is refused from then on (INVALID_ARG); what was projected from
 * it before is meaningless but in bounds.
 *   rho_dev       [nz][ny][nx] fp32, x fastest, g/cm^3; borrowed until the ingest has run
 *   material_dev  [nz][ny][nx] uint8; borrowed until the ingest has run
 *   d*_mm         voxel edge lengths; centre_mm = centre of the volume box in
 *                 world coordinates, NULL = the isocentre O
 *   workspace_dev >= gdrr_volume_workspace_bytes, 256-byte aligned, must
 *                 outlive the volume handle
 * Errors: INVALID_ARG (dims, spacings, NULLs), UNSUPPORTED (n_materials > GDRR_MAX_MATERIALS), WORKSPACE, CUDA. */
GDRR_API int gdrr_create_volume(gdrr_context* ctx, const float* rho_dev, const uint8_t* material_dev,
                       int nx, int ny, int nz, double dx_mm, double dy_mm, double dz_mm,
                       const double centre_mm[3], int n_materials, int layout,
                       void* workspace_dev, size_t workspace_bytes, void* cuda_stream,
                       gdrr_volume** out);

/* Same, from HOST arrays (pinned for overlap): copies them into the caller's device staging buffers
 * (rho_stage_dev: nx*ny*nz floats, material_stage_dev: nx*ny*nz bytes) in chunks of z slabs on a stream of the
 * context, behind the work already queued on cuda_stream, and writes the slabs of the device layout that a chunk
 * completes while the next chunk is on the bus.  Asynchronous like gdrr_create_volume; the host arrays must stay
 * valid until cuda_stream has passed this point. */
GDRR_API int gdrr_create_volume_host(gdrr_context* ctx, const float* rho_host,
                            const uint8_t* material_host,
                            int nx, int ny, int nz, double dx_mm, double dy_mm, double dz_mm,
                            const double centre_mm[3], int n_materials, int layout,
                            float* rho_stage_dev, uint8_t* material_stage_dev,
                            void* workspace_dev, size_t workspace_bytes, void* cuda_stream,
                            gdrr_volume** out);

/* Waits for the volume's ingest (and for the Siddon walk's compact copy, if a Siddon projection of this volume has
 * been queued) and returns the verdict: OK, INVALID_ARG (a material index >= n_materials was met), CUDA.  The only
 * call on a volume that blocks the host.  After it has returned OK, gdrr_project on this volume makes no stream call
 * but its kernel launches on cuda_stream (no event is waited for or queried), so it may be issued inside CUDA stream
 * capture and replayed as a graph into the same output buffers (tests/test_gpu_graph.py).  For GDRR_METHOD_SIDDON on a
 * PACKED_QUAD volume, project once before this call: the first Siddon projection makes the compact copy. */
GDRR_API int gdrr_volume_status(gdrr_context* ctx, const gdrr_volume* vol);

/* Frees the handle, never the workspace. */
GDRR_API int gdrr_destroy_volume(gdrr_volume* vol);

/* ---- geometry: PAPER.md:93-95, 282 -------------------------------------- */

/* sad = source-to-axis distance, sdd = source-to-detector distance (AID = sdd -
 * sad), theta = angle between SO and OP, phi_rad[n_proj] = gantry angles
 * (host, copied; their cos/sin are taken here with the host libm and given to
 * the kernels as data), step_mm = dl (<= 0: half the smallest voxel edge of the
 * volume given to gdrr_project).  Requires sdd > sad > 0, positive pixel
 * counts and sizes, n_proj >= 1, finite values. */
GDRR_API int gdrr_set_geometry(gdrr_context* ctx, double sad_mm, double sdd_mm, double theta_rad,
                      int nu, int nv, double du_mm, double dv_mm,
                      double u_offset_mm, double v_offset_mm,
                      int n_proj, const double* phi_rad, double step_mm);

/* General source paths (other scanner geometries "with simple
 * modifications"): instead of the circle, every projection p gives its own pose
 *   poses [n_proj][12] = source S[3], detector origin P[3], u_hat[3], v_hat[3]   (host, copied; world, mm)
 * and pixel (i, j)'s centre is D = (P + u u_hat) + v v_hat with (u, v) as above; the ray, its clipping,
 * the midpoints and everything after are unchanged (reading Q31).  u_hat and v_hat are used
 * as given (expected: unit and orthogonal).  A helix is the circle's pose with S_z and P_z advanced per
 * projection; a C-arm orbit is the circle's poses rotated.  gdrr_set_geometry is this call with
 * S = -SAD (cos phi, sin phi, 0), P = (SDD-SAD)(cos psi, sin psi, 0), u_hat = (-sin psi, cos psi, 0),
 * v_hat = +z, psi = phi + theta, and gives bit-identical results.  The bowtie thickness table stays
 * indexed by the pixel column i.
 * Errors: INVALID_ARG (non-finite values, u_hat x v_hat = 0, source in the detector plane, sizes). */
GDRR_API int gdrr_set_geometry_poses(gdrr_context* ctx, int nu, int nv, double du_mm, double dv_mm,
                            double u_offset_mm, double v_offset_mm,
                            int n_proj, const double* poses, double step_mm);

/* ---- source and detector: PAPER.md:111, 117-121, 147-149 ---------------- */

/*   phi_weight  [n_energy] per-channel spectrum weights, used as given
 *   response    [n_energy] R(E)
 *   mu_hat      [n_materials][n_energy], total over interaction types
 *   fluence_map [nv][nu] w(u) or NULL (= 1); needs gdrr_set_geometry first
 *   bowtie_mu   [n_energy] and bowtie_thickness_mm [nu], both or neither
 * All host, copied.  Values must be finite. */
GDRR_API int gdrr_set_spectrum(gdrr_context* ctx, int n_energy, int n_materials,
                      const double* phi_weight, const double* response, const double* mu_hat,
                      const float* fluence_map, const double* bowtie_mu,
                      const double* bowtie_thickness_mm);

/* Pixel-dependent detector response ("In principle, the detector response could also be pixel
 * dependent.  In our calculation, we ignore this pixel dependence"; reading Q32):
 *   gain [n_energy][nv][nu] fp32 g(E, u), host, copied to a context-owned device table (the library's one other
 *        allocation of detector-sized memory besides the fluence map), or NULL to return to g = 1.
 * The pixel's response becomes r(E, u) = response[E] * g(E, u) in every following gdrr_project; g = 1 gives the bits
 * of the pixel-independent case.  Needs gdrr_set_geometry and gdrr_set_spectrum first (its shape) and is dropped
 * when either changes the detector shape or the number of energy bins.
 * Errors: NOT_READY, INVALID_ARG (a non-finite entry), CUDA. */
GDRR_API int gdrr_set_response_gain(gdrr_context* ctx, const float* gain);

/* ---- projection: steps a1-a7 -------------------------------------------- */

/* Projects projections [proj_begin, proj_begin + proj_count) of the geometry,
 * asynchronously on `cuda_stream`; outputs are valid once the stream reaches
 * this point.
 *   signal_dev         out [proj_count][nv][nu] fp32, required
 *   line_integrals_dev out [proj_count][n_materials][nv][nu] fp32, or NULL (REQUIRED with more than four materials:
 *                      the groups' line integrals wait there for the energy sum)
 *   ray_table_dev      out [proj_count][nv][nu][2] int32 = (j0, n): index of the
 *                      first midpoint inside the box and the number of
 *                      midpoints; n = 0 for a miss; or NULL
 * Rays that miss the box get LI = 0 and the flat-field signal.
 * Errors: NOT_READY (geometry/spectrum unset, material counts differ),
 * INVALID_ARG (range, NULL signal, source inside the volume box), CUDA. */
GDRR_API int gdrr_project(gdrr_context* ctx, const gdrr_volume* vol, int proj_begin, int proj_count,
                 float* signal_dev, float* line_integrals_dev, int32_t* ray_table_dev,
                 void* cuda_stream);

/* Same, delivering the signal into HOST memory: projects in batches into the
 * caller's device scratch `signal_stage_dev` (>= min(proj_count, stage_proj) *
 * nv*nu floats, stage_proj >= 1 projections per batch) and copies each batch to
 * `signal_host` [proj_count][nv][nu]; returns after the last copy completed.
 * For overlap signal_host should be pinned.  With more than four materials the line integrals of a batch wait in a
 * context-owned device scratch (min(proj_count, batch) x n_materials x nv x nu floats, allocated on first use). */
GDRR_API int gdrr_project_host(gdrr_context* ctx, const gdrr_volume* vol, int proj_begin,
                      int proj_count, float* signal_host, float* signal_stage_dev,
                      int stage_proj, void* cuda_stream);

/* Selects the line-integral method of the following gdrr_project calls on ctx
 * (default GDRR_METHOD_TRILINEAR).  GDRR_METHOD_SIDDON ("Siddon's
 * ray-tracing algorithm is also available in gDRR for primary signal
 * calculation"): voxel (ix,iy,iz) is the homogeneous box [lo + i d, lo + (i+1) d)
 * per axis, the path is the source->pixel segment clipped to the volume box,
 * and every voxel contributes rho times the length of the ray inside it to the
 * line integral of its material; the energy sum, the outputs and the ray table
 * (which stays the midpoint table of the geometry) are unchanged.  A ray that
 * lies IN a lattice plane belongs to either neighbour (a tie).  Works on every
 * layout (a PACKED_QUAD workspace carries a compact one-word-per-voxel copy for this walk).
 * Errors: INVALID_ARG (unknown method). */
GDRR_API int gdrr_set_method(gdrr_context* ctx, int method);

/* Optional texture variant.  Copies a GDRR_LAYOUT_LINEAR volume into a 3-D CUDA
 * array (one fp32 channel per material, 1, 2 or 4 channels) and makes a texture object with linear
 * filtering, clamp addressing and unnormalised coordinates.  THE ONE PLACE THE LIBRARY ALLOCATES
 * VOLUME-SIZED DEVICE MEMORY ITSELF (a CUDA array cannot be caller memory); it is freed by
 * gdrr_destroy_volume.  Synchronises cuda_stream.  gdrr_project then uses the texture when the
 * context's method is GDRR_METHOD_TEXTURE.
 * Errors: INVALID_ARG (volume not LINEAR), CUDA. */
GDRR_API int gdrr_volume_attach_texture(gdrr_context* ctx, gdrr_volume* vol, void* cuda_stream);

/* Selects the sampling kernel for PACKED_QUAD volumes (default GDRR_SAMPLER_AUTO).
 * Errors: INVALID_ARG (unknown value). */
GDRR_API int gdrr_set_sampler(gdrr_context* ctx, int sampler);

/* Which kernel the last tri-linear gdrr_project / gdrr_project_host launch on ctx used for a PACKED_QUAD volume:
 * GDRR_SAMPLER_STAGED or GDRR_SAMPLER_GATHER; 0 before the first such launch and after a launch on an exact layout.
 * (What GDRR_SAMPLER_AUTO picks is part of the measured performance: tests/test_gpu_sampler_choice.py pins it.) */
GDRR_API int gdrr_last_sampler(const gdrr_context* ctx);

/* ---- test hooks (never needed by a user; SURVEY.md section 5 race evidence, reading Q9) ------------------- */

/* mode != 0 makes the following staged-sampler launches on ctx run a build of the kernel in which every warp sleeps,
 * before it waits on or signals a barrier of the staging ring, for a time keyed on its number and the chunk:
 * 1 pseudo-random, 2 always the same warp last, 3 the producer warp late.  The images must not change by a bit.
 * mode 0 (default) is the product kernel, which contains none of this.  Errors: INVALID_ARG (mode outside 0..3). */
GDRR_API int gdrr_debug_set_skew(gdrr_context* ctx, int mode);

/* Writes the cell (floor of the index-space position per axis, voxel (ix, iy, iz) = cell whose low corner is that
 * voxel's centre; -1 in the half-voxel rim) of every midpoint sample of the ray through pixel (i, j) of `projection`,
 * formed with the position arithmetic of the kernel named by sampler (GDRR_SAMPLER_GATHER or GDRR_SAMPLER_STAGED), into
 * cells_dev [max_samples][3] int32 (first min(n, max_samples) rows) and the ray's n into *count_dev.  Reading Q9:
 * these may differ from the oracle's fp64 cells only where a position is within 2^-12 of a cell face.
 * Asynchronous on cuda_stream.  Errors: INVALID_ARG, NOT_READY as gdrr_project; volume must be PACKED_QUAD. */
GDRR_API int gdrr_debug_ray_cells(gdrr_context* ctx, const gdrr_volume* vol, int projection, int i, int j, int sampler,
                         int32_t* cells_dev, int max_samples, int32_t* count_dev, void* cuda_stream);

/* Siddon traversal only: writes, per ray of the range, the number of voxel
 * segments of positive length into n_segments_dev [proj_count][nv][nu] int32
 * (0 for a miss).  Asynchronous on cuda_stream. */
GDRR_API int gdrr_siddon_segments(gdrr_context* ctx, const gdrr_volume* vol, int proj_begin,
                         int proj_count, int32_t* n_segments_dev, void* cuda_stream);

/* Ray setup only (step a1): writes the integer ray table and/or adds the
 * number of tri-linear samples sum(n) of the range to *n_samples_dev (a device
 * uint64 the caller zeroed).  Either output may be NULL. */
GDRR_API int gdrr_ray_setup(gdrr_context* ctx, const gdrr_volume* vol, int proj_begin, int proj_count,
                   int32_t* ray_table_dev, unsigned long long* n_samples_dev,
                   void* cuda_stream);

/* ---- scatter denoising: PAPER.md:199-218 (section 2.5) ---------------------- */

/* n_iter relaxed Jacobi sweeps of the paper's Eq. (5) on n_images detector images:
 *   S(k+1) = (1 - omega) S(k) + omega/4 [ Sum S(k) - 1/beta (1 - S_hat / S(k)) ],  S(0) = S_hat,
 * Sum = the four edge neighbours, all of sweep k.  Outside the detector the nearest pixel inside is
 * used (replicated edge); S is kept >= floor_value > 0 (S(0) = max(S_hat, floor), every iterate
 * clamped) so that empty Monte Carlo pixels are defined.  The paper uses omega = 0.8.
 *   s_hat_dev    in  [n_images][nv][nu] fp32 (the noisy scatter image)
 *   s_dev        out [n_images][nv][nu] fp32
 *   scratch_dev  work, same size as s_dev
 * Asynchronous on cuda_stream.  Errors: INVALID_ARG (NULLs, sizes, beta <= 0, floor <= 0, n_iter < 0,
 * omega outside (0, 2)), CUDA. */
GDRR_API int gdrr_denoise_scatter(gdrr_context* ctx, const float* s_hat_dev, float* s_dev, float* scratch_dev,
                         int nu, int nv, int n_images, double beta, double omega, int n_iter,
                         double floor_value, void* cuda_stream);

/* The same sweeps for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): no scratch_dev argument, and the call makes no cudaMalloc, cudaFree or allocating
 * library call.  The scratch image is a static array inside the library: every GPU that loads the library holds
 * GDRR_DENOISE_STATIC_MAX_FLOATS x 4 bytes (16 MiB) of it until the process exits.
 *   s_hat_dev, s_dev   as for gdrr_denoise_scatter (the caller's buffers; s_dev receives the result)
 * Limit: nu * nv * n_images <= GDRR_DENOISE_STATIC_MAX_FLOATS (e.g. 21 images of 512 x 384), else UNSUPPORTED with a
 * message that names the limit; other errors as gdrr_denoise_scatter.  Results are bit-identical to gdrr_denoise_scatter.
 * ALL calls, on all contexts and streams of a GPU, share the one array, and it keeps the last call's contents (which
 * no call reads: every launch writes each pixel of its destination before a later launch reads it, so nothing has to
 * start at zero).  Calls that overlap on the GPU (different streams, concurrent graph replays) RACE on it: issue them
 * on one stream, or order them yourself.  The first call on a device resolves the array's address there
 * (cudaGetSymbolAddress, once per device): make that first call outside stream capture. */
#define GDRR_DENOISE_STATIC_MAX_FLOATS 4194304
GDRR_API int gdrr_denoise_scatter_static(gdrr_context* ctx, const float* s_hat_dev, float* s_dev,
                                int nu, int nv, int n_images, double beta, double omega, int n_iter,
                                double floor_value, void* cuda_stream);

/* Number of kernels this library has launched on ctx since creation (for the
 * harness's gpu_launches count). */
GDRR_API unsigned long long gdrr_kernel_launches(const gdrr_context* ctx);

/* Library version, "major.minor". */
GDRR_API const char* gdrr_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GDRR_H */
