// Host side of the C ABI declared in include/gdrr.h: argument validation, the
// small context-owned device tables, and kernel launches.  No arithmetic of the
// method happens here except what the header says is done on the host: cos/sin
// of the gantry angles (given to the kernels as data) and table pre-scaling.
#include <cuda.h>

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/gdrr.h"
#include "denoise_static.h"
#include "gdrr_internal.h"

using namespace gdrr;

struct gdrr_context {
    int device = 0;
    std::string err;
    unsigned long long launches = 0;
    // geometry
    bool has_geom = false;
    double du = 0, dv = 0, u_off = 0, v_off = 0, step = 0;
    int nu = 0, nv = 0, n_proj = 0;
    std::vector<double> poses;      // [n_proj][12] source S, detector origin P, u_hat, v_hat
    double* poses_dev = nullptr;
    // spectrum
    bool has_spec = false;
    int n_energy = 0, n_mat = 0;
    float4* mu_dev = nullptr;       // [n_energy] log2(e) mu_hat of the first (up to) four materials
    float* mu_all_dev = nullptr;    // [n_energy][n_mat] the same for all materials (more than four: energy_sum.cu)
    float2* src_dev = nullptr;
    float* bt_dev = nullptr;
    float* flu_dev = nullptr;
    float* gain_dev = nullptr;      // [n_energy][nv][nu] response gain (gdrr_set_response_gain) or nullptr
    float* li_scratch = nullptr;    // gdrr_project_host with more than four materials: line integrals of one batch
    size_t li_scratch_floats = 0;
    // misc
    // pinned, mapped: an ingest kernel sets its volume's slot through flag_dev if it meets a bad material; the slots
    // are handed out round-robin (a slot is reused after kFlagSlots later volumes)
    static constexpr int kFlagSlots = 64;
    int* flag_host = nullptr;
    int* flag_dev = nullptr;        //   (device address of flag_host)
    unsigned next_flag = 0;
    cudaStream_t copy_stream = nullptr;
    static constexpr int kIngestChunks = 8;             // gdrr_create_volume_host: z-slab chunks of the pipelined copy
    cudaEvent_t ev_chunk[kIngestChunks] = {};
    cudaEvent_t ev_stream = nullptr;
    cudaEvent_t ev_done[2] = {nullptr, nullptr};
    cudaEvent_t ev_free[2] = {nullptr, nullptr};
    int method = GDRR_METHOD_TRILINEAR;
    int sampler = GDRR_SAMPLER_AUTO;
    int last_sampler = 0;           // kernel the last tri-linear launch on a PACKED_QUAD volume used (gdrr_last_sampler)
    unsigned debug_skew = 0;        // gdrr_debug_set_skew
};

struct gdrr_volume {
    gdrr_context* ctx;
    void* vox;
    int nx, ny, nz, px, py, pz;
    double d[3], c[3];
    // A volume of more than four materials is a chain of device volumes, one per group of four materials, each complete
    // (its own layout, tensor map, compact copy); `groups` of the first one holds the others.  n_mat: the caller's
    // count (on every member); this member holds materials [mat_lo, mat_lo + n_group).
    int n_mat, n_group, mat_lo, vw, layout;
    std::vector<gdrr_volume*> groups;
    int sy, sz;                 // PACKED_QUAD: element strides
    void* compact = nullptr;    // PACKED_QUAD: one-word-per-voxel copy, rows in groups of four (Siddon walk)
    // ... made from the quads at the first Siddon use: `compact_mu` serialises the callers, `compact_done` orders every
    // later Siddon launch, on whatever stream, behind the copy kernel (ensure_compact)
    std::mutex compact_mu;
    bool compact_launched = false;
    cudaEvent_t compact_done = nullptr;
    std::atomic<bool> compact_ready{false};   // the copy is known to have finished (gdrr_volume_status): no wait needed
    bool has_tmap = false;      // PACKED_QUAD: tensor map for the staged sampler
    // the device-side material check is read when the ingest has finished, never waited for (volume_check)
    cudaEvent_t ingest_done = nullptr;
    volatile int* bad_flag = nullptr;    // this volume's slot of ctx->flag_host
    std::atomic<bool> checked{false}, bad{false};   // (two threads may both read the verdict: they write the same values)
    cudaArray_t tex_array = nullptr;     // optional texture variant (gdrr_volume_attach_texture)
    cudaTextureObject_t tex = 0;
    alignas(64) CUtensorMap tmap;
};

static thread_local std::string g_create_err;

namespace {

int fail(gdrr_context* ctx, int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (ctx) ctx->err = buf; else g_create_err = buf;
    return code;
}

int cuda_fail(gdrr_context* ctx, cudaError_t e, const char* what) {
    return fail(ctx, GDRR_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

// Makes ctx's device current for the scope of one ABI call.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    cudaError_t status = cudaSuccess;
    explicit DeviceGuard(int dev) {
        status = cudaGetDevice(&prev);
        if (status == cudaSuccess && prev != dev) {
            status = cudaSetDevice(dev);
            switched = (status == cudaSuccess);
        }
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

int vector_width(int n_mat) { return n_mat <= 1 ? 1 : (n_mat == 2 ? 2 : 4); }

// Stored dims of the device volume: voxels N + 2 rounded up to even (BRICK, LINEAR);
// quads (N + 1) x (N + 1) x (N + 2 slabs) for PACKED_QUAD.
void stored_dims(int nx, int ny, int nz, int layout, int& px, int& py, int& pz) {
    if (layout == GDRR_LAYOUT_PACKED_QUAD) {
        px = nx + 1;
        py = ny + 1;
        pz = nz + 2;
    } else {
        px = (nx + 3) & ~1;
        py = (ny + 3) & ~1;
        pz = (nz + 3) & ~1;
    }
}

// PACKED_QUAD element strides: linear, with the row stride = 3 and the slab stride = 4 (mod 8),
// so that neighbouring elements fall in different 16-byte bank groups of the L1 data RAM in
// every direction (project_packed.cu).
void packed_strides(int px, int py, int& sy, int& sz) {
    sy = px + ((3 - px % 8) + 8) % 8;
    const long long s0 = (long long)sy * py;
    sz = (int)(s0 + ((4 - s0 % 8) + 8) % 8);
}

size_t packed_elements(int nx, int ny, int nz) {
    int px, py, pz, sy, sz;
    stored_dims(nx, ny, nz, GDRR_LAYOUT_PACKED_QUAD, px, py, pz);
    packed_strides(px, py, sy, sz);
    return (size_t)sz * pz;
}

// bytes of the 4 x 4 x 2-bricked one-word-per-voxel copy kept behind the quads (Siddon walk)
size_t compact_bytes(int nx, int ny, int nz) {        // rows in groups of four, 4 B per voxel
    return (size_t)nx * (size_t)(4 * ((ny + 3) / 4)) * (size_t)nz * 4;
}

size_t element_bytes(int n_mat, int layout) {
    return layout == GDRR_LAYOUT_PACKED_QUAD ? 16 : vector_width(n_mat) * sizeof(float);
}

bool all_finite(const double* a, size_t n) {
    for (size_t k = 0; k < n; ++k) if (!std::isfinite(a[k])) return false;
    return true;
}

template <class T> void free_dev(T*& p) { if (p) { cudaFree(p); p = nullptr; } }

int check_dims(gdrr_context* ctx, int nx, int ny, int nz, int n_materials, int layout) {
    if (nx <= 0 || ny <= 0 || nz <= 0)
        return fail(ctx, GDRR_ERR_INVALID_ARG, "volume dims must be positive (got %d %d %d)", nx, ny, nz);
    if (n_materials <= 0)
        return fail(ctx, GDRR_ERR_INVALID_ARG, "n_materials must be >= 1 (got %d)", n_materials);
    if (n_materials > GDRR_MAX_MATERIALS)
        return fail(ctx, GDRR_ERR_UNSUPPORTED, "n_materials %d > GDRR_MAX_MATERIALS %d", n_materials,
                    GDRR_MAX_MATERIALS);
    if (layout != GDRR_LAYOUT_BRICK && layout != GDRR_LAYOUT_LINEAR && layout != GDRR_LAYOUT_PACKED_QUAD)
        return fail(ctx, GDRR_ERR_INVALID_ARG, "unknown layout %d", layout);
    int px, py, pz;
    stored_dims(nx, ny, nz, layout, px, py, pz);
    double total = (double)px * py * pz;
    if (layout == GDRR_LAYOUT_PACKED_QUAD)
        total = (double)packed_elements(nx, ny, nz) + px * (double)py;
    if (total >= 2147483648.0)
        return fail(ctx, GDRR_ERR_UNSUPPORTED, "padded volume has %.0f voxels; the sampler indexes with int32", total);
    return GDRR_OK;
}

// The ingest kernels check material < n_materials on the device and raise the volume's flag (pinned host memory).
// gdrr_create_volume does not wait for that: the flag is read here, by every later call that takes the volume, once the
// ingest is known to have finished (cudaEventQuery; `wait`: cudaEventSynchronize, gdrr_volume_status).  A bad volume is
// refused from then on.  (Its ingest wrote tags "material & 3", so nothing it did was out of bounds.)
int volume_check(gdrr_context* ctx, const gdrr_volume* cvol, bool wait) {
    gdrr_volume* vol = const_cast<gdrr_volume*>(cvol);
    if (!vol->checked && vol->ingest_done) {
        DeviceGuard guard(ctx->device);
        cudaError_t e = wait ? cudaEventSynchronize(vol->ingest_done) : cudaEventQuery(vol->ingest_done);
        if (e == cudaSuccess) {
            vol->bad.store(*vol->bad_flag != 0);
            vol->checked.store(true);
        } else if (e != cudaErrorNotReady) {
            return cuda_fail(ctx, e, "waiting for the volume ingest");
        } else {
            cudaGetLastError();
        }
    }
    if (vol->bad)
        return fail(ctx, GDRR_ERR_INVALID_ARG, "a material index of this volume is >= n_materials (%d)", vol->n_mat);
    for (gdrr_volume* g : vol->groups)
        if (int rc = volume_check(ctx, g, wait)) return rc;
    return GDRR_OK;
}

// Fills the fp64 ray-setup parameters for (ctx geometry, volume).  Box bounds
// are formed exactly as DESIGN.md a1 writes them: half = 0.5 * (N * d).
int fill_geom(gdrr_context* ctx, const gdrr_volume* vol, int proj_begin, int proj_count,
              GeomParams& g) {
    if (!ctx->has_geom) return fail(ctx, GDRR_ERR_NOT_READY, "gdrr_set_geometry has not been called");
    if (!vol || vol->ctx != ctx) return fail(ctx, GDRR_ERR_INVALID_ARG, "volume is NULL or belongs to another context");
    if (int rc = volume_check(ctx, vol, false)) return rc;
    if (proj_begin < 0 || proj_count <= 0 || proj_begin > ctx->n_proj - proj_count)
        return fail(ctx, GDRR_ERR_INVALID_ARG, "projection range [%d, %d+%d) outside [0, %d)", proj_begin,
                    proj_begin, proj_count, ctx->n_proj);
    if (proj_count > 65535)
        return fail(ctx, GDRR_ERR_UNSUPPORTED, "at most 65535 projections per call (got %d)", proj_count);
    g.half_nu = 0.5 * (double)(ctx->nu - 1);
    g.half_nv = 0.5 * (double)(ctx->nv - 1);
    g.du = ctx->du; g.dv = ctx->dv; g.u_off = ctx->u_off; g.v_off = ctx->v_off;
    const int n[3] = {vol->nx, vol->ny, vol->nz};
    double dmin = vol->d[0];
    for (int a = 0; a < 3; ++a) {
        const double half = 0.5 * ((double)n[a] * vol->d[a]);
        g.lo[a] = vol->c[a] - half;
        g.hi[a] = vol->c[a] + half;
        g.c[a] = vol->c[a];
        g.d[a] = vol->d[a];
        g.inv_d[a] = 1.0 / vol->d[a];
        g.ofs[a] = 0.5 * (double)(n[a] - 1) + 1.0;
        if (vol->d[a] < dmin) dmin = vol->d[a];
    }
    g.step = ctx->step > 0.0 ? ctx->step : 0.5 * dmin;       // PAPER.md:155, reading Q8
    g.poses = ctx->poses_dev;
    g.nu = ctx->nu; g.nv = ctx->nv;
    g.proj_begin = proj_begin; g.proj_count = proj_count;
    // the source must be outside the volume box for every requested angle
    for (int p = proj_begin; p < proj_begin + proj_count; ++p) {
        const double* S = &ctx->poses[12 * (size_t)p];
        bool inside = true;
        for (int a = 0; a < 3; ++a) inside = inside && S[a] >= g.lo[a] && S[a] <= g.hi[a];
        if (inside)
            return fail(ctx, GDRR_ERR_INVALID_ARG, "source lies inside the volume box at projection %d", p);
    }
    return GDRR_OK;
}

// The device-volume part of the kernel parameters (one member of a chain of material groups).
void fill_volume(const gdrr_volume* vol, ProjectParams& P) {
    P.v.vox = vol->vox;
    P.v.nvox[0] = vol->nx; P.v.nvox[1] = vol->ny; P.v.nvox[2] = vol->nz;
    P.v.compact = vol->compact;
    P.v.cstride_y = 4 * vol->nx;
    P.v.cstride_z = 4 * vol->nx * ((vol->ny + 3) / 4);
    if (vol->layout == GDRR_LAYOUT_BRICK) {
        P.v.stride_y = 8 * (vol->px / 2);
        P.v.stride_z = 8 * (vol->px / 2) * (vol->py / 2);
    } else if (vol->layout == GDRR_LAYOUT_PACKED_QUAD) {
        P.v.stride_y = vol->sy;
        P.v.stride_z = vol->sz;
    } else {
        P.v.stride_y = vol->px;
        P.v.stride_z = vol->px * vol->py;
    }
    P.v.vox1 = (const char*)vol->vox + 16 * (size_t)vol->sz;
    P.n_mat = vol->n_group;
    P.li_mat0 = vol->mat_lo;
}

int fill_project(gdrr_context* ctx, const gdrr_volume* vol, int proj_begin, int proj_count,
                 ProjectParams& P) {
    int rc = fill_geom(ctx, vol, proj_begin, proj_count, P.g);
    if (rc) return rc;
    if (!ctx->has_spec) return fail(ctx, GDRR_ERR_NOT_READY, "gdrr_set_spectrum has not been called");
    if (ctx->n_mat != vol->n_mat)
        return fail(ctx, GDRR_ERR_NOT_READY, "spectrum has %d materials, volume has %d", ctx->n_mat, vol->n_mat);
    if (ctx->method == GDRR_METHOD_TEXTURE && !vol->groups.empty())
        return fail(ctx, GDRR_ERR_UNSUPPORTED, "GDRR_METHOD_TEXTURE holds at most four materials (four texture channels)");
    if (ctx->method == GDRR_METHOD_TEXTURE && !vol->tex)
        return fail(ctx, GDRR_ERR_NOT_READY, "GDRR_METHOD_TEXTURE needs gdrr_volume_attach_texture on this volume");
    fill_volume(vol, P);
    P.seg_table = nullptr;
    P.mu_tab = ctx->mu_dev;
    P.src_tab = ctx->src_dev;
    P.bt_thick = ctx->bt_dev;
    P.fluence = ctx->flu_dev;
    P.gain = ctx->gain_dev;
    P.n_energy = ctx->n_energy;
    P.li_only = 0; P.li_mat_total = vol->n_mat;
    P.mu_all = ctx->mu_all_dev;
    // in-chunk positions are 9.23 fixed point: keep |advance| per chunk below 128 voxels
    double dgmax = 0.0;
    for (int a = 0; a < 3; ++a) dgmax = std::fmax(dgmax, P.g.step / vol->d[a]);
    int chunk = kMaxChunk;
    if (dgmax * chunk > 120.0) chunk = (int)(120.0 / dgmax);
    if (chunk < 1)
        return fail(ctx, GDRR_ERR_UNSUPPORTED, "step %.6g mm is more than 120 voxels long", P.g.step);
    P.chunk = chunk;
    P.frac_mask = 0x007FFFFFu;
    P.one_bits = 0x3F800000u;
    P.debug_skew = ctx->debug_skew;
    for (int a = 0; a < 3; ++a) P.hull_margin[a] = 0.0;
    return GDRR_OK;
}

// Tensor map of the packed-quad volume for project_staged.cu: a 3-D tensor of 32-bit words
// (4 px words along x, py rows of pitch 16 sy bytes, pz slabs of pitch 16 sz bytes), box
// 56 words x 14 rows x 11 slabs.  The driver entry point is looked up at run time, so the
// library still links cudart only.  Returns false if the driver cannot make it.
bool make_tensor_map(gdrr_volume* v) {
    typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
        qres != cudaDriverEntryPointSuccess) {
        cudaGetLastError();
        return false;
    }
    const cuuint64_t dims[3] = {4ull * (cuuint64_t)v->px, (cuuint64_t)v->py, (cuuint64_t)v->pz};
    const cuuint64_t strides[2] = {16ull * (cuuint64_t)v->sy, 16ull * (cuuint64_t)v->sz};      // bytes, dims 1 and 2
    const cuuint32_t box[3] = {4u * kBX, (cuuint32_t)kBY, (cuuint32_t)kBZ};
    const cuuint32_t estr[3] = {1u, 1u, 1u};
    CUresult r = ((encode_fn)fn)(&v->tmap, CU_TENSOR_MAP_DATA_TYPE_UINT32, 3, v->vox, dims, strides, box, estr,
                                 CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                 CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

// Siddon on a packed volume walks the compact copy.  The first caller makes it from the quads on its own stream and
// records `compact_done` behind the copy kernel; every caller (this one included) then makes its stream wait for that
// event, so a Siddon launch on another stream, or from another thread, can never read the copy before it is filled.
cudaError_t ensure_compact(const gdrr_volume* cvol, cudaStream_t s) {
    if (cvol->layout != GDRR_LAYOUT_PACKED_QUAD) return cudaSuccess;
    gdrr_volume* vol = const_cast<gdrr_volume*>(cvol);       // the copy is a cache behind the handle, guarded by its mutex
    if (vol->compact_ready) return cudaSuccess;              // (no stream call at all: the launch can be captured)
    std::lock_guard<std::mutex> lock(vol->compact_mu);
    cudaError_t e = cudaSuccess;
    if (!vol->compact_launched) {
        if (!vol->compact_done) e = cudaEventCreateWithFlags(&vol->compact_done, cudaEventDisableTiming);
        if (e != cudaSuccess) return e;
        IngestParams ip = {};
        ip.vox = vol->vox; ip.compact = vol->compact;
        ip.nx = vol->nx; ip.ny = vol->ny; ip.nz = vol->nz;
        ip.sy = vol->sy; ip.sz = vol->sz; ip.n_mat = vol->n_mat; ip.tagged = vol->n_group > 1;
        ip.cbx = (vol->nx + 3) / 4; ip.cby = (vol->ny + 3) / 4;
        e = launch_compact_copy(ip, s);
        if (e == cudaSuccess) e = cudaEventRecord(vol->compact_done, s);
        if (e != cudaSuccess) return e;
        vol->compact_launched = true;
        vol->ctx->launches += 1;
    }
    return cudaStreamWaitEvent(s, vol->compact_done, 0);
}

// Does staging pay?  Extent, in voxels per axis, of the beam of a 16 x 16-pixel CTA over 16 steps at the
// depth of the box centre, averaged over the requested projections, against the 14 x 14 x 11-quad box (a chunk
// whose beam does not fit is gathered anyway, after its box has been refused).  Thresholds measured on C3 with the
// round-2 kernels (staged against gather, samples/s): circle and helix (mean extents 10.5, 10.5, 6.6) 7.39e11 against
// 5.03e11; orbit tilted 10 degrees (10.5, 11.8, 8.0) 6.75e11 against 4.95e11; tilted 20 degrees (10.5, 12.7, 9.0)
// 5.58e11 against 4.91e11; tilted 35 degrees (10.5, 13.4, 10.1) 4.50e11 against 4.90e11: the line is drawn halfway
// between the last two.  tests/test_gpu_sampler_choice.py pins what AUTO picks on each of these.
bool beam_fits(const gdrr_context* c, const gdrr_volume* vol, const GeomParams& g) {
    double ext[3] = {0.0, 0.0, 0.0};
    for (int p = g.proj_begin; p < g.proj_begin + g.proj_count; ++p) {
        const double* q = &c->poses[12 * (size_t)p];
        const double *S = q, *P = q + 3, *uh = q + 6, *vh = q + 9;
        const double nrm[3] = {uh[1] * vh[2] - uh[2] * vh[1], uh[2] * vh[0] - uh[0] * vh[2], uh[0] * vh[1] - uh[1] * vh[0]};
        double sp = 0.0, sc = 0.0, sdd = 0.0, nn = 0.0;
        for (int a = 0; a < 3; ++a) {
            sp += (P[a] - S[a]) * (P[a] - S[a]);
            sc += (vol->c[a] - S[a]) * (vol->c[a] - S[a]);
            sdd += (P[a] - S[a]) * nrm[a];
            nn += nrm[a] * nrm[a];
        }
        sdd = std::fabs(sdd) / std::sqrt(nn);
        const double mag = std::sqrt(sc) / sdd;
        for (int a = 0; a < 3; ++a)
            ext[a] += (16.0 * mag * (g.du * std::fabs(uh[a]) + g.dv * std::fabs(vh[a])) +
                       16.0 * g.step * std::fabs(P[a] - S[a]) / std::sqrt(sp)) / vol->d[a];
    }
    for (int a = 0; a < 3; ++a) ext[a] /= (double)g.proj_count;
    return ext[0] <= 13.05 && ext[1] <= 13.05 && ext[2] <= 9.55;
}

// The staged sampler bounds a chunk of a CTA's beam by its four CORNER rays (project_staged.cu).  How far can a ray of
// the tile lie outside their hull at equal interval index?  Sample k of the ray through detector point (u, v) is
// x = S + t_k n / |n|, n = D(u, v) - S, D affine in (u, v) with unit steps u_hat, v_hat.  For f = n_a / |n|:
// f_uu = -2 u_hat_a s / L^2 - n_a / L^3 + 3 n_a s^2 / L^3 with L = |n|, s = (n . u_hat) / L, so
// |f_uu| <= (2 s_u + 1 + 3 s_u^2) / L_min^2 =: c_u / L_min^2, where s_u bounds |s| over the detector: n . u_hat is affine in
// (u, v), so its largest magnitude is at a detector corner, and L >= L_min.  The same for v.  Bilinear interpolation
// between the corners of a tile with edges hu, hv is therefore off by at most (c_u hu^2 + c_v hv^2) / (8 L_min^2), a
// bilinear function takes its extremes at the corners, and t_k <= L_max.  In voxels of axis a:
//   margin_a = (c_u hu^2 + c_v hv^2) L_max / (8 L_min^2 d_a) + 2^-10,
// the last term for the samplers' fixed-point positions (<= 2^-19) and the fp64 rounding of the producer's own.
// L_min = distance of the source from the detector plane, L_max = its distance from the farthest detector corner,
// all over the requested projections.  (C3: 0.037 voxel, C4: 0.019, C1: 0.07.)
// Returns false if a margin exceeds 0.45 voxel (tiles too wide for the source distance): the caller then gathers.
bool hull_margins(const gdrr_context* c, const gdrr_volume* vol, const GeomParams& g, double (&margin)[3]) {
    double lmin = 1e300, lmax = 0.0, bound = 0.0;       // bound: largest (c_u hu^2 + c_v hv^2) / L_min^2 of a projection
    const double ue[2] = {(0.0 - g.half_nu) * g.du + g.u_off, ((double)(g.nu - 1) - g.half_nu) * g.du + g.u_off};
    const double ve[2] = {(0.0 - g.half_nv) * g.dv + g.v_off, ((double)(g.nv - 1) - g.half_nv) * g.dv + g.v_off};
    for (int p = g.proj_begin; p < g.proj_begin + g.proj_count; ++p) {
        const double* q = &c->poses[12 * (size_t)p];
        const double *S = q, *P = q + 3, *uh = q + 6, *vh = q + 9;
        const double nrm[3] = {uh[1] * vh[2] - uh[2] * vh[1], uh[2] * vh[0] - uh[0] * vh[2], uh[0] * vh[1] - uh[1] * vh[0]};
        double dist = 0.0, nn = 0.0, uu = 0.0, vv = 0.0;
        for (int a = 0; a < 3; ++a) {
            dist += (P[a] - S[a]) * nrm[a];
            nn += nrm[a] * nrm[a];
            uu += uh[a] * uh[a];
            vv += vh[a] * vh[a];
        }
        const double lp = std::fabs(dist) / std::sqrt(nn);           // this projection's L_min
        if (!(lp > 0.0)) return false;
        lmin = std::fmin(lmin, lp);
        double nu_max = 0.0, nv_max = 0.0;                           // largest |n . u_hat|, |n . v_hat| (unit vectors)
        for (int cu = 0; cu < 2; ++cu)
            for (int cv = 0; cv < 2; ++cv) {
                double l2 = 0.0, du_ = 0.0, dv_ = 0.0;
                for (int a = 0; a < 3; ++a) {
                    const double n = P[a] + ue[cu] * uh[a] + ve[cv] * vh[a] - S[a];
                    l2 += n * n;
                    du_ += n * uh[a];
                    dv_ += n * vh[a];
                }
                lmax = std::fmax(lmax, std::sqrt(l2));
                nu_max = std::fmax(nu_max, std::fabs(du_) / std::sqrt(uu));
                nv_max = std::fmax(nv_max, std::fabs(dv_) / std::sqrt(vv));
            }
        const double su = std::fmin(1.0, nu_max / lp), sv = std::fmin(1.0, nv_max / lp);
        const double hu = (kTileU - 1) * g.du * std::sqrt(uu), hv = (kStageTileV - 1) * g.dv * std::sqrt(vv);
        bound = std::fmax(bound, ((2.0 * su + 1.0 + 3.0 * su * su) * hu * hu + (2.0 * sv + 1.0 + 3.0 * sv * sv) * hv * hv) / (lp * lp));
    }
    bool ok = true;
    for (int a = 0; a < 3; ++a) {
        margin[a] = bound * lmax / (8.0 * vol->d[a]) + 1.0 / 1024.0;
        ok = ok && margin[a] <= 0.45;
    }
    return ok;
}

// A kernel that reads the volume on stream s must run behind its ingest, whichever stream that was queued on
// (gdrr_create_volume no longer waits for it).  Nothing to do once the ingest is known to have finished.
cudaError_t order_after_ingest(const gdrr_volume* vol, cudaStream_t s) {
    if (vol->checked || !vol->ingest_done) return cudaSuccess;
    return cudaStreamWaitEvent(s, vol->ingest_done, 0);
}

cudaError_t launch_one(const ProjectParams& P, const gdrr_volume* vol, cudaStream_t s);

// One launch for up to four materials.  More: one LI-only launch per group of four (each on its own device volume, the
// ray table written once), then the energy sum over all line integrals (energy_sum.cu); P.li is required then.
cudaError_t launch_project(const ProjectParams& P, const gdrr_volume* vol, cudaStream_t s) {
    if (vol->groups.empty()) return launch_one(P, vol, s);
    ProjectParams Pg = P;
    Pg.li_only = 1;
    for (size_t g = 0; g <= vol->groups.size(); ++g) {
        const gdrr_volume* member = g == 0 ? vol : vol->groups[g - 1];
        fill_volume(member, Pg);
        if (g > 0) Pg.ray_table = nullptr;
        if (cudaError_t e = launch_one(Pg, member, s)) return e;
        vol->ctx->launches += 1;
    }
    return launch_energy_sum(P, s);          // (the caller counts this last launch)
}

cudaError_t launch_one(const ProjectParams& P, const gdrr_volume* vol, cudaStream_t s) {
    gdrr_context* c = vol->ctx;
    if (cudaError_t e = order_after_ingest(vol, s)) return e;
    if (c->method == GDRR_METHOD_SIDDON) {
        cudaError_t e = ensure_compact(vol, s);
        if (e != cudaSuccess) return e;
        return launch_project_siddon(P, vol->vw, vol->layout, s);
    }
    if (c->method == GDRR_METHOD_TEXTURE) return launch_project_texture(P, vol->vw, (unsigned long long)vol->tex, s);
    if (vol->layout == GDRR_LAYOUT_PACKED_QUAD && vol->has_tmap && c->sampler != GDRR_SAMPLER_GATHER) {
        // AUTO: staging pays when the beam of a 16 x 16-pixel CTA over 16 steps fits the 14 x 14 x 11-quad box
        // (a chunk that does not fit is gathered anyway, after its box has been refused)
        const bool fits = beam_fits(c, vol, P.g);
        // (the staged kernel keeps a chunk's base in 5.27 fixed point: 16 steps must advance less than 16 voxels)
        const double adv16 = 16.0 * P.g.step / std::fmin(vol->d[0], std::fmin(vol->d[1], vol->d[2]));
        ProjectParams Ps = P;
        if (adv16 <= 15.0 && (fits || c->sampler == GDRR_SAMPLER_STAGED) && hull_margins(c, vol, P.g, Ps.hull_margin)) {
            c->last_sampler = GDRR_SAMPLER_STAGED;
            return launch_project_staged(Ps, vol->vw, &vol->tmap, s);
        }
    }
    if (vol->layout == GDRR_LAYOUT_PACKED_QUAD) {
        c->last_sampler = GDRR_SAMPLER_GATHER;
        return launch_project_packed(P, vol->vw, s);
    }
    c->last_sampler = 0;
    return launch_project_exact(P, vol->vw, vol->layout, s);
}

}  // namespace

extern "C" {

const char* gdrr_version(void) { return "0.1"; }

int gdrr_create_context(int cuda_device, gdrr_context** out) {
    if (!out) return fail(nullptr, GDRR_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    int count = 0;
    cudaError_t e = cudaGetDeviceCount(&count);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetDeviceCount");
    if (cuda_device < 0 || cuda_device >= count)
        return fail(nullptr, GDRR_ERR_INVALID_ARG, "cuda_device %d outside [0, %d)", cuda_device, count);
    gdrr_context* ctx = new (std::nothrow) gdrr_context;
    if (!ctx) return fail(nullptr, GDRR_ERR_INVALID_ARG, "out of host memory");
    ctx->device = cuda_device;
    DeviceGuard guard(cuda_device);
    if (guard.status != cudaSuccess) { delete ctx; return cuda_fail(nullptr, guard.status, "cudaSetDevice"); }
    e = cudaHostAlloc(&ctx->flag_host, sizeof(int) * gdrr_context::kFlagSlots, cudaHostAllocMapped);
    if (e == cudaSuccess) e = cudaHostGetDevicePointer(&ctx->flag_dev, ctx->flag_host, 0);
    if (e != cudaSuccess) {
        if (ctx->flag_host) cudaFreeHost(ctx->flag_host);
        delete ctx;
        return cuda_fail(nullptr, e, "cudaHostAlloc(flag)");
    }
    *out = ctx;
    return GDRR_OK;
}

int gdrr_destroy_context(gdrr_context* ctx) {
    if (!ctx) return GDRR_OK;
    DeviceGuard guard(ctx->device);
    free_dev(ctx->poses_dev); free_dev(ctx->mu_dev); free_dev(ctx->src_dev);
    free_dev(ctx->bt_dev); free_dev(ctx->flu_dev); free_dev(ctx->gain_dev); free_dev(ctx->mu_all_dev);
    free_dev(ctx->li_scratch);
    if (ctx->flag_host) { cudaFreeHost(ctx->flag_host); ctx->flag_host = nullptr; ctx->flag_dev = nullptr; }
    for (int k = 0; k < 2; ++k) {
        if (ctx->ev_done[k]) cudaEventDestroy(ctx->ev_done[k]);
        if (ctx->ev_free[k]) cudaEventDestroy(ctx->ev_free[k]);
    }
    for (int k = 0; k < gdrr_context::kIngestChunks; ++k)
        if (ctx->ev_chunk[k]) cudaEventDestroy(ctx->ev_chunk[k]);
    if (ctx->ev_stream) cudaEventDestroy(ctx->ev_stream);
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    delete ctx;
    return GDRR_OK;
}

const char* gdrr_last_error(const gdrr_context* ctx) {
    return ctx ? ctx->err.c_str() : g_create_err.c_str();
}

unsigned long long gdrr_kernel_launches(const gdrr_context* ctx) { return ctx ? ctx->launches : 0ull; }

// Workspace of ONE device volume holding n_group (<= 4) materials, rounded up to 256 bytes.
static size_t group_workspace_bytes(int nx, int ny, int nz, int n_group, int layout) {
    int px, py, pz;
    stored_dims(nx, ny, nz, layout, px, py, pz);
    size_t bytes = (size_t)px * py * pz * element_bytes(n_group, layout);
    if (layout == GDRR_LAYOUT_PACKED_QUAD)
        bytes = ((16 * packed_elements(nx, ny, nz) + 255) & ~(size_t)255) + compact_bytes(nx, ny, nz);
    return (bytes + 255) & ~(size_t)255;
}

int gdrr_volume_workspace_bytes(int nx, int ny, int nz, int n_materials, int layout, size_t* bytes) {
    if (!bytes) return fail(nullptr, GDRR_ERR_INVALID_ARG, "bytes is NULL");
    int rc = check_dims(nullptr, nx, ny, nz, n_materials, layout);
    if (rc) return rc;
    *bytes = 0;
    for (int lo = 0; lo < n_materials; lo += 4)          // one device volume per group of four materials
        *bytes += group_workspace_bytes(nx, ny, nz, std::min(4, n_materials - lo), layout);
    return GDRR_OK;
}

// gdrr_create_volume and gdrr_create_volume_host.  rho_host / mat_host != NULL: the inputs are first copied into
// rho_dev / mat_dev (the caller's staging buffers) in z-slab chunks on the context's copy stream, and the slabs of the
// device layout that a chunk completes are written while the next chunk is still on the bus.
static int create_group(gdrr_context* ctx, const float* rho_host, const uint8_t* mat_host,
                        float* rho_dev, uint8_t* mat_dev, int nx, int ny, int nz,
                        double dx_mm, double dy_mm, double dz_mm, const double centre_mm[3], int n_materials,
                        int mat_lo, int n_group, int layout, void* workspace_dev, void* cuda_stream, gdrr_volume** out);

// All groups of four materials, chained behind the first (the only one that copies from the host).
static int create_volume_impl(gdrr_context* ctx, const float* rho_host, const uint8_t* mat_host,
                              float* rho_dev, uint8_t* mat_dev, int nx, int ny, int nz,
                              double dx_mm, double dy_mm, double dz_mm, const double centre_mm[3], int n_materials,
                              int layout, void* workspace_dev, size_t workspace_bytes, void* cuda_stream,
                              gdrr_volume** out) {
    if (!(dx_mm > 0) || !(dy_mm > 0) || !(dz_mm > 0) || !std::isfinite(dx_mm) || !std::isfinite(dy_mm) ||
        !std::isfinite(dz_mm))
        return fail(ctx, GDRR_ERR_INVALID_ARG, "voxel sizes must be positive and finite");
    if (centre_mm && !all_finite(centre_mm, 3)) return fail(ctx, GDRR_ERR_INVALID_ARG, "centre_mm is not finite");
    size_t need = 0;
    gdrr_volume_workspace_bytes(nx, ny, nz, n_materials, layout, &need);
    if (!workspace_dev || workspace_bytes < need)
        return fail(ctx, GDRR_ERR_WORKSPACE, "workspace of %zu bytes given, %zu needed", workspace_bytes, need);
    if ((uintptr_t)workspace_dev % 256)
        return fail(ctx, GDRR_ERR_WORKSPACE, "workspace must be 256-byte aligned");
    gdrr_volume* first = nullptr;
    char* ws = (char*)workspace_dev;
    for (int lo = 0; lo < n_materials; lo += 4) {
        const int n_group = std::min(4, n_materials - lo);
        gdrr_volume* v = nullptr;
        int rc = create_group(ctx, lo == 0 ? rho_host : nullptr, lo == 0 ? mat_host : nullptr, rho_dev, mat_dev, nx, ny, nz,
                              dx_mm, dy_mm, dz_mm, centre_mm, n_materials, lo, n_group, layout, ws, cuda_stream, &v);
        if (rc) {
            if (first) gdrr_destroy_volume(first);
            return rc;
        }
        if (first) first->groups.push_back(v); else first = v;
        ws += group_workspace_bytes(nx, ny, nz, n_group, layout);
    }
    *out = first;
    return GDRR_OK;
}

static int create_group(gdrr_context* ctx, const float* rho_host, const uint8_t* mat_host,
                        float* rho_dev, uint8_t* mat_dev, int nx, int ny, int nz,
                        double dx_mm, double dy_mm, double dz_mm, const double centre_mm[3], int n_materials,
                        int mat_lo, int n_group, int layout, void* workspace_dev, void* cuda_stream, gdrr_volume** out) {
    DeviceGuard guard(ctx->device);
    if (guard.status != cudaSuccess) return cuda_fail(ctx, guard.status, "cudaSetDevice");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    gdrr_volume* v = new (std::nothrow) gdrr_volume;
    if (!v) return fail(ctx, GDRR_ERR_INVALID_ARG, "out of host memory");
    cudaError_t e = cudaEventCreateWithFlags(&v->ingest_done, cudaEventDisableTiming);
    if (e != cudaSuccess) { delete v; return cuda_fail(ctx, e, "cudaEventCreate"); }
    const unsigned slot = ctx->next_flag++ % gdrr_context::kFlagSlots;
    ctx->flag_host[slot] = 0;
    v->bad_flag = ctx->flag_host + slot;

    IngestParams ip;
    ip.rho = rho_dev; ip.mat = mat_dev; ip.vox = workspace_dev;
    ip.nx = nx; ip.ny = ny; ip.nz = nz;
    stored_dims(nx, ny, nz, layout, ip.px, ip.py, ip.pz);
    ip.n_mat = n_materials; ip.bad_flag = ctx->flag_dev + slot;
    ip.mat_lo = mat_lo; ip.n_group = n_group; ip.tagged = n_group > 1;
    ip.sy = ip.sz = 0;
    ip.compact = nullptr; ip.cbx = (nx + 3) / 4; ip.cby = (ny + 3) / 4;
    if (layout == GDRR_LAYOUT_PACKED_QUAD) {
        packed_strides(ip.px, ip.py, ip.sy, ip.sz);
        ip.compact = (char*)workspace_dev + ((16 * (size_t)ip.sz * ip.pz + 255) & ~(size_t)255);
    }
    const int vw = vector_width(n_group);
    const size_t slab = (size_t)nx * ny;
    // chunks of whole z slabs, at least ~8 MB of rho each (a chunk costs four API calls: below that the host's
    // time per chunk shows); BRICK stores 2 x 2 x 2 bricks: one chunk
    int chunks = 1;
    if (rho_host && layout != GDRR_LAYOUT_BRICK)
        chunks = (int)std::max<size_t>(1, std::min<size_t>({(size_t)gdrr_context::kIngestChunks, (size_t)nz,
                                                             slab * nz * sizeof(float) / (8u << 20)}));
    if (rho_host) {
        if (!ctx->copy_stream) e = cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking);
        for (int k = 0; k < gdrr_context::kIngestChunks && e == cudaSuccess; ++k)
            if (!ctx->ev_chunk[k]) e = cudaEventCreateWithFlags(&ctx->ev_chunk[k], cudaEventDisableTiming);
        if (e == cudaSuccess && !ctx->ev_stream) e = cudaEventCreateWithFlags(&ctx->ev_stream, cudaEventDisableTiming);
        // the staging buffers may still be read by work queued on the caller's stream: the copies start behind it
        if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_stream, s);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_stream, 0);
    }
    int stored_done = 0;                                   // stored slabs [0, stored_done) are written
    for (int c = 0; c < chunks && e == cudaSuccess; ++c) {
        const int z0 = (int)((long long)nz * c / chunks), z1 = (int)((long long)nz * (c + 1) / chunks);
        if (rho_host) {
            e = cudaMemcpyAsync(rho_dev + slab * z0, rho_host + slab * z0, slab * (z1 - z0) * sizeof(float),
                                cudaMemcpyHostToDevice, ctx->copy_stream);
            if (e == cudaSuccess)
                e = cudaMemcpyAsync(mat_dev + slab * z0, mat_host + slab * z0, slab * (z1 - z0),
                                    cudaMemcpyHostToDevice, ctx->copy_stream);
            if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_chunk[c], ctx->copy_stream);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(s, ctx->ev_chunk[c], 0);
        }
        // stored slab k reads voxel slabs clamp(k - 1) (and clamp(k) for a quad's purity tags): with voxel slabs
        // [0, z1) on the device, stored slabs up to z1 - 1 (quads), z1 (LINEAR) can be written; the last chunk the rest
        int stored_end = c + 1 == chunks ? ip.pz : (layout == GDRR_LAYOUT_PACKED_QUAD ? z1 : z1 + 1);
        if (stored_end > ip.pz) stored_end = ip.pz;
        if (e == cudaSuccess && stored_end > stored_done) {
            ip.ez0 = stored_done; ip.ezn = stored_end - stored_done;
            e = launch_ingest(ip, vw, layout, s);
            ctx->launches += 1;
            stored_done = stored_end;
        }
    }
    if (e == cudaSuccess) e = cudaEventRecord(v->ingest_done, s);
    if (e != cudaSuccess) {
        cudaEventDestroy(v->ingest_done);
        delete v;
        return cuda_fail(ctx, e, "volume ingest");
    }
    v->ctx = ctx; v->vox = workspace_dev;
    v->nx = nx; v->ny = ny; v->nz = nz; v->px = ip.px; v->py = ip.py; v->pz = ip.pz;
    v->d[0] = dx_mm; v->d[1] = dy_mm; v->d[2] = dz_mm;
    for (int a = 0; a < 3; ++a) v->c[a] = centre_mm ? centre_mm[a] : 0.0;
    v->n_mat = n_materials; v->n_group = n_group; v->mat_lo = mat_lo; v->vw = vw; v->layout = layout;
    v->sy = ip.sy; v->sz = ip.sz; v->compact = ip.compact;
    v->has_tmap = layout == GDRR_LAYOUT_PACKED_QUAD && make_tensor_map(v);
    *out = v;
    return GDRR_OK;
}

int gdrr_create_volume(gdrr_context* ctx, const float* rho_dev, const uint8_t* material_dev,
                       int nx, int ny, int nz, double dx_mm, double dy_mm, double dz_mm,
                       const double centre_mm[3], int n_materials, int layout,
                       void* workspace_dev, size_t workspace_bytes, void* cuda_stream,
                       gdrr_volume** out) {
    if (!ctx) return fail(nullptr, GDRR_ERR_INVALID_ARG, "ctx is NULL");
    if (!out) return fail(ctx, GDRR_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    int rc = check_dims(ctx, nx, ny, nz, n_materials, layout);
    if (rc) return rc;
    if (!rho_dev || !material_dev) return fail(ctx, GDRR_ERR_INVALID_ARG, "rho_dev / material_dev is NULL");
    return create_volume_impl(ctx, nullptr, nullptr, const_cast<float*>(rho_dev), const_cast<uint8_t*>(material_dev),
                              nx, ny, nz, dx_mm, dy_mm, dz_mm, centre_mm, n_materials, layout, workspace_dev,
                              workspace_bytes, cuda_stream, out);
}

int gdrr_create_volume_host(gdrr_context* ctx, const float* rho_host, const uint8_t* material_host,
                            int nx, int ny, int nz, double dx_mm, double dy_mm, double dz_mm,
                            const double centre_mm[3], int n_materials, int layout,
                            float* rho_stage_dev, uint8_t* material_stage_dev,
                            void* workspace_dev, size_t workspace_bytes, void* cuda_stream,
                            gdrr_volume** out) {
    if (!ctx) return fail(nullptr, GDRR_ERR_INVALID_ARG, "ctx is NULL");
    if (!out) return fail(ctx, GDRR_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    int rc = check_dims(ctx, nx, ny, nz, n_materials, layout);
    if (rc) return rc;
    if (!rho_host || !material_host || !rho_stage_dev || !material_stage_dev)
        return fail(ctx, GDRR_ERR_INVALID_ARG, "a host or staging pointer is NULL");
    return create_volume_impl(ctx, rho_host, material_host, rho_stage_dev, material_stage_dev, nx, ny, nz, dx_mm, dy_mm,
                              dz_mm, centre_mm, n_materials, layout, workspace_dev, workspace_bytes, cuda_stream, out);
}

int gdrr_volume_status(gdrr_context* ctx, const gdrr_volume* vol) {
    if (!ctx) return fail(nullptr, GDRR_ERR_INVALID_ARG, "ctx is NULL");
    if (!vol || vol->ctx != ctx) return fail(ctx, GDRR_ERR_INVALID_ARG, "volume is NULL or belongs to another context");
    if (int rc = volume_check(ctx, vol, true)) return rc;
    // also the Siddon walk's compact copy, where one has been launched: after this call nothing the library enqueues
    // for this volume waits on an event, which is what stream capture needs (tests/test_gpu_graph.py)
    for (size_t g = 0; g <= vol->groups.size(); ++g) {
        gdrr_volume* member = const_cast<gdrr_volume*>(g == 0 ? vol : vol->groups[g - 1]);
        std::lock_guard<std::mutex> lock(member->compact_mu);
        if (member->compact_launched && !member->compact_ready) {
            DeviceGuard guard(ctx->device);
            if (cudaError_t e = cudaEventSynchronize(member->compact_done))
                return cuda_fail(ctx, e, "waiting for the compact copy");
            member->compact_ready = true;
        }
    }
    return GDRR_OK;
}

int gdrr_destroy_volume(gdrr_volume* vol) {
    if (vol)
        for (gdrr_volume* g : vol->groups) gdrr_destroy_volume(g);
    if (vol && (vol->tex || vol->tex_array || vol->compact_done || vol->ingest_done)) {
        DeviceGuard guard(vol->ctx->device);
        if (vol->ingest_done) cudaEventDestroy(vol->ingest_done);
        if (vol->tex) cudaDestroyTextureObject(vol->tex);
        if (vol->tex_array) cudaFreeArray(vol->tex_array);
        if (vol->compact_done) cudaEventDestroy(vol->compact_done);
    }
    delete vol;
    return GDRR_OK;
}

// Installs a detector and a pose table (12 doubles per projection) as the context's geometry.
static int install_geometry(gdrr_context* ctx, int nu, int nv, double du_mm, double dv_mm, double u_offset_mm,
                            double v_offset_mm, int n_proj, std::vector<double>&& poses, double step_mm) {
    DeviceGuard guard(ctx->device);
    if (guard.status != cudaSuccess) return cuda_fail(ctx, guard.status, "cudaSetDevice");
    double* dev = nullptr;
    cudaError_t e = cudaMalloc(&dev, sizeof(double) * poses.size());
    if (e != cudaSuccess) return cuda_fail(ctx, e, "cudaMalloc(poses)");
    e = cudaMemcpy(dev, poses.data(), sizeof(double) * poses.size(), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { cudaFree(dev); return cuda_fail(ctx, e, "cudaMemcpy(poses)"); }
    if (ctx->has_geom && (nu != ctx->nu || nv != ctx->nv)) {
        // tables shaped by the old detector are no longer valid
        free_dev(ctx->flu_dev); free_dev(ctx->bt_dev); free_dev(ctx->gain_dev);
        ctx->has_spec = false;
    }
    free_dev(ctx->poses_dev);
    ctx->poses_dev = dev;
    ctx->poses = std::move(poses);
    ctx->nu = nu; ctx->nv = nv; ctx->du = du_mm; ctx->dv = dv_mm;
    ctx->u_off = u_offset_mm; ctx->v_off = v_offset_mm;
    ctx->n_proj = n_proj; ctx->step = step_mm;
    ctx->has_geom = true;
    return GDRR_OK;
}

int gdrr_set_geometry(gdrr_context* ctx, double sad_mm, double sdd_mm, double theta_rad,
                      int nu, int nv, double du_mm, double dv_mm, double u_offset_mm, double v_offset_mm,
                      int n_proj, const double* phi_rad, double step_mm) {
    if (!ctx) return fail(nullptr, GDRR_ERR_INVALID_ARG, "ctx is NULL");
    const double sc[] = {sad_mm, sdd_mm, theta_rad, du_mm, dv_mm, u_offset_mm, v_offset_mm, step_mm};
    if (!all_finite(sc, 8)) return fail(ctx, GDRR_ERR_INVALID_ARG, "a geometry scalar is not finite");
    if (!(sad_mm > 0) || !(sdd_mm > sad_mm))
        return fail(ctx, GDRR_ERR_INVALID_ARG, "need sdd > sad > 0 (got sad %g, sdd %g)", sad_mm, sdd_mm);
    if (nu <= 0 || nv <= 0 || !(du_mm > 0) || !(dv_mm > 0))
        return fail(ctx, GDRR_ERR_INVALID_ARG, "detector pixel counts and sizes must be positive");
    if (n_proj <= 0 || !phi_rad) return fail(ctx, GDRR_ERR_INVALID_ARG, "need n_proj >= 1 and phi_rad");
    if (!all_finite(phi_rad, (size_t)n_proj)) return fail(ctx, GDRR_ERR_INVALID_ARG, "a gantry angle is not finite");

    // cos/sin once, on the host; S, P, u_hat formed here in the order DESIGN.md a1 writes (plain IEEE
    // double products, this file is compiled without FMA contraction) and passed to the kernels as data
    std::vector<double> poses(12 * (size_t)n_proj, 0.0);
    const double aid = sdd_mm - sad_mm;
    for (int p = 0; p < n_proj; ++p) {
        const double phi = phi_rad[p], psi = phi + theta_rad;
        const double c = std::cos(phi), sn = std::sin(phi), cp = std::cos(psi), sp = std::sin(psi);
        double* q = &poses[12 * (size_t)p];
        q[0] = -(sad_mm * c); q[1] = -(sad_mm * sn); q[2] = 0.0;      // source on the circle of radius SAD  [Q1]
        q[3] = aid * cp;      q[4] = aid * sp;       q[5] = 0.0;      // detector origin P = AID * n_hat     [Q2]
        q[6] = -sp;           q[7] = cp;             q[8] = 0.0;      // u_hat = z_hat x n_hat               [Q3]
        q[9] = 0.0;           q[10] = 0.0;           q[11] = 1.0;     // v_hat = +z
    }
    return install_geometry(ctx, nu, nv, du_mm, dv_mm, u_offset_mm, v_offset_mm, n_proj, std::move(poses), step_mm);
}

int gdrr_set_geometry_poses(gdrr_context* ctx, int nu, int nv, double du_mm, double dv_mm,
                            double u_offset_mm, double v_offset_mm, int n_proj, const double* poses,
                            double step_mm) {
    if (!ctx) return fail(nullptr, GDRR_ERR_INVALID_ARG, "ctx is NULL");
    const double sc[] = {du_mm, dv_mm, u_offset_mm, v_offset_mm, step_mm};
    if (!all_finite(sc, 5)) return fail(ctx, GDRR_ERR_INVALID_ARG, "a geometry scalar is not finite");
    if (nu <= 0 || nv <= 0 || !(du_mm > 0) || !(dv_mm > 0))
        return fail(ctx, GDRR_ERR_INVALID_ARG, "detector pixel counts and sizes must be positive");
    if (n_proj <= 0 || !poses) return fail(ctx, GDRR_ERR_INVALID_ARG, "need n_proj >= 1 and poses");
    if (!all_finite(poses, 12 * (size_t)n_proj)) return fail(ctx, GDRR_ERR_INVALID_ARG, "a pose value is not finite");
    for (int p = 0; p < n_proj; ++p) {
        const double* q = poses + 12 * (size_t)p;
        const double *S = q, *P = q + 3, *uh = q + 6, *vh = q + 9;
        const double nrm[3] = {uh[1] * vh[2] - uh[2] * vh[1], uh[2] * vh[0] - uh[0] * vh[2], uh[0] * vh[1] - uh[1] * vh[0]};
        const double nn = nrm[0] * nrm[0] + nrm[1] * nrm[1] + nrm[2] * nrm[2];
        const double dist = (P[0] - S[0]) * nrm[0] + (P[1] - S[1]) * nrm[1] + (P[2] - S[2]) * nrm[2];
        if (!(nn > 0.0)) return fail(ctx, GDRR_ERR_INVALID_ARG, "projection %d: u_hat and v_hat do not span a plane", p);
        if (dist == 0.0) return fail(ctx, GDRR_ERR_INVALID_ARG, "projection %d: the source lies in the detector plane", p);
    }
    std::vector<double> copy(poses, poses + 12 * (size_t)n_proj);
    return install_geometry(ctx, nu, nv, du_mm, dv_mm, u_offset_mm, v_offset_mm, n_proj, std::move(copy), step_mm);
}

int gdrr_set_spectrum(gdrr_context* ctx, int n_energy, int n_materials,
                      const double* phi_weight, const double* response, const double* mu_hat,
                      const float* fluence_map, const double* bowtie_mu,
                      const double* bowtie_thickness_mm) {
    if (!ctx) return fail(nullptr, GDRR_ERR_INVALID_ARG, "ctx is NULL");
    if (n_energy <= 0 || n_energy > GDRR_MAX_ENERGIES)
        return fail(ctx, GDRR_ERR_INVALID_ARG, "n_energy must be in [1, %d] (got %d)", GDRR_MAX_ENERGIES, n_energy);
    if (n_materials <= 0) return fail(ctx, GDRR_ERR_INVALID_ARG, "n_materials must be >= 1");
    if (n_materials > GDRR_MAX_MATERIALS)
        return fail(ctx, GDRR_ERR_UNSUPPORTED, "n_materials %d > GDRR_MAX_MATERIALS %d", n_materials, GDRR_MAX_MATERIALS);
    if (!phi_weight || !response || !mu_hat) return fail(ctx, GDRR_ERR_INVALID_ARG, "a table pointer is NULL");
    if ((bowtie_mu == nullptr) != (bowtie_thickness_mm == nullptr))
        return fail(ctx, GDRR_ERR_INVALID_ARG, "bowtie_mu and bowtie_thickness_mm go together");
    if ((fluence_map || bowtie_mu) && !ctx->has_geom)
        return fail(ctx, GDRR_ERR_NOT_READY, "fluence map / bowtie need gdrr_set_geometry first (detector shape)");
    if (!all_finite(phi_weight, n_energy) || !all_finite(response, n_energy) ||
        !all_finite(mu_hat, (size_t)n_energy * n_materials) ||
        (bowtie_mu && (!all_finite(bowtie_mu, n_energy) || !all_finite(bowtie_thickness_mm, ctx->nu))))
        return fail(ctx, GDRR_ERR_INVALID_ARG, "a table entry is not finite");
    if (fluence_map) {
        const size_t n = (size_t)ctx->nu * ctx->nv;
        for (size_t k = 0; k < n; ++k)
            if (!std::isfinite(fluence_map[k])) return fail(ctx, GDRR_ERR_INVALID_ARG, "fluence map entry is not finite");
    }
    DeviceGuard guard(ctx->device);
    if (guard.status != cudaSuccess) return cuda_fail(ctx, guard.status, "cudaSetDevice");

    // exp(-tau) is evaluated as exp2(-log2(e) * tau): fold log2(e) into the tables
    const double log2e = 1.4426950408889634074;
    std::vector<float4> mu((size_t)n_energy);
    std::vector<float2> src((size_t)n_energy);
    for (int e = 0; e < n_energy; ++e) {
        float m4[4] = {0.f, 0.f, 0.f, 0.f};
        for (int m = 0; m < n_materials && m < 4; ++m) m4[m] = (float)(log2e * mu_hat[(size_t)m * n_energy + e]);
        mu[e] = make_float4(m4[0], m4[1], m4[2], m4[3]);
        src[e] = make_float2((float)(phi_weight[e] * response[e]), bowtie_mu ? (float)(log2e * bowtie_mu[e]) : 0.f);
    }
    float4* mu_dev = nullptr; float2* src_dev = nullptr; float* bt_dev = nullptr; float* flu_dev = nullptr;
    float* mu_all_dev = nullptr;
    cudaError_t e = cudaMalloc(&mu_dev, sizeof(float4) * n_energy);
    if (e == cudaSuccess && n_materials > 4) {       // the energy sum over more than four materials reads [E][M]
        std::vector<float> all((size_t)n_energy * n_materials);
        for (int en = 0; en < n_energy; ++en)
            for (int m = 0; m < n_materials; ++m)
                all[(size_t)en * n_materials + m] = (float)(log2e * mu_hat[(size_t)m * n_energy + en]);
        e = cudaMalloc(&mu_all_dev, sizeof(float) * all.size());
        if (e == cudaSuccess) e = cudaMemcpy(mu_all_dev, all.data(), sizeof(float) * all.size(), cudaMemcpyHostToDevice);
    }
    if (e == cudaSuccess) e = cudaMalloc(&src_dev, sizeof(float2) * n_energy);
    if (e == cudaSuccess) e = cudaMemcpy(mu_dev, mu.data(), sizeof(float4) * n_energy, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(src_dev, src.data(), sizeof(float2) * n_energy, cudaMemcpyHostToDevice);
    if (e == cudaSuccess && bowtie_mu) {
        std::vector<float> bt((size_t)ctx->nu);
        for (int i = 0; i < ctx->nu; ++i) bt[i] = (float)bowtie_thickness_mm[i];
        e = cudaMalloc(&bt_dev, sizeof(float) * ctx->nu);
        if (e == cudaSuccess) e = cudaMemcpy(bt_dev, bt.data(), sizeof(float) * ctx->nu, cudaMemcpyHostToDevice);
    }
    if (e == cudaSuccess && fluence_map) {
        const size_t n = (size_t)ctx->nu * ctx->nv;
        e = cudaMalloc(&flu_dev, sizeof(float) * n);
        if (e == cudaSuccess) e = cudaMemcpy(flu_dev, fluence_map, sizeof(float) * n, cudaMemcpyHostToDevice);
    }
    if (e != cudaSuccess) {
        free_dev(mu_dev); free_dev(src_dev); free_dev(bt_dev); free_dev(flu_dev); free_dev(mu_all_dev);
        return cuda_fail(ctx, e, "uploading the spectrum tables");
    }
    free_dev(ctx->mu_dev); free_dev(ctx->src_dev); free_dev(ctx->bt_dev); free_dev(ctx->flu_dev);
    if (n_energy != ctx->n_energy) free_dev(ctx->gain_dev);        // shaped by the old energy grid
    free_dev(ctx->mu_all_dev);
    ctx->mu_dev = mu_dev; ctx->src_dev = src_dev; ctx->bt_dev = bt_dev; ctx->flu_dev = flu_dev; ctx->mu_all_dev = mu_all_dev;
    ctx->n_energy = n_energy; ctx->n_mat = n_materials;
    ctx->has_spec = true;
    return GDRR_OK;
}

int gdrr_set_response_gain(gdrr_context* ctx, const float* gain) {
    if (!ctx) return fail(nullptr, GDRR_ERR_INVALID_ARG, "ctx is NULL");
    DeviceGuard guard(ctx->device);
    if (guard.status != cudaSuccess) return cuda_fail(ctx, guard.status, "cudaSetDevice");
    if (!gain) { free_dev(ctx->gain_dev); return GDRR_OK; }
    if (!ctx->has_geom || !ctx->has_spec)
        return fail(ctx, GDRR_ERR_NOT_READY, "the response gain needs gdrr_set_geometry and gdrr_set_spectrum first (its shape)");
    const size_t n = (size_t)ctx->n_energy * ctx->nv * ctx->nu;
    for (size_t k = 0; k < n; ++k)
        if (!std::isfinite(gain[k])) return fail(ctx, GDRR_ERR_INVALID_ARG, "a response gain entry is not finite");
    float* dev = nullptr;
    cudaError_t e = cudaMalloc(&dev, sizeof(float) * n);
    if (e == cudaSuccess) e = cudaMemcpy(dev, gain, sizeof(float) * n, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { free_dev(dev); return cuda_fail(ctx, e, "uploading the response gain"); }
    free_dev(ctx->gain_dev);
    ctx->gain_dev = dev;
    return GDRR_OK;
}

int gdrr_project(gdrr_context* ctx, const gdrr_volume* vol, int proj_begin, int proj_count,
                 float* signal_dev, float* line_integrals_dev, int32_t* ray_table_dev,
                 void* cuda_stream) {
    if (!ctx) return fail(nullptr, GDRR_ERR_INVALID_ARG, "ctx is NULL");
    if (!signal_dev) return fail(ctx, GDRR_ERR_INVALID_ARG, "signal_dev is NULL");
    ProjectParams P;
    int rc = fill_project(ctx, vol, proj_begin, proj_count, P);
    if (rc) return rc;
    P.signal = signal_dev; P.li = line_integrals_dev; P.ray_table = ray_table_dev;
    if (!vol->groups.empty() && !line_integrals_dev)
        return fail(ctx, GDRR_ERR_INVALID_ARG, "with more than four materials gdrr_project needs line_integrals_dev: the line "
                    "integrals of each group of four wait there for the energy sum");
    DeviceGuard guard(ctx->device);
    if (guard.status != cudaSuccess) return cuda_fail(ctx, guard.status, "cudaSetDevice");
    cudaError_t e = launch_project(P, vol, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "project kernel launch");
    ctx->launches += 1;
    return GDRR_OK;
}

int gdrr_project_host(gdrr_context* ctx, const gdrr_volume* vol, int proj_begin, int proj_count,
                      float* signal_host, float* signal_stage_dev, int stage_proj, void* cuda_stream) {
    if (!ctx) return fail(nullptr, GDRR_ERR_INVALID_ARG, "ctx is NULL");
    if (!signal_host || !signal_stage_dev || stage_proj < 1)
        return fail(ctx, GDRR_ERR_INVALID_ARG, "signal_host / signal_stage_dev is NULL or stage_proj < 1");
    ProjectParams P;
    int rc = fill_project(ctx, vol, proj_begin, proj_count, P);
    if (rc) return rc;
    DeviceGuard guard(ctx->device);
    if (guard.status != cudaSuccess) return cuda_fail(ctx, guard.status, "cudaSetDevice");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    cudaError_t e = cudaSuccess;
    if (!vol->groups.empty()) {
        // more than four materials: the groups' line integrals of one batch wait in a context-owned scratch for the
        // energy sum (the caller gave none); all batches run on stream s, so one scratch serves them in turn
        const size_t need = (size_t)std::min(proj_count, std::max(1, stage_proj / (stage_proj >= 2 ? 2 : 1))) *
                            (size_t)vol->n_mat * ctx->nu * ctx->nv;
        if (ctx->li_scratch_floats < need) {
            e = cudaStreamSynchronize(s);               // (an earlier call's batches may still read the old one)
            free_dev(ctx->li_scratch);
            ctx->li_scratch_floats = 0;
            if (e == cudaSuccess) e = cudaMalloc(&ctx->li_scratch, sizeof(float) * need);
            if (e != cudaSuccess) return cuda_fail(ctx, e, "cudaMalloc(line-integral scratch)");
            ctx->li_scratch_floats = need;
        }
    }
    if (!ctx->copy_stream) e = cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking);
    for (int k = 0; k < 2 && e == cudaSuccess; ++k) {
        if (!ctx->ev_done[k]) e = cudaEventCreateWithFlags(&ctx->ev_done[k], cudaEventDisableTiming);
        if (e == cudaSuccess && !ctx->ev_free[k]) e = cudaEventCreateWithFlags(&ctx->ev_free[k], cudaEventDisableTiming);
    }
    if (e != cudaSuccess) return cuda_fail(ctx, e, "creating the copy stream");
    // two half-buffers: the kernel fills one while the other drains to the host
    const size_t plane = (size_t)ctx->nu * ctx->nv;
    const int slots = stage_proj >= 2 ? 2 : 1;
    const int batch = stage_proj / slots;
    int used[2] = {0, 0};
    int done = 0;
    for (int b = 0; done < proj_count; ++b) {
        const int slot = b % slots;
        const int cnt = proj_count - done < batch ? proj_count - done : batch;
        float* stage = signal_stage_dev + (size_t)slot * batch * plane;
        if (used[slot]) e = cudaStreamWaitEvent(s, ctx->ev_free[slot], 0);
        if (e != cudaSuccess) break;
        ProjectParams Pb = P;
        Pb.g.proj_begin = proj_begin + done;
        Pb.g.proj_count = cnt;
        Pb.signal = stage; Pb.li = vol->groups.empty() ? nullptr : ctx->li_scratch; Pb.ray_table = nullptr;
        e = launch_project(Pb, vol, s);
        if (e != cudaSuccess) break;
        ctx->launches += 1;
        e = cudaEventRecord(ctx->ev_done[slot], s);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_done[slot], 0);
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(signal_host + (size_t)done * plane, stage, sizeof(float) * plane * cnt,
                                cudaMemcpyDeviceToHost, ctx->copy_stream);
        if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_free[slot], ctx->copy_stream);
        if (e != cudaSuccess) break;
        used[slot] = 1;
        done += cnt;
    }
    cudaError_t e2 = cudaStreamSynchronize(ctx->copy_stream);
    if (e == cudaSuccess) e = e2;
    // later work on the caller's stream must not overtake the drains either
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "gdrr_project_host");
    return GDRR_OK;
}

int gdrr_set_method(gdrr_context* ctx, int method) {
    if (!ctx) return fail(nullptr, GDRR_ERR_INVALID_ARG, "ctx is NULL");
    if (method != GDRR_METHOD_TRILINEAR && method != GDRR_METHOD_SIDDON && method != GDRR_METHOD_TEXTURE)
        return fail(ctx, GDRR_ERR_INVALID_ARG, "unknown method %d", method);
    ctx->method = method;
    return GDRR_OK;
}

int gdrr_volume_attach_texture(gdrr_context* ctx, gdrr_volume* vol, void* cuda_stream) {
    if (!ctx) return fail(nullptr, GDRR_ERR_INVALID_ARG, "ctx is NULL");
    if (!vol || vol->ctx != ctx) return fail(ctx, GDRR_ERR_INVALID_ARG, "volume is NULL or belongs to another context");
    if (vol->layout != GDRR_LAYOUT_LINEAR)
        return fail(ctx, GDRR_ERR_INVALID_ARG, "the texture variant is built from a GDRR_LAYOUT_LINEAR volume");
    if (vol->tex) return GDRR_OK;
    DeviceGuard guard(ctx->device);
    if (guard.status != cudaSuccess) return cuda_fail(ctx, guard.status, "cudaSetDevice");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const int vw = vol->vw;
    const cudaChannelFormatDesc desc = cudaCreateChannelDesc(32, vw > 1 ? 32 : 0, vw > 2 ? 32 : 0, vw > 2 ? 32 : 0,
                                                             cudaChannelFormatKindFloat);
    const cudaExtent ext = make_cudaExtent((size_t)vol->px, (size_t)vol->py, (size_t)vol->pz);
    cudaError_t e = cudaMalloc3DArray(&vol->tex_array, &desc, ext);
    if (e != cudaSuccess) { vol->tex_array = nullptr; return cuda_fail(ctx, e, "cudaMalloc3DArray"); }
    e = order_after_ingest(vol, s);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "cudaStreamWaitEvent");
    cudaMemcpy3DParms cp = {};
    cp.srcPtr = make_cudaPitchedPtr(vol->vox, (size_t)vol->px * vw * sizeof(float), (size_t)vol->px, (size_t)vol->py);
    cp.dstArray = vol->tex_array;
    cp.extent = ext;
    cp.kind = cudaMemcpyDeviceToDevice;
    e = cudaMemcpy3DAsync(&cp, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e == cudaSuccess) {
        cudaResourceDesc res = {};
        res.resType = cudaResourceTypeArray;
        res.res.array.array = vol->tex_array;
        cudaTextureDesc td = {};
        td.addressMode[0] = td.addressMode[1] = td.addressMode[2] = cudaAddressModeClamp;
        td.filterMode = cudaFilterModeLinear;
        td.readMode = cudaReadModeElementType;
        td.normalizedCoords = 0;
        e = cudaCreateTextureObject(&vol->tex, &res, &td, nullptr);
    }
    if (e != cudaSuccess) {
        cudaFreeArray(vol->tex_array);
        vol->tex_array = nullptr;
        vol->tex = 0;
        return cuda_fail(ctx, e, "building the texture");
    }
    return GDRR_OK;
}

int gdrr_denoise_scatter(gdrr_context* ctx, const float* s_hat_dev, float* s_dev, float* scratch_dev, int nu, int nv,
                         int n_images, double beta, double omega, int n_iter, double floor_value, void* cuda_stream) {
    if (!ctx) return fail(nullptr, GDRR_ERR_INVALID_ARG, "ctx is NULL");
    if (!s_hat_dev || !s_dev || !scratch_dev) return fail(ctx, GDRR_ERR_INVALID_ARG, "a device pointer is NULL");
    if (nu <= 0 || nv <= 0 || n_images <= 0 || n_iter < 0)
        return fail(ctx, GDRR_ERR_INVALID_ARG, "need positive sizes and n_iter >= 0");
    if (!(beta > 0.0) || !std::isfinite(beta) || !(floor_value > 0.0) || !(omega > 0.0) || !(omega < 2.0))
        return fail(ctx, GDRR_ERR_INVALID_ARG, "need beta > 0, floor_value > 0 and 0 < omega < 2");
    if (n_images > 65535) return fail(ctx, GDRR_ERR_UNSUPPORTED, "at most 65535 images per call");
    DeviceGuard guard(ctx->device);
    if (guard.status != cudaSuccess) return cuda_fail(ctx, guard.status, "cudaSetDevice");
    int launches = 0;
    cudaError_t e = launch_denoise(s_hat_dev, s_dev, scratch_dev, nu, nv, n_images, beta, omega, n_iter, floor_value,
                                   (cudaStream_t)cuda_stream, &launches);
    ctx->launches += launches;
    if (e != cudaSuccess) return cuda_fail(ctx, e, "denoise kernel launch");
    return GDRR_OK;
}

static_assert(kDenoiseStaticFloats == (size_t)GDRR_DENOISE_STATIC_MAX_FLOATS, "header and denoise.cu disagree");

// The denoiser for callers that cannot allocate: no cudaMalloc / cudaFree / allocating library call on this path.
int gdrr_denoise_scatter_static(gdrr_context* ctx, const float* s_hat_dev, float* s_dev, int nu, int nv, int n_images,
                                double beta, double omega, int n_iter, double floor_value, void* cuda_stream) {
    if (!ctx) return fail(nullptr, GDRR_ERR_INVALID_ARG, "ctx is NULL");
    if (!s_hat_dev || !s_dev) return fail(ctx, GDRR_ERR_INVALID_ARG, "a device pointer is NULL");
    if (nu <= 0 || nv <= 0 || n_images <= 0 || n_iter < 0)
        return fail(ctx, GDRR_ERR_INVALID_ARG, "need positive sizes and n_iter >= 0");
    if (!(beta > 0.0) || !std::isfinite(beta) || !(floor_value > 0.0) || !(omega > 0.0) || !(omega < 2.0))
        return fail(ctx, GDRR_ERR_INVALID_ARG, "need beta > 0, floor_value > 0 and 0 < omega < 2");
    if (n_images > 65535) return fail(ctx, GDRR_ERR_UNSUPPORTED, "at most 65535 images per call");
    const double pixels = (double)nu * (double)nv * (double)n_images;
    if (pixels > (double)GDRR_DENOISE_STATIC_MAX_FLOATS)
        return fail(ctx, GDRR_ERR_UNSUPPORTED,
                    "%d images of %d x %d = %.0f pixels exceed the static scratch of GDRR_DENOISE_STATIC_MAX_FLOATS = %d "
                    "pixels; use gdrr_denoise_scatter with a scratch buffer of your own, or fewer images per call",
                    n_images, nu, nv, pixels, (int)GDRR_DENOISE_STATIC_MAX_FLOATS);
    DeviceGuard guard(ctx->device);
    if (guard.status != cudaSuccess) return cuda_fail(ctx, guard.status, "cudaSetDevice");
    int launches = 0;
    cudaError_t e = launch_denoise_static(s_hat_dev, s_dev, nu, nv, n_images, beta, omega, n_iter, floor_value,
                                          (cudaStream_t)cuda_stream, &launches);
    ctx->launches += launches;
    if (e != cudaSuccess) return cuda_fail(ctx, e, "denoise kernel launch (static scratch)");
    return GDRR_OK;
}

int gdrr_set_sampler(gdrr_context* ctx, int sampler) {
    if (!ctx) return fail(nullptr, GDRR_ERR_INVALID_ARG, "ctx is NULL");
    if (sampler != GDRR_SAMPLER_AUTO && sampler != GDRR_SAMPLER_GATHER && sampler != GDRR_SAMPLER_STAGED)
        return fail(ctx, GDRR_ERR_INVALID_ARG, "unknown sampler %d", sampler);
    ctx->sampler = sampler;
    return GDRR_OK;
}

int gdrr_siddon_segments(gdrr_context* ctx, const gdrr_volume* vol, int proj_begin, int proj_count,
                         int32_t* n_segments_dev, void* cuda_stream) {
    if (!ctx) return fail(nullptr, GDRR_ERR_INVALID_ARG, "ctx is NULL");
    if (!n_segments_dev) return fail(ctx, GDRR_ERR_INVALID_ARG, "n_segments_dev is NULL");
    ProjectParams P;
    int rc = fill_project(ctx, vol, proj_begin, proj_count, P);
    if (rc) return rc;
    P.signal = nullptr; P.li = nullptr; P.ray_table = nullptr; P.seg_table = n_segments_dev;
    DeviceGuard guard(ctx->device);
    if (guard.status != cudaSuccess) return cuda_fail(ctx, guard.status, "cudaSetDevice");
    cudaError_t e = order_after_ingest(vol, (cudaStream_t)cuda_stream);
    if (e == cudaSuccess) e = ensure_compact(vol, (cudaStream_t)cuda_stream);
    if (e == cudaSuccess) e = launch_project_siddon(P, vol->vw, vol->layout, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "Siddon kernel launch");
    ctx->launches += 1;
    return GDRR_OK;
}

int gdrr_last_sampler(const gdrr_context* ctx) { return ctx ? ctx->last_sampler : 0; }

int gdrr_debug_set_skew(gdrr_context* ctx, int mode) {
    if (!ctx) return fail(nullptr, GDRR_ERR_INVALID_ARG, "ctx is NULL");
    if (mode < 0 || mode > 3) return fail(ctx, GDRR_ERR_INVALID_ARG, "skew mode must be 0..3 (got %d)", mode);
    ctx->debug_skew = (unsigned)mode;
    return GDRR_OK;
}

int gdrr_debug_ray_cells(gdrr_context* ctx, const gdrr_volume* vol, int projection, int i, int j, int sampler,
                         int32_t* cells_dev, int max_samples, int32_t* count_dev, void* cuda_stream) {
    if (!ctx) return fail(nullptr, GDRR_ERR_INVALID_ARG, "ctx is NULL");
    if (!cells_dev || !count_dev || max_samples < 0) return fail(ctx, GDRR_ERR_INVALID_ARG, "an output is NULL");
    if (sampler != GDRR_SAMPLER_GATHER && sampler != GDRR_SAMPLER_STAGED)
        return fail(ctx, GDRR_ERR_INVALID_ARG, "sampler must be GDRR_SAMPLER_GATHER or GDRR_SAMPLER_STAGED");
    ProjectParams P;
    int rc = fill_project(ctx, vol, projection, 1, P);
    if (rc) return rc;
    if (vol->layout != GDRR_LAYOUT_PACKED_QUAD) return fail(ctx, GDRR_ERR_INVALID_ARG, "the volume is not PACKED_QUAD");
    if (i < 0 || i >= ctx->nu || j < 0 || j >= ctx->nv) return fail(ctx, GDRR_ERR_INVALID_ARG, "pixel outside the detector");
    DeviceGuard guard(ctx->device);
    if (guard.status != cudaSuccess) return cuda_fail(ctx, guard.status, "cudaSetDevice");
    cudaError_t e = launch_debug_ray_cells(P, i, j, sampler == GDRR_SAMPLER_STAGED, cells_dev, max_samples, count_dev,
                                           (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "debug kernel launch");
    ctx->launches += 1;
    return GDRR_OK;
}

int gdrr_ray_setup(gdrr_context* ctx, const gdrr_volume* vol, int proj_begin, int proj_count,
                   int32_t* ray_table_dev, unsigned long long* n_samples_dev, void* cuda_stream) {
    if (!ctx) return fail(nullptr, GDRR_ERR_INVALID_ARG, "ctx is NULL");
    if (!ray_table_dev && !n_samples_dev)
        return fail(ctx, GDRR_ERR_INVALID_ARG, "both outputs are NULL");
    GeomParams g;
    int rc = fill_geom(ctx, vol, proj_begin, proj_count, g);
    if (rc) return rc;
    DeviceGuard guard(ctx->device);
    if (guard.status != cudaSuccess) return cuda_fail(ctx, guard.status, "cudaSetDevice");
    cudaError_t e = launch_ray_setup(g, ray_table_dev, n_samples_dev, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "ray-setup kernel launch");
    ctx->launches += 1;
    return GDRR_OK;
}

}  // extern "C"
