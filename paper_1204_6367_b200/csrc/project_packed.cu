// Steps a1-a7 fused, PACKED-QUAD layout (GDRR_LAYOUT_PACKED_QUAD): the fast path.
//
// Layout.  A voxel is ONE 32-bit word: fp32 rho whose three lowest mantissa
// bits carry tags (n_materials > 1): bits 0-1 the material index, bit 2 (first
// word of an element only) "all 8 corners of this cell have this material".
// Element (ix, iy, iz) of the device volume is the 2x2 quad of words
// {(ix,iy), (ix,iy+1), (ix+1,iy), (ix+1,iy+1)} of slab iz, stored for EVERY
// (ix, iy) (quads overlap, 16 B per voxel).  A sample needs two 16-byte loads
// (slabs iz and iz+1).
//
// What bounds the gather (profiles/r01_l1_model.md, measured on B200): a 16-byte
// warp-wide load is served in 4 phases of 8 lanes; inside a phase, distinct
// elements whose index is equal mod 8 (same 16-byte bank group of the L1 data
// RAM) serialise, whatever line they are in; the tag stage takes 4 lines per
// cycle.  So (1) the lanes of a warp must sample the SAME interval index k at
// the same time (intervals are laid from the source, so equal k is a sphere
// around the source and the warp's footprint stays a compact 2-D patch; starting
// every ray at its own j0 spreads the warp over up to 8 steps of depth), and
// (2) neighbouring elements must differ mod 8 in every direction: elements are
// stored linearly with the row stride = 3 and the slab stride = 4 (mod 8).
//
// Material routing.  In a segmented volume almost every cell is pure (98.8% of
// C3's cells), so the common path is one scalar tri-linear blend added to a
// running sum that is routed to its material only when the material changes;
// cells with mixed corners take a slower branch that routes each weighted
// corner.  Both give the same value.
//
// The words are used as floats as they are (|stored - rho| <= 11 ulp, DESIGN.md
// Q24); the library is compiled with -ftz=true so that rho = 0 tagged with a
// material (a denormal bit pattern) contributes exactly 0.
#include "packed_sampler.cuh"

namespace gdrr {

template <int VW>
__global__ void __launch_bounds__(kThreads, 4)
gdrr_project_packed_kernel(const ProjectParams P) {
    // the ray's line in index space (6 doubles) is needed once per chunk only: keep it in
    // shared memory, not in 12 registers of the sampling loop
    __shared__ double s_line[6][kThreads];
    __shared__ float s_acc[4][kAccStride];          // per-material sums of the rays (RayAcc)
    float4* s_mu;
    float2* s_src;
    load_tables(P, s_mu, s_src);

    int i, j;
    thread_pixel_map(i, j);
    const int pl = blockIdx.z;
    // lanes outside the detector stay in the warp (the loop below is warp-synchronous) with n = 0
    const bool valid = i < P.g.nu && j < P.g.nv;

    // ---- a1: ray setup (fp64) ------------------------------------------------
    int j0, n;
    Sampler S;
    {
        Ray r;
        ray_setup(P.g, P.g.proj_begin + pl, min(i, P.g.nu - 1), min(j, P.g.nv - 1), r);
        if (!valid) r.n = 0;
        if (valid && P.ray_table) {
            const size_t pix = ((size_t)pl * P.g.nv + j) * P.g.nu + i;
            reinterpret_cast<int2*>(P.ray_table)[pix] = make_int2(r.j0, r.n);
        }
        double gs[3], dg[3];
        index_line(P.g, r, gs, dg);
        S.dqx = __double2int_rn(dg[0] * 8388608.0);
        S.dqy = __double2int_rn(dg[1] * 8388608.0);
        S.dqz = __double2int_rn(dg[2] * 8388608.0);
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            s_line[a][threadIdx.x] = gs[a];
            s_line[3 + a][threadIdx.x] = dg[a];
        }
        j0 = r.j0;
        n = r.n;
    }
    S.sy = P.v.stride_y;
    S.sz = P.v.stride_z;
    S.vol0 = reinterpret_cast<const uint4*>(P.v.vox);
    S.vol1 = reinterpret_cast<const uint4*>(P.v.vox1);
    S.fmask = P.frac_mask;
    S.fone = P.one_bits;

    // Interval indices k are counted from the source (reading Q9), so all lanes of the
    // warp walk the same k: the warp's samples lie on a sphere around the source.
    const int kmin = __reduce_min_sync(0xffffffffu, n > 0 ? j0 : 0x7fffffff);
    const int kmax = __reduce_max_sync(0xffffffffu, n > 0 ? j0 + n : (int)0x80000000);
    const unsigned un = (unsigned)n;
    const int CH = P.chunk;

    // ---- a2-a4: sampling -------------------------------------------------------
    float acc[VW];
    RayAcc<VW> A;
    init_ray<VW>(A, &s_acc[0][threadIdx.x]);

    for (int kc = (kmin / CH) * CH; kc < kmax; kc += CH) {
        const int s0 = max(kmin - kc, 0);
        const int cnt = min(kmax - kc, CH) - s0;
        double gs[3], dg[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            gs[a] = s_line[a][threadIdx.x];
            dg[a] = s_line[3 + a][threadIdx.x];
        }
        const ChunkBase b = chunk_base(gs, dg, kc + s0);
        const unsigned rel = (unsigned)(kc + s0 - j0);
        const bool mine = rel < un && rel + (unsigned)cnt <= un;         // this lane owns the whole chunk
        if (__all_sync(0xffffffffu, mine) && !(cnt & 1))
            run_chunk_pairs<VW>(S, b, cnt, A);
        else
            run_chunk<VW, true>(S, b, cnt, rel, un, A);

        flush_chunk<VW>(A);
    }
    finish_ray<VW>(A, acc);

    if (valid) finish_pixel<VW>(P, s_mu, s_src, acc, P.g.step, pl, i, j);
}

template <int VW>
static cudaError_t launch_packed_t(const ProjectParams& p, cudaStream_t s) {
    dim3 grid((p.g.nu + kTileU - 1) / kTileU, (p.g.nv + kTileV - 1) / kTileV, p.g.proj_count);
    const size_t smem = (size_t)p.n_energy * (sizeof(float4) + sizeof(float2));
    gdrr_project_packed_kernel<VW><<<grid, kThreads, smem, s>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_project_packed(const ProjectParams& p, int vw, cudaStream_t s) {
    if (vw == 1) return launch_packed_t<1>(p, s);
    if (vw == 2) return launch_packed_t<2>(p, s);
    return launch_packed_t<4>(p, s);
}

}  // namespace gdrr
