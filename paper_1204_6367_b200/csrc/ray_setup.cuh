// Step a1: ray setup in fp64 (PAPER.md:93-95 geometry, PAPER.md:151 intervals).
//
// The integer ray table (j0, n) has one correct value per ray and is compared
// bit for bit with the CPU oracle, so every operation that feeds it is an
// explicitly rounded IEEE-754 double operation (__dadd_rn, __dmul_rn, __ddiv_rn,
// __dsqrt_rn: never contracted into an FMA) in the order DESIGN.md "a1" writes
// out.  Source and detector frame arrive as data (for the gantry: cos/sin taken
// once on the host, products formed there in the oracle's order).
#pragma once
#include "gdrr_internal.h"

namespace gdrr {

struct Ray {
    double S[3];        // source
    double dir[3];      // unit direction source -> pixel centre
    double t_in, t_out; // parameter range inside the volume box
    int j0, n;          // first midpoint index, number of midpoints (0 = miss)
    bool hit;           // the clipped segment [t_in, t_out] is not empty
};

__device__ __forceinline__ void ray_setup(const GeomParams& g, int p, int i, int j, Ray& r) {
    // the pose of projection p: source S, detector origin P, u_hat, v_hat (12 doubles).  For the
    // circular gantry the host fills it from (SAD, SDD, phi, theta) [Q1][Q2][Q3]; helical and C-arm
    // source paths give it directly [Q31]
    const double* pose = g.poses + 12 * (size_t)p;
    // one ray through the pixel centre D = (P + u u_hat) + v v_hat  [Q4][Q5]
    const double u = __dadd_rn(__dmul_rn(__dsub_rn((double)i, g.half_nu), g.du), g.u_off);
    const double v = __dadd_rn(__dmul_rn(__dsub_rn((double)j, g.half_nv), g.dv), g.v_off);
    double D[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        r.S[k] = pose[k];
        D[k] = __dadd_rn(__dadd_rn(pose[3 + k], __dmul_rn(u, pose[6 + k])), __dmul_rn(v, pose[9 + k]));
    }
    const double D0 = D[0], D1 = D[1];
    const double dx = __dsub_rn(D0, r.S[0]), dy = __dsub_rn(D1, r.S[1]), dz = __dsub_rn(D[2], r.S[2]);
    const double L = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)),
                                          __dmul_rn(dz, dz)));
    r.dir[0] = __ddiv_rn(dx, L);
    r.dir[1] = __ddiv_rn(dy, L);
    r.dir[2] = __ddiv_rn(dz, L);

    // slab clip of [0, L] against the volume box  [Q7][Q17]
    double t_in = 0.0, t_out = L;
    bool miss = false;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        if (r.dir[k] != 0.0) {
            const double t1 = __ddiv_rn(__dsub_rn(g.lo[k], r.S[k]), r.dir[k]);
            const double t2 = __ddiv_rn(__dsub_rn(g.hi[k], r.S[k]), r.dir[k]);
            const double tmin = t1 < t2 ? t1 : t2;
            const double tmax = t1 < t2 ? t2 : t1;
            if (tmin > t_in) t_in = tmin;
            if (tmax < t_out) t_out = tmax;
        } else if (r.S[k] < g.lo[k] || r.S[k] > g.hi[k]) {
            miss = true;
        }
    }
    r.t_in = t_in;
    r.t_out = t_out;
    r.hit = !miss && t_out > t_in;

    // midpoints t_k = (k + 1/2) dl laid from the source; count t_in <= t_k < t_out  [Q9]
    int j0 = 0, n = 0;
    if (!miss && t_out > t_in) {
        const double a0 = ceil(__dsub_rn(__ddiv_rn(t_in, g.step), 0.5));
        const double a1 = ceil(__dsub_rn(__ddiv_rn(t_out, g.step), 0.5));
        j0 = (int)a0;
        int j1 = (int)a1;
        if (j0 < 0) j0 = 0;
        if (j1 < j0) j1 = j0;
        n = j1 - j0;
    }
    r.j0 = j0;
    r.n = n;
}

}  // namespace gdrr
