/*
 * gdrr_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, double-precision CPU statement of the poly-energetic
 * primary-signal projector of gDRR (Jia et al., arXiv 1204.6367), Eq. (1):
 *
 *     P(u) = Int dE phi(E) w(u) r(E) exp[ - Int_L dl mu(x,E) ]
 *     mu(x,E) = rho(x) * sum_k mu_hat_k(i(x),E)
 *
 * with the energy integral a discrete sum over channels and the line integral
 * the paper's fixed-step rule: the source->pixel path is cut into intervals of
 * equal length dl, the field is tri-linearly interpolated at each interval's
 * MIDPOINT, and sum_j dl*mu(x_j,E) is the radiological length;
 * dl defaults to half the voxel size.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this file.  It shares no code with
 * paper_1204_6367_b200/ (the CUDA path) and that package never loads it.
 *
 * It is a discretisation, not a fast route to a closed form, so the oracle
 * follows the algorithm step by step in the paper's order.  Where the paper is
 * silent the readings are those of SURVEY.md section 8(c) (Q1..Q21), restated in
 * DESIGN.md; each is marked [Qn] below.  Loops are written out plainly; the
 * only parallelism is an OpenMP "parallel for" over detector rows so that it
 * can be timed on the host cores.
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): flat field, mono-
 * energetic Beer-Lambert, uniform-volume chord, tri-affine reproduction, node /
 * cell-centre values, exact piecewise-cubic line integral (independent numpy
 * code), analytic sphere chord, additivity / linearity, literal-vs-factored
 * identity, z-mirror and 90-degree rotation equivariance, shadow of the box; for the
 * Siddon option: per-voxel box clipping (brute force), uniform-volume chord, axis-parallel
 * rows, nearest-neighbour fine-step limit; for the scatter denoiser (tests/test_oracle_denoise_pins.py): a
 * numpy sweep, the constant fixed point, the eigenmode amplification factor, Eq. (4) at convergence.
 * No function here is "parity unpinned".
 *
 * Units: lengths mm, rho g/cm^3, mu_hat mm^-1 per g/cm^3, energies keV.
 * Build:  gcc -O2 -std=c99 -ffp-contract=off -fopenmp -shared -fPIC ...
 * (-ffp-contract=off: the integer ray table must not depend on FMA fusion.)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define GDRR_ORACLE_MAX_MATERIALS 16

typedef struct {
    /* volume: PAPER.md:97; axis order and placement [Q6] */
    const float *rho;          /* [nz][ny][nx], x fastest */
    const uint8_t *mat;        /* same shape */
    int n[3];                  /* nx, ny, nz */
    double d[3];               /* voxel size dx, dy, dz */
    double c[3];               /* centre of the volume box */
    int n_materials;
    /* geometry: PAPER.md:93-95 */
    double sad, sdd, theta;
    int nu, nv;
    double du, dv, u_off, v_off;
    double step;               /* dl */
    /* general source paths (helical, C-arm; "with simple modifications"): per projection
     * 12 doubles = source S, detector origin P, u_hat, v_hat; NULL = the circular gantry above */
    const double *poses;
} oracle_setup;

typedef struct {
    double S[3];               /* source */
    double dir[3];             /* unit direction source -> pixel centre */
    double L;                  /* source -> pixel distance */
    double t_in, t_out;        /* clipped parameter range inside the box */
    int hit;                   /* t_out > t_in */
    int32_t j0, n;             /* first midpoint index, number of midpoints */
} oracle_ray;

/* O1 + O2 + O3 + O4 of SURVEY.md section 8(c).  The order of the floating-point
 * operations below is part of the definition: (j0, n) is compared bit-exactly
 * with the CUDA path. */
static void ray_from_points(const oracle_setup *g, const double D[3], oracle_ray *r);

/* Pixel coordinates on the detector [Q4][Q5]. */
static void pixel_uv(const oracle_setup *g, int i, int j, double *u, double *v)
{
    *u = ((double)i - 0.5 * (double)(g->nu - 1)) * g->du + g->u_off;
    *v = ((double)j - 0.5 * (double)(g->nv - 1)) * g->dv + g->v_off;
}

static void ray_setup(const oracle_setup *g, double phi, int i, int j, oracle_ray *r)
{
    /* O1: source on the circle of radius SAD; SO makes angle phi with +x,
     * counter-clockwise seen from +z  [Q1]. */
    double c = cos(phi), s = sin(phi);
    double psi = phi + g->theta;           /* direction O->P  [Q2] */
    double cp = cos(psi), sp = sin(psi);
    double aid = g->sdd - g->sad;          /* axis-to-imager distance [Q2] */
    double Px = aid * cp, Py = aid * sp;   /* detector origin P */
    double ux = -sp, uy = cp;              /* u_hat = z_hat x n_hat  [Q3]; v_hat = +z */
    r->S[0] = -(g->sad * c);
    r->S[1] = -(g->sad * s);
    r->S[2] = 0.0;

    /* O2: one ray through the pixel centre [Q4][Q5] */
    double u, v;
    pixel_uv(g, i, j, &u, &v);
    double D[3];
    D[0] = Px + u * ux;
    D[1] = Py + u * uy;
    D[2] = v;
    ray_from_points(g, D, r);
}

/* O1-G + O2 for a general pose [Q31]: the source and the detector frame are given per projection,
 * pixel centre D = P + u u_hat + v v_hat, summed in that order.  With S, P, u_hat of the circular
 * gantry and v_hat = +z this is ray_setup() bit for bit (tests/test_oracle_pose_pins.py). */
static void ray_setup_pose(const oracle_setup *g, const double *pose, int i, int j, oracle_ray *r)
{
    const double *S = pose, *P = pose + 3, *uh = pose + 6, *vh = pose + 9;
    double u, v;
    pixel_uv(g, i, j, &u, &v);
    double D[3];
    for (int a = 0; a < 3; ++a) {
        r->S[a] = S[a];
        D[a] = (P[a] + u * uh[a]) + v * vh[a];
    }
    ray_from_points(g, D, r);
}

/* Tail of O2, O3, O4: the ray from r->S through the pixel centre D. */
static void ray_from_points(const oracle_setup *g, const double D[3], oracle_ray *r)
{
    double dx = D[0] - r->S[0], dy = D[1] - r->S[1], dz = D[2] - r->S[2];
    double L = sqrt((dx * dx + dy * dy) + dz * dz);
    r->L = L;
    r->dir[0] = dx / L;
    r->dir[1] = dy / L;
    r->dir[2] = dz / L;

    /* O3: slab clip of [0, L] against the volume box [Q7][Q17] */
    double t_in = 0.0, t_out = L;
    int miss = 0;
    for (int a = 0; a < 3; ++a) {
        double half = 0.5 * ((double)g->n[a] * g->d[a]);
        double lo = g->c[a] - half, hi = g->c[a] + half;
        if (r->dir[a] != 0.0) {
            double t1 = (lo - r->S[a]) / r->dir[a];
            double t2 = (hi - r->S[a]) / r->dir[a];
            double tmin = t1 < t2 ? t1 : t2;
            double tmax = t1 < t2 ? t2 : t1;
            if (tmin > t_in) t_in = tmin;
            if (tmax < t_out) t_out = tmax;
        } else if (r->S[a] < lo || r->S[a] > hi) {
            miss = 1;
        }
    }
    r->t_in = t_in;
    r->t_out = t_out;
    r->hit = (!miss && t_out > t_in);

    /* O4: intervals of length dl are laid from the SOURCE (t = 0); interval k
     * has midpoint t_k = (k + 1/2) dl; a midpoint counts iff
     * t_in <= t_k < t_out  [Q9]. */
    if (r->hit) {
        double a0 = ceil(t_in / g->step - 0.5);
        double a1 = ceil(t_out / g->step - 0.5);
        int32_t j0 = (int32_t)a0;
        int32_t j1 = (int32_t)a1;
        if (j0 < 0) j0 = 0;
        if (j1 < j0) j1 = j0;
        r->j0 = j0;
        r->n = j1 - j0;
    } else {
        r->j0 = 0;
        r->n = 0;
    }
}

/* Index-space coordinate of the world point S + t*dir: integer g <-> voxel
 * centre  [Q6]. */
static void index_coords(const oracle_setup *g, const oracle_ray *r, double t, double gi[3])
{
    for (int a = 0; a < 3; ++a) {
        double x = r->S[a] + t * r->dir[a];
        gi[a] = (x - g->c[a]) / g->d[a] + 0.5 * (double)(g->n[a] - 1);
    }
}

/* The 8 corners and weights of tri-linear interpolation at index coordinate
 * gi, with clamp-to-edge outside the lattice of voxel centres  [Q7].
 * PAPER.md:151 ("tri-linear interpolation scheme"). */
static void trilinear_stencil(const oracle_setup *g, const double gi[3],
                              int64_t lin[8], double w[8], int32_t cell[3])
{
    int i0[3], i1[3];
    double f[3];
    for (int a = 0; a < 3; ++a) {
        double fl = floor(gi[a]);
        int b = (int)fl;
        f[a] = gi[a] - fl;
        cell[a] = b;
        int lo = b, hi = b + 1;
        if (lo < 0) lo = 0;
        if (lo > g->n[a] - 1) lo = g->n[a] - 1;
        if (hi < 0) hi = 0;
        if (hi > g->n[a] - 1) hi = g->n[a] - 1;
        i0[a] = lo;
        i1[a] = hi;
    }
    int q = 0;
    for (int qz = 0; qz < 2; ++qz)
        for (int qy = 0; qy < 2; ++qy)
            for (int qx = 0; qx < 2; ++qx, ++q) {
                int ix = qx ? i1[0] : i0[0];
                int iy = qy ? i1[1] : i0[1];
                int iz = qz ? i1[2] : i0[2];
                double wx = qx ? f[0] : 1.0 - f[0];
                double wy = qy ? f[1] : 1.0 - f[1];
                double wz = qz ? f[2] : 1.0 - f[2];
                lin[q] = ((int64_t)iz * g->n[1] + iy) * g->n[0] + ix;
                w[q] = wx * wy * wz;
            }
}

/* O5: per-material line integrals  LI_m = dl * sum_k trilinear(rho_m)(x_k),
 * rho_m = rho * [material == m]   (north_star's factored form; identical to
 * the paper's per-energy form by linearity of the interpolant, [Q10]). */
static void ray_line_integrals(const oracle_setup *g, const oracle_ray *r, double *LI)
{
    for (int m = 0; m < g->n_materials; ++m) LI[m] = 0.0;
    for (int32_t k = r->j0; k < r->j0 + r->n; ++k) {
        double t = ((double)k + 0.5) * g->step;
        double gi[3], w[8];
        int64_t lin[8];
        int32_t cell[3];
        index_coords(g, r, t, gi);
        trilinear_stencil(g, gi, lin, w, cell);
        for (int q = 0; q < 8; ++q)
            LI[g->mat[lin[q]]] += w[q] * (double)g->rho[lin[q]];
    }
    for (int m = 0; m < g->n_materials; ++m) LI[m] *= g->step;
}

/* O5': the paper-literal form.  For ONE energy channel the voxel field is
 * mu_E(voxel) = rho(voxel) * mu_hat[mat(voxel)][E] and the
 * radiological length is dl * sum_j trilinear(mu_E)(x_j). */
static double ray_radiological_length(const oracle_setup *g, const oracle_ray *r,
                                      const double *mu_hat_E /* [n_materials] */)
{
    double tau = 0.0;
    for (int32_t k = r->j0; k < r->j0 + r->n; ++k) {
        double t = ((double)k + 0.5) * g->step;
        double gi[3], w[8];
        int64_t lin[8];
        int32_t cell[3];
        index_coords(g, r, t, gi);
        trilinear_stencil(g, gi, lin, w, cell);
        double mu = 0.0;
        for (int q = 0; q < 8; ++q)
            mu += w[q] * ((double)g->rho[lin[q]] * mu_hat_E[g->mat[lin[q]]]);
        tau += mu;
    }
    return tau * g->step;
}

/* O5-S: Siddon's exact radiological path ("this line integral is usually
 * evaluated using Siddon's ray-tracing algorithm", "also available in gDRR",
 * ref. 3 at PAPER.md:442).  The voxels are homogeneous boxes; voxel (ix, iy, iz) occupies
 * [lo_a + i_a d_a, lo_a + (i_a + 1) d_a) on each axis [Q26], and
 *     LI_m = sum over voxels of  rho(voxel) [material(voxel) == m] * |ray /\ voxel| .
 * Siddon's construction, step by step: (1) the parameter values at which the ray crosses
 * the x-, y- and z-planes of the lattice, kept if they fall inside the clipped range
 * (t_in, t_out) of O3; (2) merged with t_in and t_out into one sorted list; (3) each pair of
 * neighbours is one voxel's segment: its length is the difference, its voxel is the one that
 * contains the segment's midpoint.  Segments of zero length (the ray passes through a lattice
 * edge or corner) contribute nothing, so ties need no rule.  Returns the number of segments
 * of positive length. */
static int cmp_double(const void *a, const void *b)
{
    double x = *(const double *)a, y = *(const double *)b;
    return (x > y) - (x < y);
}

static int ray_siddon(const oracle_setup *g, const oracle_ray *r, double *LI)
{
    for (int m = 0; m < g->n_materials; ++m) LI[m] = 0.0;
    if (!r->hit) return 0;
    int cap = g->n[0] + g->n[1] + g->n[2] + 5, cnt = 0;
    double *t = (double *)malloc(sizeof(double) * (size_t)cap);
    double lo[3];
    if (!t) return -1;
    t[cnt++] = r->t_in;
    for (int a = 0; a < 3; ++a) {
        lo[a] = g->c[a] - 0.5 * ((double)g->n[a] * g->d[a]);
        if (r->dir[a] == 0.0) continue;
        for (int i = 0; i <= g->n[a]; ++i) {
            double plane = lo[a] + (double)i * g->d[a];
            double tt = (plane - r->S[a]) / r->dir[a];
            if (tt > r->t_in && tt < r->t_out) t[cnt++] = tt;
        }
    }
    t[cnt++] = r->t_out;
    qsort(t, (size_t)cnt, sizeof(double), cmp_double);
    int nseg = 0;
    for (int q = 0; q + 1 < cnt; ++q) {
        double len = t[q + 1] - t[q];
        if (!(len > 0.0)) continue;
        double tm = 0.5 * (t[q] + t[q + 1]);
        int64_t idx[3];
        for (int a = 0; a < 3; ++a) {
            double x = r->S[a] + tm * r->dir[a];
            int64_t v = (int64_t)floor((x - lo[a]) / g->d[a]);
            if (v < 0) v = 0;
            if (v > g->n[a] - 1) v = g->n[a] - 1;
            idx[a] = v;
        }
        int64_t lin = (idx[2] * g->n[1] + idx[1]) * g->n[0] + idx[0];
        LI[g->mat[lin]] += (double)g->rho[lin] * len;
        ++nseg;
    }
    free(t);
    return nseg;
}

static int fill_setup(oracle_setup *g, const float *rho, const uint8_t *mat,
                      int nx, int ny, int nz, double dx, double dy, double dz,
                      const double *centre, int n_materials,
                      double sad, double sdd, double theta,
                      int nu, int nv, double du, double dv, double u_off, double v_off,
                      double step)
{
    if (nx <= 0 || ny <= 0 || nz <= 0 || dx <= 0 || dy <= 0 || dz <= 0) return -1;
    if (n_materials <= 0 || n_materials > GDRR_ORACLE_MAX_MATERIALS) return -1;
    if (!(sdd > sad) || !(sad > 0) || nu <= 0 || nv <= 0 || du <= 0 || dv <= 0) return -1;
    g->rho = rho; g->mat = mat;
    g->n[0] = nx; g->n[1] = ny; g->n[2] = nz;
    g->d[0] = dx; g->d[1] = dy; g->d[2] = dz;
    for (int a = 0; a < 3; ++a) g->c[a] = centre ? centre[a] : 0.0;
    g->n_materials = n_materials;
    g->sad = sad; g->sdd = sdd; g->theta = theta;
    g->nu = nu; g->nv = nv; g->du = du; g->dv = dv; g->u_off = u_off; g->v_off = v_off;
    if (step <= 0.0) {                     /* [Q8]: half the smallest voxel edge */
        double m = dx < dy ? dx : dy;
        if (dz < m) m = dz;
        step = 0.5 * m;
    }
    g->step = step;
    g->poses = NULL;
    return 0;
}

/* O6: energy sum for one pixel.  PAPER.md:147 with the integral over E a sum
 * over channels and the source model of [Q13]:
 * phi_b(E,u) = phi_E * w(u) * exp(-mu_bt(E) * t_bt(u)). */
static double energy_sum(int n_energy, int n_materials, const double *phi_w,
                         const double *resp, const double *mu_hat, double w_pix,
                         const double *bt_mu, double bt_t, const double *LI,
                         const float *gain_pix /* NULL, or this pixel's g(E, u) with stride gain_stride [Q32] */,
                         size_t gain_stride)
{
    double P = 0.0;
    for (int e = 0; e < n_energy; ++e) {
        double tau = 0.0;
        for (int m = 0; m < n_materials; ++m)
            tau += mu_hat[(size_t)m * n_energy + e] * LI[m];
        double src = phi_w[e] * w_pix;
        if (bt_mu) src *= exp(-bt_mu[e] * bt_t);
        /* r(E, u) = r(E) g(E, u): "In principle, the detector response could also be pixel dependent"
         * (PAPER.md:111); g = 1 (NULL) is the paper's own pixel-independent case, bit for bit  [Q32] */
        double r = gain_pix ? resp[e] * (double)gain_pix[(size_t)e * gain_stride] : resp[e];
        P += src * r * exp(-tau);
    }
    return P;
}

/* ---------------------------------------------------------------- exports */

/* Geometry of one ray.  out[0..2]=S, [3..5]=dir, [6]=L, [7]=t_in, [8]=t_out;
 * table[0]=j0, table[1]=n, table[2]=hit. */
int gdrr_oracle_ray(int nx, int ny, int nz, double dx, double dy, double dz,
                    const double *centre, double sad, double sdd, double theta,
                    int nu, int nv, double du, double dv, double u_off, double v_off,
                    double step, double phi, int i, int j, double *out, int32_t *table)
{
    oracle_setup g;
    if (fill_setup(&g, NULL, NULL, nx, ny, nz, dx, dy, dz, centre, 1, sad, sdd, theta,
                   nu, nv, du, dv, u_off, v_off, step)) return -1;
    oracle_ray r;
    ray_setup(&g, phi, i, j, &r);
    for (int a = 0; a < 3; ++a) { out[a] = r.S[a]; out[3 + a] = r.dir[a]; }
    out[6] = r.L; out[7] = r.t_in; out[8] = r.t_out;
    table[0] = r.j0; table[1] = r.n; table[2] = r.hit;
    return 0;
}

/* Tri-linear interpolant of rho (all materials together) at n_pts index-space
 * points gi[n_pts][3]; clamp-to-edge.  For the P4/P5 pins. */
int gdrr_oracle_trilinear(const float *rho, int nx, int ny, int nz,
                          int n_pts, const double *gi, double *out)
{
    oracle_setup g;
    memset(&g, 0, sizeof g);
    g.n[0] = nx; g.n[1] = ny; g.n[2] = nz;
    for (int p = 0; p < n_pts; ++p) {
        int64_t lin[8];
        double w[8];
        int32_t cell[3];
        trilinear_stencil(&g, gi + 3 * (size_t)p, lin, w, cell);
        double v = 0.0;
        for (int q = 0; q < 8; ++q) v += w[q] * (double)rho[lin[q]];
        out[p] = v;
    }
    return 0;
}

/* Per-sample index coordinates and cells of one ray (for the cell-index check
 * [Q9]).  Writes at most max_samples entries; returns n (or <0 on error). */
int gdrr_oracle_ray_samples(int nx, int ny, int nz, double dx, double dy, double dz,
                            const double *centre, double sad, double sdd, double theta,
                            int nu, int nv, double du, double dv, double u_off, double v_off,
                            double step, double phi, int i, int j,
                            int max_samples, double *gi_out /* [n][3] */,
                            int32_t *cell_out /* [n][3] */)
{
    oracle_setup g;
    if (fill_setup(&g, NULL, NULL, nx, ny, nz, dx, dy, dz, centre, 1, sad, sdd, theta,
                   nu, nv, du, dv, u_off, v_off, step)) return -1;
    oracle_ray r;
    ray_setup(&g, phi, i, j, &r);
    for (int32_t k = 0; k < r.n && k < max_samples; ++k) {
        double t = ((double)(r.j0 + k) + 0.5) * g.step;
        double gi[3];
        index_coords(&g, &r, t, gi);
        for (int a = 0; a < 3; ++a) {
            gi_out[3 * (size_t)k + a] = gi[a];
            cell_out[3 * (size_t)k + a] = (int32_t)floor(gi[a]);
        }
    }
    return r.n;
}

/*
 * The projector.  Computes the listed pixels, or every pixel of every
 * projection when n_pix == 0.
 *   pix            [n_pix][3] = (projection p, column i, row j), or NULL
 *   signal         out, [n_proj][nv][nu] (all pixels) or [n_pix]
 *   line_integrals out or NULL, [n_proj][M][nv][nu] or [n_pix][M]
 *   ray_table      out or NULL, [n_proj][nv][nu][2] or [n_pix][2] = (j0, n)
 *   n_threads      <= 0: OpenMP default
 * Returns 0, or -1 on invalid arguments.
 */
static int project_impl(int method /* 0 tri-linear midpoint rule, 1 Siddon */, int32_t *n_segments,
                        const double *poses /* [n_proj][12] or NULL = circular gantry */,
                        const float *response_gain /* [n_energy][nv][nu] g(E, u) or NULL = 1  [Q32] */,
                        const float *rho, const uint8_t *mat,
                        int nx, int ny, int nz, double dx, double dy, double dz,
                        const double *centre, int n_materials,
                        double sad, double sdd, double theta,
                        int nu, int nv, double du, double dv, double u_off, double v_off,
                        int n_proj, const double *phi, double step,
                        int n_energy, const double *phi_w, const double *resp,
                        const double *mu_hat, const float *fluence,
                        const double *bt_mu, const double *bt_thick,
                        int64_t n_pix, const int32_t *pix,
                        double *signal, double *line_integrals, int32_t *ray_table,
                        int n_threads)
{
    oracle_setup g;
    if (fill_setup(&g, rho, mat, nx, ny, nz, dx, dy, dz, centre, n_materials, sad, sdd,
                   theta, nu, nv, du, dv, u_off, v_off, step)) return -1;
    if (n_proj <= 0 || n_energy <= 0 || (!phi && !poses) || !phi_w || !resp || !mu_hat || !signal)
        return -1;
    if ((bt_mu == NULL) != (bt_thick == NULL)) return -1;
    g.poses = poses;
    const int M = n_materials;
    const int64_t total = n_pix > 0 ? n_pix : (int64_t)n_proj * nv * nu;
    int bad = 0;
#ifdef _OPENMP
#pragma omp parallel for schedule(static, 256) num_threads(n_threads > 0 ? n_threads : omp_get_max_threads())
#endif
    for (int64_t q = 0; q < total; ++q) {
        int p, i, j;
        if (n_pix > 0) {
            p = pix[3 * q]; i = pix[3 * q + 1]; j = pix[3 * q + 2];
            if (p < 0 || p >= n_proj || i < 0 || i >= nu || j < 0 || j >= nv) {
#ifdef _OPENMP
#pragma omp atomic write
#endif
                bad = 1;
                continue;
            }
        } else {
            p = (int)(q / ((int64_t)nv * nu));
            int64_t rem = q - (int64_t)p * nv * nu;
            j = (int)(rem / nu);
            i = (int)(rem - (int64_t)j * nu);
        }
        oracle_ray r;
        double LI[GDRR_ORACLE_MAX_MATERIALS];
        if (g.poses) ray_setup_pose(&g, g.poses + 12 * (size_t)p, i, j, &r);
        else ray_setup(&g, phi[p], i, j, &r);
        if (method == 1) {
            int nseg = ray_siddon(&g, &r, LI);
            if (n_segments) n_segments[q] = nseg;
        } else {
            ray_line_integrals(&g, &r, LI);
        }
        double w_pix = fluence ? (double)fluence[(size_t)j * nu + i] : 1.0;
        double bt_t = bt_thick ? bt_thick[i] : 0.0;
        signal[q] = energy_sum(n_energy, M, phi_w, resp, mu_hat, w_pix, bt_mu, bt_t, LI,
                               response_gain ? response_gain + (size_t)j * nu + i : NULL, (size_t)nv * nu);
        if (line_integrals) {
            if (n_pix > 0) {
                for (int m = 0; m < M; ++m) line_integrals[(size_t)q * M + m] = LI[m];
            } else {
                for (int m = 0; m < M; ++m)
                    line_integrals[(((size_t)p * M + m) * nv + j) * nu + i] = LI[m];
            }
        }
        if (ray_table) {
            ray_table[2 * q] = r.j0;
            ray_table[2 * q + 1] = r.n;
        }
    }
    return bad ? -1 : 0;
}

int gdrr_oracle_project(const float *rho, const uint8_t *mat,
                        int nx, int ny, int nz, double dx, double dy, double dz,
                        const double *centre, int n_materials,
                        double sad, double sdd, double theta,
                        int nu, int nv, double du, double dv, double u_off, double v_off,
                        int n_proj, const double *phi, double step,
                        int n_energy, const double *phi_w, const double *resp,
                        const double *mu_hat, const float *fluence,
                        const double *bt_mu, const double *bt_thick,
                        int64_t n_pix, const int32_t *pix,
                        double *signal, double *line_integrals, int32_t *ray_table,
                        int n_threads)
{
    return project_impl(0, NULL, NULL, NULL, rho, mat, nx, ny, nz, dx, dy, dz, centre, n_materials, sad, sdd, theta,
                        nu, nv, du, dv, u_off, v_off, n_proj, phi, step, n_energy, phi_w, resp, mu_hat,
                        fluence, bt_mu, bt_thick, n_pix, pix, signal, line_integrals, ray_table, n_threads);
}

/* The same projector with the line integrals of O5-S (Siddon) instead of O5.
 *   n_segments  out or NULL, [n_proj][nv][nu] or [n_pix]: voxel segments of positive length */
int gdrr_oracle_project_siddon(const float *rho, const uint8_t *mat,
                        int nx, int ny, int nz, double dx, double dy, double dz,
                        const double *centre, int n_materials,
                        double sad, double sdd, double theta,
                        int nu, int nv, double du, double dv, double u_off, double v_off,
                        int n_proj, const double *phi, double step,
                        int n_energy, const double *phi_w, const double *resp,
                        const double *mu_hat, const float *fluence,
                        const double *bt_mu, const double *bt_thick,
                        int64_t n_pix, const int32_t *pix,
                        double *signal, double *line_integrals, int32_t *ray_table,
                        int32_t *n_segments, int n_threads)
{
    return project_impl(1, n_segments, NULL, NULL, rho, mat, nx, ny, nz, dx, dy, dz, centre, n_materials, sad, sdd,
                        theta, nu, nv, du, dv, u_off, v_off, n_proj, phi, step, n_energy, phi_w, resp,
                        mu_hat, fluence, bt_mu, bt_thick, n_pix, pix, signal, line_integrals, ray_table,
                        n_threads);
}

/* The same projector (method 0 tri-linear, 1 Siddon) on a general source path [Q31]:
 *   poses  [n_proj][12] = per projection source S, detector origin P, u_hat, v_hat (world, mm)
 * The detector frame is used as given (u_hat, v_hat are expected to be unit and orthogonal). */
int gdrr_oracle_project_poses(int method, const float *rho, const uint8_t *mat,
                        int nx, int ny, int nz, double dx, double dy, double dz,
                        const double *centre, int n_materials,
                        int nu, int nv, double du, double dv, double u_off, double v_off,
                        int n_proj, const double *poses, double step,
                        int n_energy, const double *phi_w, const double *resp,
                        const double *mu_hat, const float *fluence,
                        const double *bt_mu, const double *bt_thick,
                        int64_t n_pix, const int32_t *pix,
                        double *signal, double *line_integrals, int32_t *ray_table,
                        int32_t *n_segments, int n_threads)
{
    if (!poses || (method != 0 && method != 1)) return -1;
    /* sad, sdd are not used on this path: any valid pair passes fill_setup */
    return project_impl(method, method == 1 ? n_segments : NULL, poses, NULL, rho, mat, nx, ny, nz, dx, dy, dz,
                        centre, n_materials, 1.0, 2.0, 0.0, nu, nv, du, dv, u_off, v_off, n_proj, NULL,
                        step, n_energy, phi_w, resp, mu_hat, fluence, bt_mu, bt_thick, n_pix, pix, signal,
                        line_integrals, ray_table, n_threads);
}

/* The projector with every option: method 0 / 1, the circular gantry (phi, poses == NULL) or a general source path
 * (poses, phi == NULL; sad, sdd, theta then unused), and a pixel-dependent detector response [Q32]
 *   response_gain  [n_energy][nv][nu] float32 g(E, u), or NULL (= 1): r(E, u) = r(E) g(E, u). */
int gdrr_oracle_project_general(int method, const float *rho, const uint8_t *mat,
                        int nx, int ny, int nz, double dx, double dy, double dz,
                        const double *centre, int n_materials,
                        double sad, double sdd, double theta,
                        int nu, int nv, double du, double dv, double u_off, double v_off,
                        int n_proj, const double *phi, const double *poses, double step,
                        int n_energy, const double *phi_w, const double *resp,
                        const double *mu_hat, const float *fluence,
                        const double *bt_mu, const double *bt_thick, const float *response_gain,
                        int64_t n_pix, const int32_t *pix,
                        double *signal, double *line_integrals, int32_t *ray_table,
                        int32_t *n_segments, int n_threads)
{
    if ((method != 0 && method != 1) || ((phi == NULL) == (poses == NULL))) return -1;
    if (poses) { sad = 1.0; sdd = 2.0; theta = 0.0; }
    return project_impl(method, method == 1 ? n_segments : NULL, poses, response_gain, rho, mat, nx, ny, nz,
                        dx, dy, dz, centre, n_materials, sad, sdd, theta, nu, nv, du, dv, u_off, v_off, n_proj,
                        phi, step, n_energy, phi_w, resp, mu_hat, fluence, bt_mu, bt_thick, n_pix, pix, signal,
                        line_integrals, ray_table, n_threads);
}

/* Geometry of one ray of a general pose; outputs as gdrr_oracle_ray. */
int gdrr_oracle_ray_pose(int nx, int ny, int nz, double dx, double dy, double dz,
                         const double *centre, int nu, int nv, double du, double dv,
                         double u_off, double v_off, double step, const double *pose,
                         int i, int j, double *out, int32_t *table)
{
    oracle_setup g;
    if (!pose || fill_setup(&g, NULL, NULL, nx, ny, nz, dx, dy, dz, centre, 1, 1.0, 2.0, 0.0,
                            nu, nv, du, dv, u_off, v_off, step)) return -1;
    oracle_ray r;
    ray_setup_pose(&g, pose, i, j, &r);
    for (int a = 0; a < 3; ++a) { out[a] = r.S[a]; out[3 + a] = r.dir[a]; }
    out[6] = r.L; out[7] = r.t_in; out[8] = r.t_out;
    table[0] = r.j0; table[1] = r.n; table[2] = r.hit;
    return 0;
}

/*
 * Paper-literal form (O5'): one full ray trace per energy channel on the field
 * mu_E = rho * mu_hat[mat][E], then Eq. (1).  n_pix listed pixels only (it is
 * n_energy / n_materials times slower).
 *   tau     out or NULL, [n_pix][n_energy] radiological lengths
 *   signal  out, [n_pix]
 */
int gdrr_oracle_project_literal(const float *rho, const uint8_t *mat,
                                int nx, int ny, int nz, double dx, double dy, double dz,
                                const double *centre, int n_materials,
                                double sad, double sdd, double theta,
                                int nu, int nv, double du, double dv, double u_off, double v_off,
                                int n_proj, const double *phi, double step,
                                int n_energy, const double *phi_w, const double *resp,
                                const double *mu_hat, const float *fluence,
                                const double *bt_mu, const double *bt_thick,
                                int64_t n_pix, const int32_t *pix,
                                double *signal, double *tau_out, int n_threads)
{
    oracle_setup g;
    if (fill_setup(&g, rho, mat, nx, ny, nz, dx, dy, dz, centre, n_materials, sad, sdd,
                   theta, nu, nv, du, dv, u_off, v_off, step)) return -1;
    if (n_pix <= 0 || !pix || n_proj <= 0 || n_energy <= 0 || !signal) return -1;
    if ((bt_mu == NULL) != (bt_thick == NULL)) return -1;
    const int M = n_materials;
#ifdef _OPENMP
#pragma omp parallel for schedule(static, 16) num_threads(n_threads > 0 ? n_threads : omp_get_max_threads())
#endif
    for (int64_t q = 0; q < n_pix; ++q) {
        int p = pix[3 * q], i = pix[3 * q + 1], j = pix[3 * q + 2];
        oracle_ray r;
        ray_setup(&g, phi[p], i, j, &r);
        double w_pix = fluence ? (double)fluence[(size_t)j * nu + i] : 1.0;
        double bt_t = bt_thick ? bt_thick[i] : 0.0;
        double P = 0.0;
        for (int e = 0; e < n_energy; ++e) {       /* "Within each energy channel ..." PAPER.md:151 */
            double mu_E[GDRR_ORACLE_MAX_MATERIALS];
            for (int m = 0; m < M; ++m) mu_E[m] = mu_hat[(size_t)m * n_energy + e];
            double tau = ray_radiological_length(&g, &r, mu_E);
            if (tau_out) tau_out[(size_t)q * n_energy + e] = tau;
            double src = phi_w[e] * w_pix;
            if (bt_mu) src *= exp(-bt_mu[e] * bt_t);
            P += src * resp[e] * exp(-tau);
        }
        signal[q] = P;
    }
    return 0;
}

/*
 * Scatter denoising, PAPER.md:199-218 (section 2.5).  The noisy scatter image S_hat is modelled as
 * Poisson with a smooth mean S minimising  E[S] = Int (S - S_hat log S) + beta/2 Int |grad S|^2
 * (Eq. (2)); with the 5-point Laplacian the optimality condition is Eq. (4)
 * and the paper iterates Eq. (5):
 *
 *   S(k+1)(i,j) = (1 - w) S(k)(i,j) + w/4 [ Sum S(k)(i,j) - 1/beta (1 - S_hat(i,j) / S(k)(i,j)) ],
 *   Sum S(i,j) = S(i+1,j) + S(i,j+1) + S(i-1,j) + S(i,j-1),   w = 0.8,   S(0) = S_hat.
 *
 * Every value on the right is of iteration k (a relaxed Jacobi sweep), exactly as printed.
 * Readings where the paper is silent: [Q28] neighbours outside the detector are replaced by the
 * nearest pixel inside (replicate = zero normal derivative, the natural boundary condition of
 * the |grad S|^2 penalty); [Q29] S is kept >= floor > 0 (S(0) = max(S_hat, floor), each iterate
 * clamped) so that S_hat / S is defined where the Monte Carlo image has empty pixels; [Q30] a
 * fixed number of sweeps n_iter (the paper gives no stopping rule).
 *   s_hat  in  [nv][nu];  s0 in [nv][nu] or NULL (= s_hat);  s_out out [nv][nu];  work [nv][nu] scratch
 * Returns 0, or -1 on invalid arguments.
 */
int gdrr_oracle_denoise(const double *s_hat, const double *s0, int nu, int nv, double beta, double omega,
                        int n_iter, double floor_value, double *s_out, double *work)
{
    if (!s_hat || !s_out || !work || nu <= 0 || nv <= 0 || !(beta > 0.0) || n_iter < 0 || !(floor_value > 0.0))
        return -1;
    double *cur = s_out, *nxt = work;
    for (int q = 0; q < nu * nv; ++q) {
        double v = s0 ? s0[q] : s_hat[q];
        cur[q] = v > floor_value ? v : floor_value;
    }
    for (int k = 0; k < n_iter; ++k) {
        for (int j = 0; j < nv; ++j) {
            for (int i = 0; i < nu; ++i) {
                int ip = i + 1 < nu ? i + 1 : nu - 1, im = i > 0 ? i - 1 : 0;       /* [Q28] */
                int jp = j + 1 < nv ? j + 1 : nv - 1, jm = j > 0 ? j - 1 : 0;
                double s = cur[j * nu + i];
                double sum = cur[j * nu + ip] + cur[jp * nu + i] + cur[j * nu + im] + cur[jm * nu + i];
                double v = (1.0 - omega) * s + (omega / 4.0) * (sum - (1.0 / beta) * (1.0 - s_hat[j * nu + i] / s));
                nxt[j * nu + i] = v > floor_value ? v : floor_value;                    /* [Q29] */
            }
        }
        double *t = cur; cur = nxt; nxt = t;
    }
    if (cur != s_out)
        for (int q = 0; q < nu * nv; ++q) s_out[q] = cur[q];
    return 0;
}

int gdrr_oracle_max_materials(void) { return GDRR_ORACLE_MAX_MATERIALS; }
