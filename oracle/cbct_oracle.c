/*
 * cbct_oracle.c -- plain, slow, double-precision CPU oracle for the hot path of
 * Jia et al., "GPU-based Fast Low-dose Cone Beam CT Reconstruction via Total
 * Variation" (arxiv 1001.0599).  Citations are PAPER.md line numbers.
 *
 * THIS IS TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may load it.  It shares no
 * code, header, table or helper with paper_1001_0599_b200/csrc (the CUDA
 * product path) and neither includes the other.
 *
 * Everything is double precision; arrays are row-major
 *   volume      f[(k*ny + j)*nx + i]            (x fastest)
 *   projections p[(a*nv + jv)*nu + iu]          (u fastest, a = view index)
 * OpenMP is used only over independent outputs (rays, voxels, z-slices) or with
 * thread-private accumulators reduced in thread order.
 *
 * Parity status (see tests/test_oracle_*.py):
 *   ray_box_len, forward_brute, forward, back_scatter, back_brute  pinned (P1-P6)
 *   tv_energy, tv_gradient, tv_prox                                 pinned (P7-P10)
 *   fbs                                                             pinned (P11, P12, P14)
 *   restrict / prolong / bin                                        pinned (P13)
 *   back_eq6 (NEXT-1, Eq. 6)                                        pinned (P4, P15, P16)
 *   PARITY UNPINNED: the *choice* of binned detectors on coarse levels (S12) and
 *   the defaults eps_delta, lambda_0 = 1/beta, max_inner (design choices the
 *   paper does not fix; the oracle is their definition).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define BC_ZERO 0
#define BC_REFLECT 1

typedef struct {
    int nx, ny, nz;
    double hx, hy, hz;
    double off[3];          /* volume centre offset from the isocentre, mm */
    int nu, nv;
    double du, dv, offu, offv;
    double sad, sdd;        /* source-axis distance; source-detector distance L0 */
    int n_proj;
    const double *angles;   /* n_proj view angles, radians */
    int bc_xy, bc_z;
} ogeom;

int oracle_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---------------------------------------------------------------------- */
/* Geometry: PAPER.md:L89-L93 (Eq. 1), L104 (Fig. 1 caption), L374 (A2)    */
/* ---------------------------------------------------------------------- */

/* Source position S and the vector D = P(u,v) - S for pixel (iu, iv) of view a.
 * e_n = (cos t, sin t, 0), e_u = (sin t, -cos t, 0), e_v = (0,0,1);
 * S = -SAD e_n;  P = S + L0 e_n + u e_u + v e_v.  At t = 0: D = (L0, -u, v),
 * which is L(u,v) * n of Eq. (A2). */
static void ray_of_pixel(const ogeom *g, int a, int iu, int iv, double S[3], double D[3])
{
    double t = g->angles[a], c = cos(t), s = sin(t);
    double u = (iu - 0.5 * (g->nu - 1)) * g->du + g->offu;
    double v = (iv - 0.5 * (g->nv - 1)) * g->dv + g->offv;
    S[0] = -g->sad * c; S[1] = -g->sad * s; S[2] = 0.0;
    D[0] = g->sdd * c + u * s;
    D[1] = g->sdd * s - u * c;
    D[2] = v;
}

void oracle_ray(const ogeom *g, int a, int iu, int iv, double *S, double *D)
{
    ray_of_pixel(g, a, iu, iv, S, D);
}

/* Where the line source -> point X meets the detector: (u*, v*) and l = |X - S|
 * (Eq. A6, written for a general view angle). */
void oracle_voxel_to_detector(const ogeom *g, int a, const double *X, double *ustar,
                              double *vstar, double *l)
{
    double t = g->angles[a], c = cos(t), s = sin(t);
    double S[3] = { -g->sad * c, -g->sad * s, 0.0 };
    double r[3] = { X[0] - S[0], X[1] - S[1], X[2] - S[2] };
    double rn = r[0] * c + r[1] * s;          /* (X-S).e_n */
    double ru = r[0] * s - r[1] * c;          /* (X-S).e_u */
    double rv = r[2];                         /* (X-S).e_v */
    *ustar = g->sdd * ru / rn;
    *vstar = g->sdd * rv / rn;
    *l = sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2]);
}

/* Length (mm) of { S + t D : 0 <= t <= 1 } inside the box [lo, hi): the slab
 * method.  A direction component below 1e-12 counts as parallel: the slab is
 * then either missed or imposes no limit (half-open test, S3). */
double oracle_ray_box_len(const double *S, const double *D, const double *lo, const double *hi)
{
    double t0 = 0.0, t1 = 1.0;
    for (int a = 0; a < 3; ++a) {
        if (fabs(D[a]) < 1e-12) {
            if (!(lo[a] <= S[a] && S[a] < hi[a])) return 0.0;
        } else {
            double ta = (lo[a] - S[a]) / D[a], tb = (hi[a] - S[a]) / D[a];
            if (ta > tb) { double x = ta; ta = tb; tb = x; }
            if (ta > t0) t0 = ta;
            if (tb < t1) t1 = tb;
        }
    }
    if (t1 <= t0) return 0.0;
    return (t1 - t0) * sqrt(D[0] * D[0] + D[1] * D[1] + D[2] * D[2]);
}

static void voxel_box(const ogeom *g, int i, int j, int k, double lo[3], double hi[3])
{
    double cx = (i - 0.5 * (g->nx - 1)) * g->hx + g->off[0];
    double cy = (j - 0.5 * (g->ny - 1)) * g->hy + g->off[1];
    double cz = (k - 0.5 * (g->nz - 1)) * g->hz + g->off[2];
    lo[0] = cx - 0.5 * g->hx; hi[0] = cx + 0.5 * g->hx;
    lo[1] = cy - 0.5 * g->hy; hi[1] = cy + 0.5 * g->hy;
    lo[2] = cz - 0.5 * g->hz; hi[2] = cz + 0.5 * g->hz;
}

/* ---------------------------------------------------------------------- */
/* O1 forward projector, by definition: (P f)[r] = sum_v a(r,v) f_v with    */
/* a(r,v) = length of ray r inside voxel v (Eq. 1 on a          */
/* piecewise-constant f; "ray-tracing ... such as Siddon's", L187, L243).    */
/* Brute force over every voxel: tiny grids only.                            */
/* ---------------------------------------------------------------------- */
void oracle_forward_brute(const ogeom *g, const double *f, double *p)
{
    long nray = (long)g->n_proj * g->nv * g->nu;
#pragma omp parallel for schedule(static)
    for (long r = 0; r < nray; ++r) {
        int iu = (int)(r % g->nu), iv = (int)((r / g->nu) % g->nv), a = (int)(r / ((long)g->nu * g->nv));
        double S[3], D[3], lo[3], hi[3], acc = 0.0;
        ray_of_pixel(g, a, iu, iv, S, D);
        for (int k = 0; k < g->nz; ++k)
            for (int j = 0; j < g->ny; ++j)
                for (int i = 0; i < g->nx; ++i) {
                    voxel_box(g, i, j, k, lo, hi);
                    acc += oracle_ray_box_len(S, D, lo, hi) * f[((long)k * g->ny + j) * g->nx + i];
                }
        p[r] = acc;
    }
}

/* Exact-transpose back-projector by definition (gather): tiny grids only. */
void oracle_back_brute(const ogeom *g, const double *p, double *b)
{
    long nvox = (long)g->nx * g->ny * g->nz;
#pragma omp parallel for schedule(static)
    for (long v = 0; v < nvox; ++v) {
        int i = (int)(v % g->nx), j = (int)((v / g->nx) % g->ny), k = (int)(v / ((long)g->nx * g->ny));
        double lo[3], hi[3], S[3], D[3], acc = 0.0;
        voxel_box(g, i, j, k, lo, hi);
        for (int a = 0; a < g->n_proj; ++a)
            for (int iv = 0; iv < g->nv; ++iv)
                for (int iu = 0; iu < g->nu; ++iu) {
                    ray_of_pixel(g, a, iu, iv, S, D);
                    acc += oracle_ray_box_len(S, D, lo, hi) * p[((long)a * g->nv + iv) * g->nu + iu];
                }
        b[v] = acc;
    }
}

/* ---------------------------------------------------------------------- */
/* Incremental traversal (Siddon, refs 46-48 of the paper, L187): walk the   */
/* sorted plane crossings of one ray; each consecutive pair of crossing      */
/* parameters bounds one voxel, identified from the segment MIDPOINT.        */
/* visit(ctx, voxel_index, length_mm) is called once per crossed voxel.       */
/* Returns the number of voxels visited with positive length.                */
/* ---------------------------------------------------------------------- */
typedef void (*visit_fn)(void *ctx, long vox, double len);

static long traverse(const ogeom *g, const double S[3], const double D[3], visit_fn visit, void *ctx)
{
    const int n[3] = { g->nx, g->ny, g->nz };
    const double h[3] = { g->hx, g->hy, g->hz };
    double org[3];                       /* coordinate of plane 0 on each axis */
    for (int a = 0; a < 3; ++a) org[a] = g->off[a] - 0.5 * n[a] * h[a];
    double L = sqrt(D[0] * D[0] + D[1] * D[1] + D[2] * D[2]);

    /* parameter range inside the bounding box, clipped to the segment [0,1] */
    double t0 = 0.0, t1 = 1.0;
    for (int a = 0; a < 3; ++a) {
        double lo = org[a], hi = org[a] + n[a] * h[a];
        if (fabs(D[a]) < 1e-12) {
            if (!(lo <= S[a] && S[a] < hi)) return 0;
        } else {
            double ta = (lo - S[a]) / D[a], tb = (hi - S[a]) / D[a];
            if (ta > tb) { double x = ta; ta = tb; tb = x; }
            if (ta > t0) t0 = ta;
            if (tb < t1) t1 = tb;
        }
    }
    if (t1 <= t0) return 0;

    /* next plane index on each axis and its parameter; planes are computed by
     * multiplication (org + p*h), never by running addition */
    int pl[3], step[3];
    double tn[3];
    for (int a = 0; a < 3; ++a) {
        if (fabs(D[a]) < 1e-12) { tn[a] = INFINITY; step[a] = 0; pl[a] = 0; continue; }
        double pos = (S[a] + t0 * D[a] - org[a]) / h[a];   /* plane coordinate at entry */
        if (D[a] > 0) { step[a] = 1;  pl[a] = (int)floor(pos + 1e-9) + 1; }
        else          { step[a] = -1; pl[a] = (int)ceil(pos - 1e-9) - 1; }
        tn[a] = (org[a] + pl[a] * h[a] - S[a]) / D[a];
        /* guard against a crossing at (or rounding below) the entry parameter */
        while (tn[a] <= t0) { pl[a] += step[a]; tn[a] = (org[a] + pl[a] * h[a] - S[a]) / D[a]; }
    }

    long count = 0;
    double tc = t0;
    while (tc < t1) {
        int a = 0;
        if (tn[1] < tn[a]) a = 1;
        if (tn[2] < tn[a]) a = 2;
        double te = tn[a] < t1 ? tn[a] : t1;
        if (te > tc) {
            double tm = 0.5 * (tc + te);
            int idx[3], inside = 1;
            for (int b = 0; b < 3; ++b) {
                idx[b] = (int)floor((S[b] + tm * D[b] - org[b]) / h[b]);
                if (idx[b] < 0 || idx[b] >= n[b]) inside = 0;
            }
            if (inside) {
                visit(ctx, ((long)idx[2] * n[1] + idx[1]) * n[0] + idx[0], (te - tc) * L);
                ++count;
            }
        }
        tc = te;
        if (tn[a] >= t1) break;
        pl[a] += step[a];
        tn[a] = (org[a] + pl[a] * h[a] - S[a]) / D[a];
    }
    return count;
}

typedef struct { const double *f; double acc; } fwd_ctx;
static void fwd_visit(void *c, long vox, double len) { fwd_ctx *x = c; x->acc += len * x->f[vox]; }

/* O1 at real sizes.  Returns S = number of (ray, voxel) pairs with a > 0. */
long oracle_forward(const ogeom *g, const double *f, double *p)
{
    long nray = (long)g->n_proj * g->nv * g->nu, total = 0;
#pragma omp parallel for schedule(dynamic, 256) reduction(+ : total)
    for (long r = 0; r < nray; ++r) {
        int iu = (int)(r % g->nu), iv = (int)((r / g->nu) % g->nv), a = (int)(r / ((long)g->nu * g->nv));
        double S[3], D[3];
        ray_of_pixel(g, a, iu, iv, S, D);
        fwd_ctx c = { f, 0.0 };
        total += traverse(g, S, D, fwd_visit, &c);
        p[r] = c.acc;
    }
    return total;
}

typedef struct { double *b; double w; } bck_ctx;
static void bck_visit(void *c, long vox, double len) { bck_ctx *x = c; x->b[vox] += len * x->w; }

/* O2: (P^T p)_v = sum_r a(r,v) p_r with the SAME a -- scatter along each ray
 * (the operation the paper describes at L187-L191).  Views are dealt to threads;
 * each thread owns a private volume; the privates are added in thread order. */
void oracle_back(const ogeom *g, const double *p, double *b)
{
    long nvox = (long)g->nx * g->ny * g->nz;
    int nt = oracle_threads();
    if (nt > g->n_proj) nt = g->n_proj;
    if (nt < 1) nt = 1;
    double *priv = calloc((size_t)nvox * nt, sizeof(double));
#pragma omp parallel num_threads(nt)
    {
#ifdef _OPENMP
        int me = omp_get_thread_num();
#else
        int me = 0;
#endif
        double *mine = priv + (size_t)me * nvox;
        for (int a = me; a < g->n_proj; a += nt)
            for (int iv = 0; iv < g->nv; ++iv)
                for (int iu = 0; iu < g->nu; ++iu) {
                    double S[3], D[3];
                    ray_of_pixel(g, a, iu, iv, S, D);
                    bck_ctx c = { mine, p[((long)a * g->nv + iv) * g->nu + iu] };
                    if (c.w != 0.0) traverse(g, S, D, bck_visit, &c);
                }
    }
#pragma omp parallel for schedule(static)
    for (long v = 0; v < nvox; ++v) {
        double s = 0.0;
        for (int t = 0; t < nt; ++t) s += priv[(size_t)t * nvox + v];
        b[v] = s;
    }
    free(priv);
}

/* ---------------------------------------------------------------------- */
/* O4: smoothed TV energy, its gradient, and the ROF sub-solver             */
/* (PAPER.md:L100 E1, L151 E3, L155-L161).                                   */
/* Forward differences in physical units.  Neighbour outside the grid:       */
/* value 0 under BC_ZERO, own value under BC_REFLECT (L161).                  */
/* NEXT-1: the paper's own gradient of E2, Eq. (6) -- the continuum adjoint, NOT the
 * transpose of the ray-tracing matrix:
 *     b6(X) = (dV / (du dv)) * sum_theta  L^3(u*,v*) / (L0 l^2(X)) * T^theta(u*, v*)
 * with (u*, v*) and l from Eq. (A6) (oracle_voxel_to_detector), L = sqrt(L0^2 + u*^2 + v*^2) (A2), and
 * T^theta(u*, v*) by BILINEAR interpolation between pixel centres (L199).  The factor dV/(du dv) (voxel volume
 * over pixel area) puts b6 on the scale of P^T T (sum_r a(r,v) = dV L^3/(l^2 du dv L0), survey S1), so that it can
 * replace P^T T in step 1 of Algorithm A1 with the same step size.  Reading S19: a tap outside the detector is 0. */
void oracle_back_eq6(const ogeom *g, const double *T, double *b)
{
    const double scale = g->hx * g->hy * g->hz / (g->du * g->dv);
#pragma omp parallel for schedule(static)
    for (int k = 0; k < g->nz; ++k)
        for (int j = 0; j < g->ny; ++j)
            for (int i = 0; i < g->nx; ++i) {
                double X[3] = { (i - 0.5 * (g->nx - 1)) * g->hx + g->off[0],
                                (j - 0.5 * (g->ny - 1)) * g->hy + g->off[1],
                                (k - 0.5 * (g->nz - 1)) * g->hz + g->off[2] };
                double acc = 0.0;
                for (int a = 0; a < g->n_proj; ++a) {
                    double us, vs, l;
                    oracle_voxel_to_detector(g, a, X, &us, &vs, &l);
                    double L = sqrt(g->sdd * g->sdd + us * us + vs * vs);
                    double fu = (us - g->offu) / g->du + 0.5 * (g->nu - 1);      /* fractional pixel index */
                    double fv = (vs - g->offv) / g->dv + 0.5 * (g->nv - 1);
                    double iu0 = floor(fu), iv0 = floor(fv), tu = fu - iu0, tv = fv - iv0;
                    double val = 0.0;
                    for (int dv = 0; dv < 2; ++dv)
                        for (int du = 0; du < 2; ++du) {
                            long iu = (long)iu0 + du, iv = (long)iv0 + dv;
                            if (iu < 0 || iu >= g->nu || iv < 0 || iv >= g->nv) continue;
                            val += (du ? tu : 1.0 - tu) * (dv ? tv : 1.0 - tv) * T[((long)a * g->nv + iv) * g->nu + iu];
                        }
                    acc += L * L * L / (g->sdd * l * l) * val;
                }
                b[((long)k * g->ny + j) * g->nx + i] = scale * acc;
            }
}

/* ---------------------------------------------------------------------- */
static inline double fwd_diff(double here, double next_or_nan, int at_edge, int bc, double h)
{
    if (!at_edge) return (next_or_nan - here) / h;
    return bc == BC_ZERO ? (0.0 - here) / h : 0.0;
}

static void grad_at(const ogeom *g, const double *f, int i, int j, int k, double gr[3])
{
    long nx = g->nx, ny = g->ny;
    long c = ((long)k * ny + j) * nx + i;
    int ex = (i == g->nx - 1), ey = (j == g->ny - 1), ez = (k == g->nz - 1);
    gr[0] = fwd_diff(f[c], ex ? 0.0 : f[c + 1], ex, g->bc_xy, g->hx);
    gr[1] = fwd_diff(f[c], ey ? 0.0 : f[c + nx], ey, g->bc_xy, g->hy);
    gr[2] = fwd_diff(f[c], ez ? 0.0 : f[c + nx * ny], ez, g->bc_z, g->hz);
}

/* E1^delta[f] = (1/N_vox) sum_v sqrt(|grad f|^2 + delta^2)   (L100; S6) */
double oracle_tv_energy(const ogeom *g, const double *f, double delta)
{
    double s = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : s)
    for (int k = 0; k < g->nz; ++k)
        for (int j = 0; j < g->ny; ++j)
            for (int i = 0; i < g->nx; ++i) {
                double gr[3];
                grad_at(g, f, i, j, k, gr);
                s += sqrt(gr[0] * gr[0] + gr[1] * gr[1] + gr[2] * gr[2] + delta * delta);
            }
    return s / ((double)g->nx * g->ny * g->nz);
}

/* E_ROF[f] = E1^delta[f] + (beta/2) (1/N_vox) sum (f-g)^2   (L151, L155) */
double oracle_rof_energy(const ogeom *g, const double *f, const double *gg, double beta, double delta)
{
    long nvox = (long)g->nx * g->ny * g->nz;
    double q = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : q)
    for (long v = 0; v < nvox; ++v) q += (f[v] - gg[v]) * (f[v] - gg[v]);
    return oracle_tv_energy(g, f, delta) + 0.5 * beta * q / (double)nvox;
}

/* d = N_vox * dE_ROF/df = -div p + beta (f - g),  p = grad f / |grad f|_delta,
 * (div p)_i = (p_i - p_{i-1})/h per axis with p_{-1} := 0: the exact negative
 * transpose of the forward difference under both boundary conditions.
 * gg may be NULL (beta ignored): then d is N_vox * dE1/df alone. */
void oracle_rof_gradient(const ogeom *g, const double *f, const double *gg, double beta,
                         double delta, double *d)
{
    long nx = g->nx, ny = g->ny;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < g->nz; ++k)
        for (int j = 0; j < g->ny; ++j)
            for (int i = 0; i < g->nx; ++i) {
                long c = ((long)k * ny + j) * nx + i;
                double gr[3], q[3], nrm, div;
                grad_at(g, f, i, j, k, gr);
                nrm = sqrt(gr[0] * gr[0] + gr[1] * gr[1] + gr[2] * gr[2] + delta * delta);
                div = gr[0] / nrm / g->hx + gr[1] / nrm / g->hy + gr[2] / nrm / g->hz;
                if (i > 0) {
                    grad_at(g, f, i - 1, j, k, q);
                    div -= q[0] / sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + delta * delta) / g->hx;
                }
                if (j > 0) {
                    grad_at(g, f, i, j - 1, k, q);
                    div -= q[1] / sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + delta * delta) / g->hy;
                }
                if (k > 0) {
                    grad_at(g, f, i, j, k - 1, q);
                    div -= q[2] / sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + delta * delta) / g->hz;
                }
                d[c] = -div + (gg ? beta * (f[c] - gg[c]) : 0.0);
            }
}

typedef struct {
    double eps_delta;
    int max_inner, max_backtracks;
    double armijo_c, shrink_alpha, rel_tol;
} otv_params;

typedef struct { int inner_iters, trials; double e_first, e_last; } otv_report;

/* TV-prox_w(g) ~ argmin_f E1^delta[f] + (1/2w) mean (f-g)^2, w = 1/beta, by the
 * gradient descent with Armijo line search of L155-L159:
 *   start f = g (S8); each inner iteration: E0, d, D = mean d^2; lambda = 1/beta;
 *   trial E_new = E[f - lambda d]; accept if E_new <= E0 - c lambda D (Eq. 5,
 *   S10), else lambda <- alpha lambda (at most max_backtracks shrinks; if none
 *   is accepted stop and keep f); on accept f <- f - lambda d and stop when
 *   |E_new - E0| / E0 < rel_tol (L159) or after max_inner accepted steps.
 * w == 0 means TV off: f = g. */
void oracle_tv_prox(const ogeom *g, const double *gg, double *f, double w,
                    const otv_params *tp, otv_report *rep)
{
    long nvox = (long)g->nx * g->ny * g->nz;
    otv_report r = { 0, 0, 0.0, 0.0 };
    memcpy(f, gg, sizeof(double) * nvox);
    if (w <= 0.0) { if (rep) *rep = r; return; }
    double beta = 1.0 / w;
    double *d = malloc(sizeof(double) * nvox), *ft = malloc(sizeof(double) * nvox);
    double E0 = oracle_rof_energy(g, f, gg, beta, tp->eps_delta);
    r.e_first = r.e_last = E0;
    for (int it = 0; it < tp->max_inner; ++it) {
        oracle_rof_gradient(g, f, gg, beta, tp->eps_delta, d);
        double D = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : D)
        for (long v = 0; v < nvox; ++v) D += d[v] * d[v];
        D /= (double)nvox;
        double lam = 1.0 / beta, Enew = E0;
        int accepted = 0;
        for (int bt = 0; bt <= tp->max_backtracks; ++bt) {
#pragma omp parallel for schedule(static)
            for (long v = 0; v < nvox; ++v) ft[v] = f[v] - lam * d[v];
            Enew = oracle_rof_energy(g, ft, gg, beta, tp->eps_delta);
            ++r.trials;
            if (Enew <= E0 - tp->armijo_c * lam * D) { accepted = 1; break; }
            lam *= tp->shrink_alpha;
        }
        if (!accepted) break;
        memcpy(f, ft, sizeof(double) * nvox);
        ++r.inner_iters;
        double rel = fabs(Enew - E0) / E0;
        E0 = Enew;
        r.e_last = Enew;
        if (rel < tp->rel_tol) break;
    }
    free(d); free(ft);
    if (rep) *rep = r;
}

/* ---------------------------------------------------------------------- */
/* O5: grid transfers (S12, S13)                         */
/* ---------------------------------------------------------------------- */

/* 2x2x2 mean: fine [nz,ny,nx] -> coarse [nz/2,ny/2,nx/2] */
void oracle_restrict(int nx, int ny, int nz, const double *fine, double *coarse)
{
    int cx = nx / 2, cy = ny / 2, cz = nz / 2;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < cz; ++k)
        for (int j = 0; j < cy; ++j)
            for (int i = 0; i < cx; ++i) {
                double s = 0.0;
                for (int c = 0; c < 2; ++c)
                    for (int b = 0; b < 2; ++b)
                        for (int a = 0; a < 2; ++a)
                            s += fine[((long)(2 * k + c) * ny + (2 * j + b)) * nx + (2 * i + a)];
                coarse[((long)k * cy + j) * cx + i] = s / 8.0;
            }
}

/* 2x2 mean over detector pixels of every view: [np,nv,nu] -> [np,nv/2,nu/2] */
void oracle_bin(int nu, int nv, int np, const double *fine, double *coarse)
{
    int cu = nu / 2, cv = nv / 2;
#pragma omp parallel for schedule(static)
    for (int a = 0; a < np; ++a)
        for (int j = 0; j < cv; ++j)
            for (int i = 0; i < cu; ++i) {
                const double *s = fine + ((long)a * nv + 2 * j) * nu + 2 * i;
                coarse[((long)a * cv + j) * cu + i] = 0.25 * (s[0] + s[1] + s[nu] + s[nu + 1]);
            }
}

/* coarse value at index i along an axis of n cells, with the boundary rule */
static inline long clamp_idx(long i, long n) { return i < 0 ? 0 : (i >= n ? n - 1 : i); }

/* "smoothly extend" (L223): cell-centred trilinear interpolation.  Per axis
 * F[2i] = 3/4 C[i] + 1/4 C[i-1],  F[2i+1] = 3/4 C[i] + 1/4 C[i+1]; a missing
 * neighbour is 0 under BC_ZERO and the edge value under BC_REFLECT. */
void oracle_prolong(int cx, int cy, int cz, int bc_xy, int bc_z, const double *coarse, double *fine)
{
    int nx = 2 * cx, ny = 2 * cy, nz = 2 * cz;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                int ci[2] = { i / 2, (i % 2) ? i / 2 + 1 : i / 2 - 1 };
                int cj[2] = { j / 2, (j % 2) ? j / 2 + 1 : j / 2 - 1 };
                int ck[2] = { k / 2, (k % 2) ? k / 2 + 1 : k / 2 - 1 };
                const double wt[2] = { 0.75, 0.25 };
                double s = 0.0;
                for (int c = 0; c < 2; ++c)
                    for (int b = 0; b < 2; ++b)
                        for (int a = 0; a < 2; ++a) {
                            int ox = ci[a] < 0 || ci[a] >= cx, oy = cj[b] < 0 || cj[b] >= cy;
                            int oz = ck[c] < 0 || ck[c] >= cz;
                            if ((bc_xy == BC_ZERO && (ox || oy)) || (bc_z == BC_ZERO && oz)) continue;
                            s += wt[a] * wt[b] * wt[c] *
                                 coarse[(clamp_idx(ck[c], cz) * cy + clamp_idx(cj[b], cy)) * cx +
                                        clamp_idx(ci[a], cx)];
                        }
                fine[((long)k * ny + j) * nx + i] = s;
            }
}

/* ---------------------------------------------------------------------- */
/* O3: forward-backward splitting, Algorithm A1, in the */
/* normalised discrete form of DESIGN.md reading S5:                          */
/*   E1 = mean_v |grad f|_delta, E2 = mean_{view,pixel} (P f - y)^2 (L100),   */
/*   c_norm = 2 N_vox / (N_view N_pix)  so that  N_vox dE2/df = c_norm P^T T, */
/*   step 1 (L147):  g = f - tau c_norm P^T (P f - y),  tau = mu/beta,         */
/*   step 2 (L148):  f = TVprox_w(g),  w = 1/beta = tau * tv_weight,           */
/*   step 3 (L149):  f = max(f, 0).                                            */
/* tau = step / Lhat with Lhat = c_norm max_v [P^T (P 1)]_v  (row-sum bound on */
/* the largest eigenvalue of c_norm P^T P).                                    */
/* ---------------------------------------------------------------------- */
double oracle_step_bound(const ogeom *g)
{
    long nvox = (long)g->nx * g->ny * g->nz, nray = (long)g->n_proj * g->nv * g->nu;
    double *one = malloc(sizeof(double) * nvox), *p1 = malloc(sizeof(double) * nray);
    double *q = malloc(sizeof(double) * nvox), m = 0.0;
    for (long v = 0; v < nvox; ++v) one[v] = 1.0;
    oracle_forward(g, one, p1);
    oracle_back(g, p1, q);
    for (long v = 0; v < nvox; ++v) if (q[v] > m) m = q[v];
    free(one); free(p1); free(q);
    return 2.0 * (double)nvox / (double)nray * m;
}

/* n_iter iterations at one level.  objective[it] = tv_weight * E1^delta(f) +
 * E2(f) for the f that ENTERS iteration it (may be NULL).  Returns tau. */
double oracle_fbs_level(const ogeom *g, const double *y, double *f, double tv_weight, double step,
                        int n_iter, int nonneg, int use_eq6, double conv_tol, const otv_params *tp,
                        double *objective, int *inner_total, int *trials_total, int *iters_done)
{
    long nvox = (long)g->nx * g->ny * g->nz, nray = (long)g->n_proj * g->nv * g->nu;
    double c_norm = 2.0 * (double)nvox / (double)nray;
    double Lhat = oracle_step_bound(g);
    double tau = step / Lhat, w = tau * tv_weight;
    double *T = malloc(sizeof(double) * nray), *b = malloc(sizeof(double) * nvox);
    double *gg = malloc(sizeof(double) * nvox);
    double *prev = malloc(sizeof(double) * nvox);
    int done = 0;
    for (int it = 0; it < n_iter; ++it) {
        memcpy(prev, f, sizeof(double) * nvox);
        oracle_forward(g, f, T);
        double E2 = 0.0;
        for (long r = 0; r < nray; ++r) { T[r] -= y[r]; E2 += T[r] * T[r]; }
        E2 /= (double)nray;
        if (objective) objective[it] = tv_weight * oracle_tv_energy(g, f, tp->eps_delta) + E2;
        if (use_eq6) oracle_back_eq6(g, T, b);      /* the paper's step 1: Eq. 6 in place of P^T T (L195) */
        else oracle_back(g, T, b);
        for (long v = 0; v < nvox; ++v) gg[v] = f[v] - tau * c_norm * b[v];
        otv_report rep;
        oracle_tv_prox(g, gg, f, w, tp, &rep);
        if (inner_total) *inner_total += rep.inner_iters;
        if (trials_total) *trials_total += rep.trials;
        if (nonneg)
            for (long v = 0; v < nvox; ++v) if (f[v] < 0.0) f[v] = 0.0;
        ++done;
        if (conv_tol > 0.0) {   /* "until convergence" (L145, L223; reading S20): relative change of the volume */
            double d2 = 0.0, p2 = 0.0;
            for (long v = 0; v < nvox; ++v) { double d = f[v] - prev[v]; d2 += d * d; p2 += prev[v] * prev[v]; }
            if (p2 > 0.0 && d2 <= conv_tol * conv_tol * p2) break;
        }
    }
    if (iters_done) *iters_done = done;
    free(T); free(b); free(gg); free(prev);
    return tau;
}

/* Multi-grid driver (L215-L223): level l = n_levels-1 (coarsest) ... 0.
 * Level l has volume dims / 2^l at spacing * 2^l and detector dims / 2^l at
 * pitch * 2^l with y binned 2x2 per level (S12).  iters[] runs coarsest ->
 * finest.  f is the finest volume: the initial guess when use_initial (it is
 * restricted to the coarsest level), the result on return.  objective has
 * sum(iters) entries (may be NULL); step_abs[n_levels] receives tau per level
 * in the same coarsest -> finest order (may be NULL). */
void oracle_fbs(const ogeom *g0, const double *y0, double *f, double tv_weight, double step,
                int n_levels, const int *iters, int nonneg, int use_initial, int use_eq6, double conv_tol,
                const otv_params *tp, double *objective, double *step_abs, int *inner_total,
                int *trials_total, int *iters_done)
{
    ogeom *gl = malloc(sizeof(ogeom) * n_levels);
    double **yl = malloc(sizeof(double *) * n_levels);
    gl[0] = *g0;
    yl[0] = (double *)y0;
    for (int l = 1; l < n_levels; ++l) {
        gl[l] = gl[l - 1];
        gl[l].nx /= 2; gl[l].ny /= 2; gl[l].nz /= 2;
        gl[l].hx *= 2; gl[l].hy *= 2; gl[l].hz *= 2;
        gl[l].nu /= 2; gl[l].nv /= 2; gl[l].du *= 2; gl[l].dv *= 2;
        yl[l] = malloc(sizeof(double) * gl[l].n_proj * gl[l].nv * gl[l].nu);
        oracle_bin(gl[l - 1].nu, gl[l - 1].nv, gl[l].n_proj, yl[l - 1], yl[l]);
    }
    /* initial volume on the coarsest level */
    long nv0 = (long)g0->nx * g0->ny * g0->nz;
    double *cur = malloc(sizeof(double) * nv0);
    if (use_initial) memcpy(cur, f, sizeof(double) * nv0); else memset(cur, 0, sizeof(double) * nv0);
    for (int l = 1; l < n_levels; ++l) {
        double *c = malloc(sizeof(double) * (long)gl[l].nx * gl[l].ny * gl[l].nz);
        oracle_restrict(gl[l - 1].nx, gl[l - 1].ny, gl[l - 1].nz, cur, c);
        free(cur); cur = c;
    }
    if (inner_total) *inner_total = 0;
    if (trials_total) *trials_total = 0;
    int done = 0;
    for (int l = n_levels - 1; l >= 0; --l) {
        int n_it = iters[n_levels - 1 - l];
        int ran = 0;
        double tau = oracle_fbs_level(&gl[l], yl[l], cur, tv_weight, step, n_it, nonneg, use_eq6, conv_tol, tp,
                                      objective ? objective + done : NULL, inner_total, trials_total, &ran);
        if (step_abs) step_abs[n_levels - 1 - l] = tau;
        if (iters_done) iters_done[n_levels - 1 - l] = ran;
        done += ran;
        if (l > 0) {
            double *fine = malloc(sizeof(double) * (long)gl[l - 1].nx * gl[l - 1].ny * gl[l - 1].nz);
            oracle_prolong(gl[l].nx, gl[l].ny, gl[l].nz, g0->bc_xy, g0->bc_z, cur, fine);
            free(cur); cur = fine;
        }
    }
    memcpy(f, cur, sizeof(double) * nv0);
    free(cur);
    for (int l = 1; l < n_levels; ++l) free(yl[l]);
    free(yl); free(gl);
}
