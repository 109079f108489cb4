/*
 * ulens_oracle.c -- CPU ORACLE. TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, obviously-correct implementation of what the hot path computes:
 * the finite-source magnification of an N-point-mass lens, written out from its
 * DEFINITION (Eqs. 5-6):
 *
 *     A(w_c, rho, u1) = (1/F0) * Int Int  Theta(rho - |w(z) - w_c|) * I(|w(z)-w_c|/rho) d^2 z
 *     w(z)  = z - sum_i eps_i / conj(z - a_i)                 (Eq. 1)
 *     I(x)  = 1 - u1 * (1 - sqrt(1 - x^2))                    (Eq. A6, un-normalised)
 *     F0    = Int_{disk} I d^2 w = pi rho^2 (1 - u1/3)        (== rho^2 once I0 of P:415 is folded in)
 *
 * evaluated by brute-force inverse ray shooting on ONE origin-aligned uniform
 * Cartesian lattice of pitch h = rho/n_rho (BASELINE.json north_star: "brute-force
 * inverse ray shooting on a dense uniform Cartesian image-plane grid"). The lattice
 * is reached through a quadtree whose nodes are discarded only when a Lipschitz
 * bound of Eq. 1 PROVES that no point of the node maps into the source disk, so
 * every image is covered without any root finder and every cell is visited once.
 *
 * Also: point-source quantities (Eqs. 2-3), the lens polynomial (Eq. 4,
 * P:74-78; coefficients derived in DESIGN.md "oracle polynomial") in __float128,
 * and an extended-precision polish/classification of companion-matrix roots
 * (the eigenvalue route; the eigenvalues themselves come from LAPACK via
 * numpy in oracle/oracle.py).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference leg may call this. It shares no code, header, table or constant
 * with paper_2510_02639_b200/csrc. No fast-math. double unless stated.
 *
 * Pins (tests/test_oracle_pins.py): single-lens closed forms (sqrt(1+4/rho^2) at
 * u=0; Witt & Mao elliptic form elsewhere; limb-darkened annulus decomposition),
 * rho->0 point-source limit, far field 1+2/|w|^4, Vieta sums, lens-equation
 * residuals, image-count and parity-sum rules, symmetries.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <quadmath.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int n;            /* number of point masses, 1..3 */
    double eps[3];    /* mass fractions, sum = 1 */
    double ax[3];     /* lens positions, Einstein radii of the total mass */
    double ay[3];
} orc_lens;

/* ---- geometry (readings G3, G4, G5 of DESIGN.md) ------------------------------------- */

/* Binary: origin = barycentre of M1, M2 (Fig. 3 caption P:203). Reading G4: primary M1
 * (eps1 = 1/(1+q)) at x = -s q/(1+q), secondary M2 (eps2 = q/(1+q)) at x = +s/(1+q). */
int orc_lens_binary(orc_lens *L, double s, double q)
{
    if (!(s > 0) || !(q > 0) || !isfinite(s) || !isfinite(q)) return -1;
    memset(L, 0, sizeof *L);
    L->n = 2;
    L->eps[0] = 1.0 / (1.0 + q);
    L->eps[1] = q / (1.0 + q);
    L->ax[0] = -s * q / (1.0 + q);
    L->ax[1] = s / (1.0 + q);
    return 0;
}

/* Triple (Fig. 3 caption P:203; reading G5): q3 = M3/M1, M3 at polar (r3, psi) from the
 * MIDPOINT of M1-M2; lengths in Einstein radii of the three-body total mass. */
int orc_lens_triple(orc_lens *L, double s, double q, double q3, double r3, double psi)
{
    if (!(s > 0) || !(q > 0) || !(q3 >= 0) || !(r3 > 0)) return -1;
    memset(L, 0, sizeof *L);
    double tot = 1.0 + q + q3;
    L->n = 3;
    L->eps[0] = 1.0 / tot;
    L->eps[1] = q / tot;
    L->eps[2] = q3 / tot;
    L->ax[0] = -s * q / (1.0 + q);
    L->ax[1] = s / (1.0 + q);
    double mid = 0.5 * (L->ax[0] + L->ax[1]);
    L->ax[2] = mid + r3 * cos(psi);
    L->ay[2] = r3 * sin(psi);
    return 0;
}

/* Single lens of unit mass at the origin (closed-form pins). */
int orc_lens_single(orc_lens *L)
{
    memset(L, 0, sizeof *L);
    L->n = 1;
    L->eps[0] = 1.0;
    return 0;
}

/* Trajectory (reading G3): tau = (t-t0)/tE,
 * w_c = (tau cos a - u0 sin a) + i (tau sin a + u0 cos a). */
void orc_trajectory(double t0, double u0, double tE, double alpha, int n, const double *t,
                    double *wx, double *wy)
{
    double ca = cos(alpha), sa = sin(alpha);
    for (int k = 0; k < n; ++k) {
        double tau = (t[k] - t0) / tE;
        wx[k] = tau * ca - u0 * sa;
        wy[k] = tau * sa + u0 * ca;
    }
}

/* ---- Eq. 1, Eqs. 2-3 ------------------------------------------------------------------- */

/* w = z - sum eps_i / conj(z - a_i) = z - sum eps_i (z - a_i)/|z - a_i|^2.   Eq. 1 */
void orc_lens_map(const orc_lens *L, double zx, double zy, double *wx, double *wy)
{
    double sx = 0.0, sy = 0.0;
    for (int i = 0; i < L->n; ++i) {
        double dx = zx - L->ax[i], dy = zy - L->ay[i];
        double r2 = dx * dx + dy * dy;
        sx += L->eps[i] * dx / r2;
        sy += L->eps[i] * dy / r2;
    }
    *wx = zx - sx;
    *wy = zy - sy;
}

/* det J = 1 - | sum eps_i / conj(z - a_i)^2 |^2.   Eq. 3 */
double orc_detJ(const orc_lens *L, double zx, double zy)
{
    double gx = 0.0, gy = 0.0;
    for (int i = 0; i < L->n; ++i) {
        double dx = zx - L->ax[i], dy = -(zy - L->ay[i]);   /* conj(z - a_i) */
        double r2 = dx * dx + dy * dy;
        /* 1/(dx + i dy)^2 = (dx - i dy)^2 / r2^2 */
        double px = (dx * dx - dy * dy) / (r2 * r2);
        double py = (-2.0 * dx * dy) / (r2 * r2);
        gx += L->eps[i] * px;
        gy += L->eps[i] * py;
    }
    return 1.0 - (gx * gx + gy * gy);
}

/* ---- finite-source magnification from the definition (Eqs. 5-6) ----------------- */

typedef struct {
    const orc_lens *L;
    double wcx, wcy, rho, rho2, u1;
    double h;          /* lattice pitch rho / n_rho */
    int ss;            /* sub-samples per side in unresolved cells */
    double x2_smooth;  /* limb-darkened: cells provably inside d^2/rho^2 < x2_smooth use the midpoint rule */
    double flux;       /* accumulated Int chi I d^2z */
    long long n_eval;  /* lens-map evaluations */
} orc_fs;

/* I(x) of Eq. A6 without I0; x2 = d^2/rho^2 in [0,1]. */
static double orc_brightness(double u1, double x2)
{
    if (u1 == 0.0) return 1.0;
    double m = 1.0 - x2;
    if (m < 0.0) m = 0.0;
    return 1.0 - u1 * (1.0 - sqrt(m));
}

/* Distance of w(z) from the source centre, and the Lipschitz constant of Eq. 1 over the disk
 * |z - z0| <= delta:  |w(z)-w(z0)| <= delta * (1 + sum eps_i / D_i^2),  D_i = |z0-a_i| - delta > 0.
 * Returns lip = +inf if the disk touches a lens. */
static void orc_node_bound(orc_fs *S, double zx, double zy, double delta, double *dist, double *lip)
{
    const orc_lens *L = S->L;
    double sx = 0.0, sy = 0.0, lsum = 1.0;
    int touch = 0;
    for (int i = 0; i < L->n; ++i) {
        double dx = zx - L->ax[i], dy = zy - L->ay[i];
        double r2 = dx * dx + dy * dy;
        double D = sqrt(r2) - delta;
        if (D <= 0.0) touch = 1; else lsum += L->eps[i] / (D * D);
        if (r2 > 0.0) { sx += L->eps[i] * dx / r2; sy += L->eps[i] * dy / r2; }
        else touch = 1;
    }
    S->n_eval++;
    double ex = zx - sx - S->wcx, ey = zy - sy - S->wcy;
    *dist = sqrt(ex * ex + ey * ey);
    *lip = touch ? INFINITY : lsum;
}

/* One lattice cell [ix h,(ix+1)h) x [iy h,(iy+1)h). */
static void orc_leaf(orc_fs *S, int64_t ix, int64_t iy)
{
    double h = S->h;
    double cx = ((double)ix + 0.5) * h, cy = ((double)iy + 0.5) * h;
    double delta = h * M_SQRT1_2, dist, lip;
    orc_node_bound(S, cx, cy, delta, &dist, &lip);
    double reach = delta * lip;                 /* may be inf */
    if (dist - reach > S->rho) return;          /* provably outside */
    double rin = (S->u1 == 0.0) ? S->rho : S->rho * sqrt(S->x2_smooth);
    if (dist + reach <= rin) {                  /* provably inside (and brightness smooth): midpoint */
        S->flux += orc_brightness(S->u1, dist * dist / S->rho2) * h * h;
        return;
    }
    /* unresolved: ss x ss sub-samples, each added iff inside, brightness at the sub-sample */
    int ss = S->ss;
    double hs = h / ss, acc = 0.0;
    const orc_lens *L = S->L;
    for (int j = 0; j < ss; ++j) {
        double zy = (double)iy * h + (j + 0.5) * hs;
        for (int i = 0; i < ss; ++i) {
            double zx = (double)ix * h + (i + 0.5) * hs;
            double sx = 0.0, sy = 0.0;
            int bad = 0;
            for (int k = 0; k < L->n; ++k) {
                double dx = zx - L->ax[k], dy = zy - L->ay[k];
                double r2 = dx * dx + dy * dy;
                if (r2 > 0.0) { sx += L->eps[k] * dx / r2; sy += L->eps[k] * dy / r2; }
                else bad = 1;                    /* a ray exactly on a lens maps to infinity: outside */
            }
            if (bad) continue;
            double ex = zx - sx - S->wcx, ey = zy - sy - S->wcy;
            double d2 = ex * ex + ey * ey;
            if (d2 < S->rho2) acc += orc_brightness(S->u1, d2 / S->rho2);
        }
    }
    S->n_eval += (long long)ss * ss;
    S->flux += acc * hs * hs;
}

/* Quadtree node: cells [ix, ix+size) x [iy, iy+size), size a power of two. */
static void orc_descend(orc_fs *S, int64_t ix, int64_t iy, int64_t size)
{
    if (size == 1) { orc_leaf(S, ix, iy); return; }
    double h = S->h;
    double cx = ((double)ix + 0.5 * (double)size) * h, cy = ((double)iy + 0.5 * (double)size) * h;
    double delta = (double)size * h * M_SQRT1_2, dist, lip;
    orc_node_bound(S, cx, cy, delta, &dist, &lip);
    if (dist - delta * lip > S->rho) return;     /* Lipschitz bound: no point of the node is inside */
    int64_t hs = size / 2;
    orc_descend(S, ix, iy, hs);
    orc_descend(S, ix + hs, iy, hs);
    orc_descend(S, ix, iy + hs, hs);
    orc_descend(S, ix + hs, iy + hs, hs);
}

/* A at lattice pitch rho/n_rho. Returns 0, or -1 on a bad argument.
 * Outside |Re z|,|Im z| <= R = 2 + |w_c| + rho + max|a_i| no point can map into the source:
 * there |z - a_i| > 2 + |w_c| + rho  so  |w - z| <= sum eps_i/|z-a_i| < 1/2  while  |z - w_c| > 2 + rho. */
int orc_mag_fs_pitch(const orc_lens *L, double wcx, double wcy, double rho, double u1, double h, int ss,
                     double *A_out, long long *n_eval_out);

int orc_mag_fs(const orc_lens *L, double wcx, double wcy, double rho, double u1, int n_rho, int ss,
               double *A_out, long long *n_eval_out)
{
    if (!(rho > 0) || n_rho < 1) return -1;
    return orc_mag_fs_pitch(L, wcx, wcy, rho, u1, rho / n_rho, ss, A_out, n_eval_out);
}

/* The same with the lattice pitch h given explicitly, so that a finite-difference derivative with respect
 * to rho (or anything else) can hold the lattice fixed (DESIGN.md 7.2 "derivative reference"). */
int orc_mag_fs_pitch(const orc_lens *L, double wcx, double wcy, double rho, double u1, double h, int ss,
                     double *A_out, long long *n_eval_out)
{
    if (!L || L->n < 1 || L->n > 3 || !(rho > 0) || !(u1 >= 0 && u1 <= 1) || !(h > 0) || ss < 1) return -1;
    orc_fs S;
    S.L = L; S.wcx = wcx; S.wcy = wcy; S.rho = rho; S.rho2 = rho * rho; S.u1 = u1;
    S.h = h; S.ss = ss; S.x2_smooth = 0.81; S.flux = 0.0; S.n_eval = 0;
    double amax = 0.0;
    for (int i = 0; i < L->n; ++i) { double a = hypot(L->ax[i], L->ay[i]); if (a > amax) amax = a; }
    double R = 2.0 + hypot(wcx, wcy) + rho + amax;
    int64_t half = 1;
    while ((double)half * S.h < R) half *= 2;
    orc_descend(&S, -half, -half, half);
    orc_descend(&S, 0, -half, half);
    orc_descend(&S, -half, 0, half);
    orc_descend(&S, 0, 0, half);
    double F0 = M_PI * rho * rho * (1.0 - u1 / 3.0);
    *A_out = S.flux / F0;
    if (n_eval_out) *n_eval_out = S.n_eval;
    return 0;
}

/* Batch over points (OpenMP over points; each point is the serial routine above).
 * lens_idx[k] selects lenses[lens_idx[k]]; rho, u1 per point. Two pitches are run: n_rho and 2 n_rho
 * (self-error): A_coarse, A_fine. */
int orc_mag_fs_batch(const orc_lens *lenses, const int *lens_idx, int n_pts, const double *wcx,
                     const double *wcy, const double *rho, const double *u1, int n_rho, int ss,
                     int n_threads, double *A_coarse, double *A_fine, long long *n_eval)
{
    int bad = 0;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel for schedule(dynamic, 1) reduction(| : bad)
    for (int k = 0; k < n_pts; ++k) {
        long long e1 = 0, e2 = 0;
        const orc_lens *L = &lenses[lens_idx ? lens_idx[k] : 0];
        int r1 = orc_mag_fs(L, wcx[k], wcy[k], rho[k], u1[k], n_rho, ss, &A_coarse[k], &e1);
        int r2 = orc_mag_fs(L, wcx[k], wcy[k], rho[k], u1[k], 2 * n_rho, ss, &A_fine[k], &e2);
        if (n_eval) n_eval[k] = e1 + e2;
        if (r1 || r2) bad |= 1;
    }
    return bad ? -1 : 0;
}

/* Batch at one explicit pitch per point and one lens per point (finite-difference stencils: every
 * perturbed evaluation has its own lens, source and radius but the unperturbed point's lattice). */
int orc_mag_fs_pitch_batch(const orc_lens *lenses, int n_pts, const double *wcx, const double *wcy,
                           const double *rho, const double *u1, const double *h, int ss, int n_threads,
                           double *A, long long *n_eval)
{
    int bad = 0;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel for schedule(dynamic, 1) reduction(| : bad)
    for (int k = 0; k < n_pts; ++k) {
        long long e = 0;
        if (orc_mag_fs_pitch(&lenses[k], wcx[k], wcy[k], rho[k], u1[k], h[k], ss, &A[k], &e)) bad |= 1;
        if (n_eval) n_eval[k] = e;
    }
    return bad ? -1 : 0;
}

int orc_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---- lens polynomial (Eq. 4) in __float128 ------------------------------------------
 * The paper does not print b_l (reading G1). Derivation: conjugate
 * Eq. 1:  conj(z) = conj(w) + G(z)/Q(z),   Q(z) = prod_k (z - a_k),  G(z) = sum_k eps_k prod_{m!=k}(z - a_m).
 * Then conj(z) - conj(a_i) = H_i(z)/Q(z),  H_i(z) = (conj(w) - conj(a_i)) Q(z) + G(z), and Eq. 1 becomes
 *     P(z) = (z - w) prod_i H_i(z)  -  Q(z) sum_i eps_i prod_{j!=i} H_j(z) = 0,   degree N^2 + 1
 * (2, 5, 10 for N = 1, 2, 3; the paper's 5(N-1) agrees for N = 2, 3). */

#define ORC_MAXDEG 10
typedef __complex128 qc;
typedef struct { int deg; qc c[ORC_MAXDEG + 2]; } qpoly;     /* c[l] multiplies z^l */

static qpoly qp_const(qc v) { qpoly p; memset(&p, 0, sizeof p); p.deg = 0; p.c[0] = v; return p; }
static qpoly qp_linear(qc root) { qpoly p; memset(&p, 0, sizeof p); p.deg = 1; p.c[0] = -root; p.c[1] = 1; return p; }
static qpoly qp_mul(const qpoly *a, const qpoly *b)
{
    qpoly p; memset(&p, 0, sizeof p);
    p.deg = a->deg + b->deg;
    for (int i = 0; i <= a->deg; ++i)
        for (int j = 0; j <= b->deg; ++j) p.c[i + j] += a->c[i] * b->c[j];
    return p;
}
static qpoly qp_axpy(qc alpha, const qpoly *x, const qpoly *y)   /* alpha x + y */
{
    qpoly p; memset(&p, 0, sizeof p);
    p.deg = x->deg > y->deg ? x->deg : y->deg;
    for (int i = 0; i <= x->deg; ++i) p.c[i] += alpha * x->c[i];
    for (int i = 0; i <= y->deg; ++i) p.c[i] += y->c[i];
    return p;
}

static void orc_build_poly(const orc_lens *L, double wx, double wy, qpoly *P)
{
    int n = L->n;
    qc a[3], w, wbar;
    __real__ w = wx; __imag__ w = wy;
    wbar = conjq(w);
    for (int i = 0; i < n; ++i) { __real__ a[i] = L->ax[i]; __imag__ a[i] = L->ay[i]; }
    qpoly Q = qp_const(1), G = qp_const(0);
    for (int k = 0; k < n; ++k) { qpoly f = qp_linear(a[k]); Q = qp_mul(&Q, &f); }
    for (int k = 0; k < n; ++k) {
        qpoly t = qp_const((__float128)L->eps[k]);
        for (int m = 0; m < n; ++m) if (m != k) { qpoly f = qp_linear(a[m]); t = qp_mul(&t, &f); }
        G = qp_axpy(1, &t, &G);
    }
    qpoly H[3];
    for (int i = 0; i < n; ++i) H[i] = qp_axpy(wbar - conjq(a[i]), &Q, &G);
    qpoly first = qp_linear(w);
    for (int i = 0; i < n; ++i) first = qp_mul(&first, &H[i]);
    qpoly second = qp_const(0);
    for (int i = 0; i < n; ++i) {
        qpoly t = qp_const((__float128)L->eps[i]);
        for (int j = 0; j < n; ++j) if (j != i) t = qp_mul(&t, &H[j]);
        second = qp_axpy(1, &t, &second);
    }
    second = qp_mul(&Q, &second);
    *P = qp_axpy(-1, &second, &first);
    P->deg = n * n + 1;
}

/* Coefficients rounded to double (starting values for the companion matrix in oracle.py). */
int orc_poly_coeffs(const orc_lens *L, double wx, double wy, double *b_re, double *b_im)
{
    if (!L || L->n < 1 || L->n > 3) return -1;
    qpoly P; orc_build_poly(L, wx, wy, &P);
    for (int l = 0; l <= P.deg; ++l) { b_re[l] = (double)crealq(P.c[l]); b_im[l] = (double)cimagq(P.c[l]); }
    return P.deg;
}

static void qp_eval(const qpoly *P, qc z, qc *p, qc *dp)
{
    qc v = P->c[P->deg], d = 0;
    for (int l = P->deg - 1; l >= 0; --l) { d = d * z + v; v = v * z + P->c[l]; }
    *p = v; *dp = d;
}

/* Extended-precision refinement of ALL roots from double starting values (companion-matrix
 * eigenvalues): simultaneous Newton steps with the Aberth repulsion term so that two starts
 * cannot fall onto one root, in __float128, until every step is < 1e-28 max(1,|z|).
 * Then classification on Eq. 1 ("substituting it back"): image iff the residual of Eq. 1 is
 * < 1e-18 (spurious roots have O(1e-3..1) residuals except within ~1e-30 of a caustic).
 * Outputs per root: position (double), is_image, Eq.-1 residual, det J (Eq. 3), and the condition
 * estimate kappa_k = sum_l |b_l||z_k|^l / (|z_k| |P'(z_k)|)  (relative root perturbation per
 * relative coefficient perturbation). Returns the degree. */
int orc_roots_refine(const orc_lens *L, double wx, double wy, double *z_re, double *z_im,
                     int *is_image, double *resid, double *detJ, double *kappa)
{
    if (!L || L->n < 1 || L->n > 3) return -1;
    qpoly P; orc_build_poly(L, wx, wy, &P);
    int n = P.deg;
    qc z[ORC_MAXDEG];
    for (int k = 0; k < n; ++k) { __real__ z[k] = z_re[k]; __imag__ z[k] = z_im[k]; }
    for (int it = 0; it < 200; ++it) {
        __float128 worst = 0;
        for (int k = 0; k < n; ++k) {
            qc p, dp; qp_eval(&P, z[k], &p, &dp);
            if (cabsq(p) == 0) continue;
            qc newton = p / dp, rep = 0;
            for (int j = 0; j < n; ++j) if (j != k) rep += 1 / (z[k] - z[j]);
            qc step = newton / (1 - newton * rep);
            z[k] -= step;                              /* Gauss-Seidel order: uses updated z[j<k] */
            __float128 rel = cabsq(step) / (cabsq(z[k]) > 1 ? cabsq(z[k]) : 1);
            if (rel > worst) worst = rel;
        }
        if (worst < 1e-28Q) break;
    }
    qc w; __real__ w = wx; __imag__ w = wy;
    for (int k = 0; k < n; ++k) {
        qc s = 0, g = 0;
        for (int i = 0; i < L->n; ++i) {
            qc a; __real__ a = L->ax[i]; __imag__ a = L->ay[i];
            qc dzb = conjq(z[k] - a);
            s += (__float128)L->eps[i] / dzb;
            g += (__float128)L->eps[i] / (dzb * dzb);
        }
        __float128 r = cabsq(z[k] - s - w);
        z_re[k] = (double)crealq(z[k]); z_im[k] = (double)cimagq(z[k]);
        resid[k] = (double)r;
        is_image[k] = r < 1e-18Q;
        detJ[k] = (double)(1 - crealq(g * conjq(g)));
        qc p, dp; qp_eval(&P, z[k], &p, &dp);
        __float128 zz = cabsq(z[k]), pw = 1, sum = 0;
        for (int l = 0; l <= n; ++l) { sum += cabsq(P.c[l]) * pw; pw *= zz; }
        kappa[k] = (double)(sum / ((zz > 1e-300Q ? zz : 1e-300Q) * cabsq(dp)));
    }
    return n;
}
