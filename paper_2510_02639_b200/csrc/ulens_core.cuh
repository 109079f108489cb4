// ulens_core.cuh -- per-thread arithmetic of the ICRS hot path (device code; also compiles as plain
// C++ so that host logic tests can include it -- the product has no CPU path, see ulens_api.cu).
//
// Citations "P:<line>" are to /root/reference/PAPER.md. Readings "G<n>" are listed in DESIGN.md.
//
//   lens map, Jacobian                      Eq. 1-3
//   lens polynomial (own derivation, G1)    Eq. 4
//   Ehrlich-Aberth iteration (G6)           Eq. 7
//   root validation + polish on Eq. 1 (G7)
//   ring quadrature along theta (G9-G13)    App. A
//
// This file shares nothing with oracle/ (different polynomial construction, different integration
// rule, different code).
#pragma once
#include <math.h>
#include <stdint.h>

#if defined(__CUDACC__)
#define UL_HD __host__ __device__ __forceinline__
#define UL_HDN __host__ __device__
#define UL_HDNI __host__ __device__ __noinline__
#else
#define UL_HD inline
#define UL_HDN inline
#define UL_HDNI inline
#endif

namespace ulens {

// ------------------------------------------------------------------------------------------------
// data shared by the kernels
// ------------------------------------------------------------------------------------------------

struct Lens {            // same layout as ulens_lens (include/ulens.h)
    int n;
    double eps[3], ax[3], ay[3];
};

// Polynomial basis of one lens: T_k(z) = Q(z)^k G(z)^(N-k), k = 0..N, where
//   Q(z) = prod_i (z - a_i),  G(z) = sum_i eps_i prod_{m != i} (z - a_m)      (conj of Eq. 1: conj z = conj w + G/Q).
// With c_i = conj(w) - conj(a_i):  conj(z) - conj(a_i) = (c_i Q + G)/Q, so Eq. 1 times prod_i (c_i Q + G) is
//   P(z) = (z - w) sum_{k=0..N} e_k(c) T_k(z)  -  sum_{k=0..N-1} f_k(c) T_{k+1}(z),      degree N^2 + 1,
// e_k = k-th elementary symmetric polynomial of c_1..c_N, f_k = sum_i eps_i e_k(c without c_i).
// T_k has degree N(N-1) + k <= N^2 (<= 9): 10 coefficients each, filled on the host once per lens.
struct LensPoly {
    double tr[4][10], ti[4][10];
};

struct PointCfg {        // per (lens, source) configuration
    Lens lens;
    double rho, u1;
};

// sector ("patch") descriptor, written by k_regions and read by k_shoot
struct Patch {
    double r0, dr;       // ring i at r0 + (i + 1/2) dr, i = 0..n_r-1   (G11: midpoint nodes, empty end rings)
    double th0, dth;     // ray j at th0 + (j + 1/2) dth, j = 0..n_th-1
    int n_r, n_th;
    int point;           // global point index
    int unit0;           // first 32-ring work unit of this patch in the unit arrays
    int flags;           // UL_PATCH_*: periodic in theta (full ring); scan lines are radial (lanes = theta); sin-spaced rings
    int n_units;         // 32-line work units
    double kap_lo, kap_hi; // across-line margins as fractions of the image extent (the dual variant moves them with it)
};

#define UL_PATCH_PERIODIC 1
#define UL_PATCH_SCAN_R 2
#define UL_PATCH_SINR 4      // ring i of n_r at r_c + h sin(phi_i), phi_i = -pi/2 + (i + 1/2) pi / n_r, weight h cos(phi_i) pi / n_r

// status bits (mirror include/ulens.h)
#define UL_ST_EA_NOCONV  0x0001u
#define UL_ST_IMG_PARITY 0x0002u
#define UL_ST_PATCH_CAP  0x0004u
#define UL_ST_RES_CAP    0x0008u
#define UL_ST_CLIPPED    0x0010u
#define UL_ST_UNIT_OVF   0x0020u
#define UL_ST_ERR_HIGH   0x0040u
#define UL_ST_NO_IMAGE   0x0080u
#define UL_ST_POINT_SRC  0x1000u
#define UL_ST_RETRIED    0x2000u

#define UL_PI 3.14159265358979323846
// the 8 directions k pi/4 (seeds on a light lens's Einstein ring)
#define UL_RING8_X(k) ((k) == 0 ? 1.0 : (k) == 4 ? -1.0 : ((k) == 2 || (k) == 6) ? 0.0 : ((k) == 1 || (k) == 7) ? 0.70710678118654752 : -0.70710678118654752)
#define UL_RING8_Y(k) ((k) == 2 ? 1.0 : (k) == 6 ? -1.0 : ((k) == 0 || (k) == 4) ? 0.0 : ((k) == 1 || (k) == 3) ? 0.70710678118654752 : -0.70710678118654752)
#define UL_BIG 1e100

UL_HD double ul_min(double a, double b) { return a < b ? a : b; }
UL_HD double ul_rsqrt(double x)
{
#ifdef __CUDA_ARCH__
    return rsqrt(x);
#else
    return 1.0 / sqrt(x);
#endif
}
UL_HD double ul_max(double a, double b) { return a > b ? a : b; }

// ------------------------------------------------------------------------------------------------
// Eq. 1-3: lens map residual and its conj-derivative g = sum eps_i / conj(z - a_i)^2
// ------------------------------------------------------------------------------------------------

// f = z - sum eps_i/conj(z - a_i) - w ;  g = d w / d conj(z) = sum eps_i / conj(z - a_i)^2 ;  dmin2 = min |z - a_i|^2
template <int N>
UL_HD void lens_resid(const Lens& L, double zx, double zy, double wx, double wy,
                      double& fx, double& fy, double& gx, double& gy, double& dmin2)
{
    double sx = 0.0, sy = 0.0;
    gx = 0.0; gy = 0.0; dmin2 = 1e300;
#pragma unroll
    for (int i = 0; i < N; ++i) {
        double dx = zx - L.ax[i], dy = zy - L.ay[i];
        double r2 = dx * dx + dy * dy;
        double inv = 1.0 / r2;
        dmin2 = ul_min(dmin2, r2);
        // eps/conj(d) = eps d/|d|^2
        sx += L.eps[i] * dx * inv;
        sy += L.eps[i] * dy * inv;
        // eps/conj(d)^2 = eps d^2/|d|^4
        double inv2 = inv * inv;
        gx += L.eps[i] * (dx * dx - dy * dy) * inv2;
        gy += L.eps[i] * (2.0 * dx * dy) * inv2;
    }
    fx = zx - sx - wx;
    fy = zy - sy - wy;
}

// Damped Newton on Eq. 1 itself (G7 "polish"): delta w = dz + g conj(dz)  =>  dz = (b - g conj(b))/(1 - |g|^2), b = -f.
// The step is limited to half the distance to the nearest lens. Returns true when the final residual
// (or the last Newton step) is below tol * max(1, |z|); z is updated in place; detJ = 1 - |g|^2 (Eq. 3).
template <int N>
UL_HD bool polish_image(const Lens& L, double wx, double wy, double& zx, double& zy, int max_it,
                        double tol, double& detJ, double& resid, double& gx, double& gy, double reject_frac2 = 0.0,
                        bool refine = true)
{
    double fx, fy, dmin2;
    bool ok = false;
    double r2 = 1e300;
    detJ = 0.0;
    const double tol2 = tol * tol;
    for (int it = 0; it <= max_it; ++it) {
        lens_resid<N>(L, zx, zy, wx, wy, fx, fy, gx, gy, dmin2);
        detJ = 1.0 - (gx * gx + gy * gy);
        r2 = fx * fx + fy * fy;
        const double scale2 = ul_max(1.0, zx * zx + zy * zy);       // compared squared: no square roots in the loop
        if (!(r2 == r2)) { resid = r2; return false; }
        // refine: keep iterating down to the rounding floor (step a2: images to 1e-15); the limb solves of the
        // region builder stop as soon as the residual is below tol
        if (r2 <= tol2 * scale2) { ok = true; if (!refine || r2 <= 1.6e-31 * scale2) break; }
        if (it == max_it) break;
        if (fabs(detJ) < 1e-14) break;
        double bx = -fx, by = -fy;
        // g conj(b)
        double qx = gx * bx + gy * by, qy = gy * bx - gx * by;
        const double idet = 1.0 / detJ;
        double sx = (bx - qx) * idet, sy = (by - qy) * idet;
        double s2 = sx * sx + sy * sy;
        // region builder only: a start whose FIRST Newton step already exceeds sqrt(reject_frac2) of its distance
        // to the nearest lens is a spurious root of the polynomial, not an image known to ~1e-7
        if (it == 0 && reject_frac2 > 0.0 && s2 > reject_frac2 * dmin2) { resid = sqrt(r2); return false; }
        double lim2 = 0.25 * dmin2;
        if (s2 > lim2) { double k = sqrt(lim2 / s2); sx *= k; sy *= k; }
        zx += sx; zy += sy;
        // converged in POSITION: next to a light lens |g| ~ 1e5 and the rounding floor of the residual
        // (~1e-16 |a| |g|) is far above tol although the image is located to ~1e-16
        if (s2 <= tol2 * scale2 && r2 <= 1e-12 * scale2) { ok = true; break; }
    }
    resid = sqrt(r2);
    return ok;
}

// ------------------------------------------------------------------------------------------------
// Eq. 4: coefficients b_0..b_DEG of the lens polynomial for source position w
// ------------------------------------------------------------------------------------------------

// e_0..e_N = elementary symmetric polynomials of c_i = conj(w) - conj(a_i), f_k = sum_i eps_i e_k(c without c_i)
template <int N>
UL_HD void poly_sym(const Lens& L, double wx, double wy, double* ex, double* ey, double* fx, double* fy)
{
    // c_i = conj(w) - conj(a_i)
    double cx[N], cy[N];
#pragma unroll
    for (int i = 0; i < N; ++i) { cx[i] = wx - L.ax[i]; cy[i] = -(wy - L.ay[i]); }
    // a source centre exactly on a projected lens position makes the leading coefficient vanish
    // (prod c_i): nudge that c_i (images move by ~1e-13, far below every tolerance here)
#pragma unroll
    for (int i = 0; i < N; ++i)
        if (cx[i] * cx[i] + cy[i] * cy[i] < 1e-26) cx[i] += 1e-13;
    ex[0] = 1.0; ey[0] = 0.0;
#pragma unroll
    for (int k = 1; k <= N; ++k) { ex[k] = 0.0; ey[k] = 0.0; }
#pragma unroll
    for (int i = 0; i < N; ++i) {
#pragma unroll
        for (int k = N; k >= 1; --k) {
            if (k <= i + 1) {
                double tx = ex[k - 1] * cx[i] - ey[k - 1] * cy[i];
                double ty = ex[k - 1] * cy[i] + ey[k - 1] * cx[i];
                ex[k] += tx; ey[k] += ty;
            }
        }
    }
    if constexpr (N == 1) {
        fx[0] = L.eps[0]; fy[0] = 0.0;
    } else if constexpr (N == 2) {
        fx[0] = L.eps[0] + L.eps[1]; fy[0] = 0.0;
        fx[1] = L.eps[0] * cx[1] + L.eps[1] * cx[0];
        fy[1] = L.eps[0] * cy[1] + L.eps[1] * cy[0];
    } else {
        fx[0] = L.eps[0] + L.eps[1] + L.eps[2]; fy[0] = 0.0;
        fx[1] = L.eps[0] * (cx[1] + cx[2]) + L.eps[1] * (cx[0] + cx[2]) + L.eps[2] * (cx[0] + cx[1]);
        fy[1] = L.eps[0] * (cy[1] + cy[2]) + L.eps[1] * (cy[0] + cy[2]) + L.eps[2] * (cy[0] + cy[1]);
        double p12x = cx[1] * cx[2] - cy[1] * cy[2], p12y = cx[1] * cy[2] + cy[1] * cx[2];
        double p02x = cx[0] * cx[2] - cy[0] * cy[2], p02y = cx[0] * cy[2] + cy[0] * cx[2];
        double p01x = cx[0] * cx[1] - cy[0] * cy[1], p01y = cx[0] * cy[1] + cy[0] * cx[1];
        fx[2] = L.eps[0] * p12x + L.eps[1] * p02x + L.eps[2] * p01x;
        fy[2] = L.eps[0] * p12y + L.eps[1] * p02y + L.eps[2] * p01y;
    }
}

template <int N>
UL_HD void poly_coeffs(const Lens& L, const LensPoly& T, double wx, double wy, double* br, double* bi)
{
    constexpr int DEG = N * N + 1;
    double ex[N + 1], ey[N + 1], fx[N], fy[N];
    poly_sym<N>(L, wx, wy, ex, ey, fx, fy);
    // S(z) = sum_k e_k T_k(z)   (degree N^2),  R(z) = sum_k f_k T_{k+1}(z)   (degree N^2)
    // P = (z - w) S - R :  b_l = S_{l-1} - w S_l - R_l
    double sr[DEG], si[DEG];          // S_0..S_{N^2}  (DEG = N^2+1 entries)
#pragma unroll
    for (int l = 0; l < DEG; ++l) {
        double ar = 0.0, ai = 0.0, rr = 0.0, ri = 0.0;
#pragma unroll
        for (int k = 0; k <= N; ++k) {
            double tr = T.tr[k][l], ti = T.ti[k][l];
            ar += ex[k] * tr - ey[k] * ti;
            ai += ex[k] * ti + ey[k] * tr;
            if (k >= 1) {
                rr += fx[k - 1] * tr - fy[k - 1] * ti;
                ri += fx[k - 1] * ti + fy[k - 1] * tr;
            }
        }
        sr[l] = ar; si[l] = ai;
        br[l] = -(wx * ar - wy * ai) - rr;
        bi[l] = -(wx * ai + wy * ar) - ri;
    }
    br[DEG] = 0.0; bi[DEG] = 0.0;
#pragma unroll
    for (int l = 1; l <= DEG; ++l) { br[l] += sr[l - 1]; bi[l] += si[l - 1]; }
}

// ------------------------------------------------------------------------------------------------
// Eq. 7: Ehrlich-Aberth simultaneous iteration (Newton form, G6), Gauss-Seidel order
// ------------------------------------------------------------------------------------------------

template <int DEG>
UL_HD void horner2(const double* br, const double* bi, double x, double y,
                   double& pr, double& pi, double& dr, double& di)
{
    pr = br[DEG]; pi = bi[DEG]; dr = 0.0; di = 0.0;
#pragma unroll
    for (int l = DEG - 1; l >= 0; --l) {
        double t = dr * x - di * y + pr;
        di = dr * y + di * x + pi;
        dr = t;
        t = pr * x - pi * y + br[l];
        pi = pr * y + pi * x + bi[l];
        pr = t;
    }
}

// Initial guesses on the Cauchy-bound circle (G6: radius 1 + max_{l<n} |b_l/b_n|, phase offset 0.4 rad).
template <int DEG>
UL_HD void ea_init(const double* br, const double* bi, double* zr, double* zi)
{
    double ln2 = br[DEG] * br[DEG] + bi[DEG] * bi[DEG];
    double m2 = 0.0;
#pragma unroll
    for (int l = 0; l < DEG; ++l) m2 = ul_max(m2, br[l] * br[l] + bi[l] * bi[l]);
    double R = 1.0 + sqrt(m2 / ln2);
    // the lens-polynomial roots all lie within a few Einstein radii; a huge Cauchy bound (tiny leading
    // coefficient) only slows the first iterations down, so start no further out than 8
    R = ul_min(R, 8.0);
    // centroid of the roots = -b_{n-1}/(n b_n)
    double qx = (br[DEG - 1] * br[DEG] + bi[DEG - 1] * bi[DEG]) / ln2;
    double qy = (bi[DEG - 1] * br[DEG] - br[DEG - 1] * bi[DEG]) / ln2;
    double cx = -qx / DEG, cy = -qy / DEG;
    if (!(cx * cx + cy * cy < 16.0)) { cx = 0.0; cy = 0.0; }
#pragma unroll
    for (int k = 0; k < DEG; ++k) {
        double ph = 0.4 + 2.0 * UL_PI * k / DEG;
        zr[k] = cx + R * cos(ph);
        zi[k] = cy + R * sin(ph);
    }
}

// Iterate until every root is settled, or max_it. A root is settled (frozen, but still repelling the others)
// once its relative step is < sqrt(tol2), or its step is below 1e-3 and no longer shrinking by 1.41x per
// iteration: the evaluation-noise floor, which for the spurious-root clusters next to a light lens is as
// high as 1e-5 relative (degree 10). Near-double roots converge linearly at rate 1/2 and are NOT stopped by
// the second rule. The images are polished on Eq. 1 afterwards, so EA only has to reach Newton's basin.
// Returns the iterations used (max_it+1 if the cap was hit with a root still moving).
template <int DEG>
UL_HD int ea_iterate(const double* br, const double* bi, double* zr, double* zi, int max_it, double tol2 = 1e-28)
{
    double prev[DEG];
#pragma unroll
    for (int k = 0; k < DEG; ++k) prev[k] = 1e300;
    unsigned done = 0;
    const unsigned all = (1u << DEG) - 1u;
    for (int it = 1; it <= max_it; ++it) {
        bool bad = false;
#pragma unroll
        for (int k = 0; k < DEG; ++k) {
            if (done & (1u << k)) continue;
            double pr, pi, dr, di;
            horner2<DEG>(br, bi, zr[k], zi[k], pr, pi, dr, di);
            double p2 = pr * pr + pi * pi;
            if (p2 == 0.0) { done |= 1u << k; continue; }
            // Newton ratio n = P/P'
            double d2 = dr * dr + di * di;
            double nx, ny;
            if (d2 > 0.0) { double id = 1.0 / d2; nx = (pr * dr + pi * di) * id; ny = (pi * dr - pr * di) * id; }
            else { nx = 1e-3; ny = 1e-3; }
            // repulsion S = sum_{j != k} 1/(z_k - z_j)
            double sx = 0.0, sy = 0.0;
#pragma unroll
            for (int j = 0; j < DEG; ++j) {
                if (j == k) continue;
                double ux = zr[k] - zr[j], uy = zi[k] - zi[j];
                double u2 = ux * ux + uy * uy;
                if (u2 > 0.0) { double iu = 1.0 / u2; sx += ux * iu; sy -= uy * iu; }
            }
            // step = n / (1 - n S)
            double ax = 1.0 - (nx * sx - ny * sy), ay = -(nx * sy + ny * sx);
            double a2 = ax * ax + ay * ay;
            double stx, sty;
            if (a2 > 1e-300) { double ia = 1.0 / a2; stx = (nx * ax + ny * ay) * ia; sty = (ny * ax - nx * ay) * ia; }
            else { stx = nx; sty = ny; }
            zr[k] -= stx; zi[k] -= sty;
            double z2 = zr[k] * zr[k] + zi[k] * zi[k];
            double rel = (stx * stx + sty * sty) / (z2 + 1e-12);
            if (!(rel == rel)) bad = true;
            if (rel < tol2 || (rel < 1e-6 && rel > 0.5 * prev[k])) done |= 1u << k;
            prev[k] = rel;
        }
        if (bad) return max_it + 1;
        if (done == all) return it;
    }
    return max_it + 1;
}

// Keep root identities along a path in w: permute the new roots so that slot j holds the one nearest to
// slot j's previous position (greedy in slot order). Roots move continuously with w, so after this a slot
// can only confuse roots that are closer to each other than one step of the path.
template <int DEG>
UL_HD void match_roots(const double* ozr, const double* ozi, double* zr, double* zi, unsigned fixed = 0)
{
    double nr[DEG], ni[DEG];
    unsigned used = fixed;               // slots in `fixed` keep their root (continued images)
    bool ident = true;
#pragma unroll
    for (int j = 0; j < DEG; ++j) {
        if (fixed & (1u << j)) { nr[j] = zr[j]; ni[j] = zi[j]; continue; }
        int best = -1; double bd = 1e300;
#pragma unroll
        for (int k = 0; k < DEG; ++k) {
            if (used & (1u << k)) continue;
            double dx = zr[k] - ozr[j], dy = zi[k] - ozi[j];
            double d = dx * dx + dy * dy;
            if (d < bd || best < 0) { bd = d; best = k; }
        }
        used |= 1u << best;
        nr[j] = zr[best]; ni[j] = zi[best];
        ident = ident && (best == j);
    }
    if (!ident) {
#pragma unroll
        for (int j = 0; j < DEG; ++j) { zr[j] = nr[j]; zi[j] = ni[j]; }
    }
}

// Out-of-line copies for the region builder: k_regions calls these from several places inside loops over
// the root slots; inlined and unrolled they made a 0.5-1 MB kernel that stalled on instruction fetch
// (ncu: stall_no_instruction 11.8 per issue). The arithmetic is the same.
// ea_iterate with the loop over the roots kept rolled (the root arrays are indexed dynamically and live in
// local memory, L1-resident): one fifth / one tenth of the code of the unrolled form, same arithmetic.
template <int DEG>
UL_HDNI int ea_iterate_ni(const double* br_, const double* bi_, double* zr, double* zi, int max_it, double tol2,
                          unsigned done0 = 0)
{
    double br[DEG + 1], bi[DEG + 1], prev[DEG];
#pragma unroll
    for (int l = 0; l <= DEG; ++l) { br[l] = br_[l]; bi[l] = bi_[l]; }
#pragma unroll
    for (int k = 0; k < DEG; ++k) prev[k] = 1e300;
    unsigned done = done0;               // roots known exactly beforehand: frozen, but still repelling the others
    const unsigned all = (1u << DEG) - 1u;
    if (done == all) return 1;
    for (int it = 1; it <= max_it; ++it) {
        bool bad = false;
#pragma unroll 1
        for (int k = 0; k < DEG; ++k) {
            if (done & (1u << k)) continue;
            const double zkr = zr[k], zki = zi[k];
            double pr, pi, dr, di;
            horner2<DEG>(br, bi, zkr, zki, pr, pi, dr, di);
            double p2 = pr * pr + pi * pi;
            if (p2 == 0.0) { done |= 1u << k; continue; }
            double d2 = dr * dr + di * di;
            double nx, ny;
            if (d2 > 0.0) { double id = 1.0 / d2; nx = (pr * dr + pi * di) * id; ny = (pi * dr - pr * di) * id; }
            else { nx = 1e-3; ny = 1e-3; }
            double sx = 0.0, sy = 0.0;
#pragma unroll 1
            for (int j = 0; j < DEG; ++j) {
                if (j == k) continue;
                double ux = zkr - zr[j], uy = zki - zi[j];
                double u2 = ux * ux + uy * uy;
                if (u2 > 0.0) { double iu = 1.0 / u2; sx += ux * iu; sy -= uy * iu; }
            }
            double ax = 1.0 - (nx * sx - ny * sy), ay = -(nx * sy + ny * sx);
            double a2 = ax * ax + ay * ay;
            double stx, sty;
            if (a2 > 1e-300) { double ia = 1.0 / a2; stx = (nx * ax + ny * ay) * ia; sty = (ny * ax - nx * ay) * ia; }
            else { stx = nx; sty = ny; }
            const double nzr = zkr - stx, nzi = zki - sty;
            zr[k] = nzr; zi[k] = nzi;
            double z2 = nzr * nzr + nzi * nzi;
            double rel = (stx * stx + sty * sty) / (z2 + 1e-12);
            if (!(rel == rel)) bad = true;
            if (rel < tol2 || (rel < 1e-6 && rel > 0.5 * prev[k])) done |= 1u << k;
            prev[k] = rel;
        }
        if (bad) return max_it + 1;
        if (done == all) return it;
    }
    return max_it + 1;
}
template <int DEG>
UL_HDNI void ea_init_ni(const double* br, const double* bi, double* zr, double* zi) { ea_init<DEG>(br, bi, zr, zi); }
template <int N>
UL_HDNI bool polish_image_ni(const Lens& L, double wx, double wy, double& zx, double& zy, int max_it,
                             double tol, double& detJ, double& resid, double& gx, double& gy, double reject_frac2 = 0.0)
{
    return polish_image<N>(L, wx, wy, zx, zy, max_it, tol, detJ, resid, gx, gy, reject_frac2, false);
}
template <int N>
UL_HDNI void poly_coeffs_ni(const Lens& L, const LensPoly& T, double wx, double wy, double* br, double* bi)
{
    poly_coeffs<N>(L, T, wx, wy, br, bi);
}

// ------------------------------------------------------------------------------------------------
// Step a2 for one source position: all N^2+1 roots (Eq. 4, Eq. 7), validated and polished on Eq. 1 (G7).
// zr/zi: the roots (images polished); mask: which slots are images. Returns the status word
// (UL_ST_EA_NOCONV, UL_ST_IMG_PARITY, image count << 8).
// ------------------------------------------------------------------------------------------------
template <int N>
UL_HDN unsigned centre_images(const Lens& L, const LensPoly& T, double wx, double wy, double* zr, double* zi, unsigned& mask,
                              bool warm = false)
{
    constexpr int DEG = N * N + 1;
    double br[DEG + 1], bi[DEG + 1];
    poly_coeffs<N>(L, T, wx, wy, br, bi);
    if (!warm) ea_init<DEG>(br, bi, zr, zi);            // warm: zr, zi hold the roots of a nearby source position
    int it = ea_iterate<DEG>(br, bi, zr, zi, 100);
    unsigned st = (it > 100) ? UL_ST_EA_NOCONV : 0u;
    // validate + polish (G7): damped Newton on Eq. 1 from every root; accept converged, un-moved, distinct ones
    double ix[DEG], iy[DEG];
    int n_img = 0;
    mask = 0;
#pragma unroll
    for (int k = 0; k < DEG; ++k) {
        double zx = zr[k], zy = zi[k], detJ, resid, gx, gy;
        // a polish that converges IS an image wherever it started (Eq. 1 is the definition); starts
        // from spurious roots may land on an image already found: the duplicate test below drops those
        bool ok = polish_image<N>(L, wx, wy, zx, zy, 16, 1e-13, detJ, resid, gx, gy);
        if (ok) {
            double sc = ul_max(1.0, zx * zx + zy * zy);
            for (int q = 0; q < n_img; ++q) {
                double ddx = zx - ix[q], ddy = zy - iy[q];
                if (ddx * ddx + ddy * ddy < 1e-18 * sc) ok = false;
            }
        }
        if (ok) { ix[n_img] = zx; iy[n_img] = zy; ++n_img; mask |= 1u << k; zr[k] = zx; zi[k] = zy; }
    }
    // An image count of the wrong parity almost always means the ultra-faint image next to a light
    // lens was lost: it sits at z ~ a_i + eps_i / conj(a_i - w - sum_{j!=i} eps_j/conj(a_i - a_j)), inside
    // the cluster of spurious roots around a_i that EA cannot resolve in double (degree 10). Seed it there.
    if constexpr (N > 1) {
        if (((n_img - (N + 1)) & 1) != 0 || n_img < N + 1) {
#pragma unroll
            for (int a = 0; a < N; ++a) {
                double tx = L.ax[a] - wx, ty = L.ay[a] - wy;
#pragma unroll
                for (int b = 0; b < N; ++b) {
                    if (b == a) continue;
                    double dx = L.ax[a] - L.ax[b], dy = L.ay[a] - L.ay[b];
                    double i2 = L.eps[b] / (dx * dx + dy * dy);
                    tx -= dx * i2; ty -= dy * i2;               // eps_b / conj(d) = eps_b d / |d|^2
                }
                double t2 = tx * tx + ty * ty;
                if (!(t2 > 0.0)) continue;
                double zx = L.ax[a] + L.eps[a] * tx / t2, zy = L.ay[a] + L.eps[a] * ty / t2;   // eps/conj(t) = eps t/|t|^2
                double detJ, resid, gx, gy;
                bool ok = polish_image<N>(L, wx, wy, zx, zy, 12, 1e-13, detJ, resid, gx, gy);
                if (ok) {
                    double sc = ul_max(1.0, zx * zx + zy * zy);
                    for (int q = 0; q < n_img; ++q) {
                        double ddx = zx - ix[q], ddy = zy - iy[q];
                        if (ddx * ddx + ddy * ddy < 1e-18 * sc) ok = false;
                    }
                }
                if (!ok) continue;
                // put it in the non-image slot nearest to it
                int slot = -1; double bd = 1e300;
#pragma unroll
                for (int k = 0; k < DEG; ++k) {
                    if (mask & (1u << k)) continue;
                    double ddx = zr[k] - zx, ddy = zi[k] - zy, d = ddx * ddx + ddy * ddy;
                    if (d < bd) { bd = d; slot = k; }
                }
                if (slot < 0) continue;
                ix[n_img] = zx; iy[n_img] = zy; ++n_img; mask |= 1u << slot; zr[slot] = zx; zi[slot] = zy;
            }
        }
    }
    // Still the wrong parity: images next to a LIGHT lens (eps_a < 1e-2: the pair a planetary caustic adds, of ordinary
    // brightness) hide in the same unresolved cluster (seen on C3 with q3 ~ 1e-5: A off by 10-40 %).
    // Seed Eq. 1 from 8 points of that lens's own Einstein ring |z - a| = sqrt(eps_a), where those images live.
    if constexpr (N > 1) {
#pragma unroll 1
        for (int a = 0; a < N; ++a) {
            if (!(L.eps[a] < 1e-2)) continue;
            const double re = sqrt(L.eps[a]);
            // a missing PAIR leaves the parity right: where the source sits on this lens's planetary caustic (centre
            // w_a = a_a - sum_{b != a} eps_b/conj(a_a - a_b), a few sqrt(eps_a) across) the ring is seeded regardless
            bool near = false;
            if (N == 3) {
                double tx = L.ax[a] - wx, ty = L.ay[a] - wy;
#pragma unroll
                for (int b = 0; b < N; ++b) {
                    if (b == a) continue;
                    double dx = L.ax[a] - L.ax[b], dy = L.ay[a] - L.ay[b];
                    double i2 = L.eps[b] / (dx * dx + dy * dy);
                    tx -= dx * i2; ty -= dy * i2;
                }
                near = tx * tx + ty * ty < 64.0 * L.eps[a];
            }
            if (!near && !(((n_img - (N + 1)) & 1) != 0 || n_img < N + 1)) continue;
#pragma unroll 1
            for (int k = 0; k < 8; ++k) {
                double zx = L.ax[a] + re * UL_RING8_X(k), zy = L.ay[a] + re * UL_RING8_Y(k);
                double detJ, resid, gx, gy;
                bool ok = polish_image<N>(L, wx, wy, zx, zy, 12, 1e-13, detJ, resid, gx, gy);
                if (ok) {
                    double sc = ul_max(1.0, zx * zx + zy * zy);
                    for (int q = 0; q < n_img; ++q) {
                        double ddx = zx - ix[q], ddy = zy - iy[q];
                        if (ddx * ddx + ddy * ddy < 1e-18 * sc) ok = false;
                    }
                }
                if (!ok || n_img >= DEG) continue;
                int slot = -1; double bd = 1e300;
                for (int m = 0; m < DEG; ++m) {
                    if (mask & (1u << m)) continue;
                    double ddx = zr[m] - zx, ddy = zi[m] - zy, d = ddx * ddx + ddy * ddy;
                    if (d < bd) { bd = d; slot = m; }
                }
                if (slot < 0) continue;
                ix[n_img] = zx; iy[n_img] = zy; ++n_img; mask |= 1u << slot; zr[slot] = zx; zi[slot] = zy;
            }
        }
    }
    if (((n_img - (N + 1)) & 1) != 0 || n_img < N + 1) st |= UL_ST_IMG_PARITY;
    st |= (unsigned)(n_img & 0xf) << 8;
    return st;
}

// ------------------------------------------------------------------------------------------------
// App. A: ring quadrature along theta
// ------------------------------------------------------------------------------------------------

// zeta(-1/2, u) and zeta(-3/2, u) for u in (0, 1]: Hurwitz zeta = u^(-s) + zeta(s, 1+u); the smooth part
// zeta(s, 1+u) is a degree-9 least-squares fit at 64 Chebyshev nodes of [0,1] (max error 6e-10 / 2e-10). The ONE copy
// of the tables; paper_2510_02639_b200/csrc/fit_zeta_tables.py regenerates them (mpmath) and tests/test_host_logic.py
// checks them against mpmath.zeta to 1e-9 and against the script's output.
#define UL_ZETA_M12_COEFFS {-0.207886224399935288, -0.730177374187579331, -0.326542779711049336, \
                            0.0837867303083785903, -0.0436173603868350857, 0.0271895277281179355, \
                            -0.0166136306767131411, 0.00831433648693249115, -0.00278385068661135939, \
                            0.0004444009766404081}
#define UL_ZETA_M32_COEFFS {-0.0254852020332272215, -0.311829307850673643, -0.547633958335979165, \
                            -0.163259739667364207, 0.0313455313556175105, -0.0128110506256419159, \
                            0.00618207285304185443, -0.0027041446390176113, 0.000838584837043554769, \
                            -0.000127987893602585462}
// value and derivative of the degree-9 polynomial c[0] + c[1] u + ...
UL_HD void zeta_poly(const double (&c)[10], double u, double& p, double& dp)
{
    p = c[9]; dp = 0.0;
#pragma unroll
    for (int i = 8; i >= 0; --i) { dp = dp * u + p; p = p * u + c[i]; }
}
UL_HD double zeta_m12(double u)
{
    const double c[10] = UL_ZETA_M12_COEFFS;
    double p = c[9];
#pragma unroll
    for (int i = 8; i >= 0; --i) p = p * u + c[i];
    return sqrt(u) + p;
}
UL_HD double zeta_m32(double u)
{
    const double c[10] = UL_ZETA_M32_COEFFS;
    double p = c[9];
#pragma unroll
    for (int i = 8; i >= 0; --i) p = p * u + c[i];
    return u * sqrt(u) + p;
}
// the same with d/du (forward-mode variant). d sqrt(u)/du is singular at u = 0 (a node exactly on the edge: the
// rule is not differentiable there). That term is the counterpart of the first inside node's own weight
// -1/(2 sqrt(-F)): the two cancel to leading order, so they are kept or dropped TOGETHER. keep_sing = the scan loop
// kept the node's weight (-F above UL_DUAL_SING_FLOOR rho^2, ulens_dual.cuh).
UL_HD void zeta_m12_du(double u, bool keep_sing, double& z, double& dz)
{
    const double c[10] = UL_ZETA_M12_COEFFS;
    double p, dp; zeta_poly(c, u, p, dp);
    const double su = sqrt(u);
    z = su + p; dz = ((keep_sing && u > 1e-14) ? 0.5 / su : 0.0) + dp;
}
UL_HD void zeta_m32_du(double u, double& z, double& dz)
{
    const double c[10] = UL_ZETA_M32_COEFFS;
    double p, dp; zeta_poly(c, u, p, dp);
    const double su = sqrt(u);
    z = u * su + p; dz = 1.5 * su + dp;
}

// F(z) = |w(z) - w_c|^2 - rho^2  (inside the source image <=> F < 0), one reciprocal per ray.
// A ray on a lens gives inf/NaN -> clamped to +UL_BIG (outside), never NaN.
template <int N>
UL_HD double ray_F(const Lens& L, double x, double y, double wcx, double wcy, double rho2)
{
    double ux = x - wcx, uy = y - wcy;
    double F;
    if constexpr (N == 1) {
        double dx = x - L.ax[0], dy = y - L.ay[0];
        double inv = L.eps[0] / (dx * dx + dy * dy);
        double ex = ux - dx * inv, ey = uy - dy * inv;
        F = ex * ex + ey * ey - rho2;
    } else if constexpr (N == 2) {
        double d1x = x - L.ax[0], d1y = y - L.ay[0];
        double d2x = x - L.ax[1], d2y = y - L.ay[1];
        double D1 = d1x * d1x + d1y * d1y, D2 = d2x * d2x + d2y * d2y;
        double inv = 1.0 / (D1 * D2);
        double e1 = L.eps[0] * D2 * inv, e2 = L.eps[1] * D1 * inv;
        double ex = ux - e1 * d1x - e2 * d2x, ey = uy - e1 * d1y - e2 * d2y;
        F = ex * ex + ey * ey - rho2;
    } else {
        double d1x = x - L.ax[0], d1y = y - L.ay[0];
        double d2x = x - L.ax[1], d2y = y - L.ay[1];
        double d3x = x - L.ax[2], d3y = y - L.ay[2];
        double D1 = d1x * d1x + d1y * d1y, D2 = d2x * d2x + d2y * d2y, D3 = d3x * d3x + d3y * d3y;
        double D12 = D1 * D2;
        double inv = 1.0 / (D12 * D3);
        double e1 = L.eps[0] * D2 * D3 * inv, e2 = L.eps[1] * D1 * D3 * inv, e3 = L.eps[2] * D12 * inv;
        double ex = ux - e1 * d1x - e2 * d2x - e3 * d3x, ey = uy - e1 * d1y - e2 * d2y - e3 * d3y;
        F = ex * ex + ey * ey - rho2;
    }
    return fmin(F, UL_BIG);    // fmin returns the non-NaN operand
}

// One boundary crossing between nodes 1 and 2 of the window (f0, f1, f2, f3) at x = -1, 0, 1, 2
// (cubic Lagrange interpolant, App. A.1, G13; linear fallback if the cubic has no root in the cell).
// Returns u = distance (in cells) from the crossing to the first inside node, entering = node 1 outside,
// and dS = the end correction of the midpoint sum of sqrt(-F) over the inside run (in cells):
//   sum - integral = sqrt(sigma) [ zeta(-1/2,u) + t2 zeta(-3/2,u) ],   -F ~ sigma xi (1 + 2 t2 xi) from the edge
// (Navot's correction for an x^(1/2) end singularity; its first cell is the paper's f(delta) b(delta),
// Eqs. A7-A8, G12). The uniform part follows from u: zeta(0,u) = 1/2 - u (== Eq. A3 point-centred, G9/G10).
// t2_extra adds the logarithmic slope of a smooth weight (the r of r dr on radial scan lines).
UL_HD void edge_event(double f0, double f1, double f2, double f3, bool want_S, double t2_extra,
                      double& u, bool& entering, double& dS)
{
    double c0 = f1;
    double c1 = (-2.0 * f0 - 3.0 * f1 + 6.0 * f2 - f3) * (1.0 / 6.0);
    double c2 = (f0 - 2.0 * f1 + f2) * 0.5;
    double c3 = (-f0 + 3.0 * f1 - 3.0 * f2 + f3) * (1.0 / 6.0);
    double x = f1 / (f1 - f2);                       // linear guess, in (0,1) because the signs differ
    bool cubic_ok = true;
#pragma unroll 1
    for (int it = 0; it < 4; ++it) {
        double p = c0 + x * (c1 + x * (c2 + x * c3));
        double dp = c1 + x * (2.0 * c2 + 3.0 * x * c3);
        double xn = x - p / dp;
        if (!(xn >= 0.0 && xn <= 1.0)) { cubic_ok = false; break; }
        x = xn;
    }
    double dp, d2p;
    if (cubic_ok) {
        dp = c1 + x * (2.0 * c2 + 3.0 * x * c3);
        d2p = 2.0 * c2 + 6.0 * x * c3;
    } else {                                        // G13 fallback: linear interpolation
        x = f1 / (f1 - f2);
        dp = f2 - f1; d2p = 0.0;
    }
    entering = !(f1 < 0.0);                         // node 1 outside, node 2 inside
    u = entering ? 1.0 - x : x;
    dS = 0.0;
    if (want_S) {
        double sigma = entering ? -dp : dp;         // slope of -F away from the edge, per cell
        double tau = -0.5 * d2p;
        if (sigma > 0.0) {
            double ss = sqrt(sigma);
            double corr = ss * zeta_m12(u);
            double t2 = tau / (2.0 * sigma) + (entering ? t2_extra : -t2_extra);
            if (fabs(t2) < 0.5) corr += ss * t2 * zeta_m32(u);
            dS = -corr;
        }
    }
}

// The edge events of a scan line are DEFERRED: each of the 32 lines of a work unit meets the image edge at its own node,
// so an event evaluated on the spot runs with 1-2 lanes of the warp active (round 1, ncu: 19 % of k_shoot's warp
// instructions, 24 of 32 lanes active on average). The loop only notes the node index of a sign change (two slots: a line
// through one image has an entry and an exit); the events are resolved after the loop, where the lanes of the warp are
// together again, from the four window rays recomputed at the noted node. A third event on a line resolves the oldest
// one on the spot. The recomputed window may differ from the loop's values in the last bit (another rounding path), which
// can flip the sign of a node sitting exactly on the edge: the loop's classification (entering: node 1 outside, node 2
// inside) is authoritative, a disagreeing node is moved onto the edge.
UL_HD void enforce_crossing(double& w1, double& w2, bool entering)
{
    if (entering) { if (w1 < 0.0) w1 = 0.0; if (!(w2 < 0.0)) w2 = -1e-9 * fabs(w1) - 1e-300; }
    else { if (!(w1 < 0.0)) w1 = -1e-9 * fabs(w2) - 1e-300; if (w2 < 0.0) w2 = 0.0; }
}

// the event noted at node pj of a ring: pair (pj-2, pj-1), window nodes pj-3 .. pj at angles th0 + (k + 1/2) dth
template <int N, bool LD>
UL_HD void ring_event(const Lens& L, double wcx, double wcy, double rho2, double r, double th0, double dth, double cd, double sd,
                      int pj, bool entering, double& U, double& S)
{
    const double a = th0 + (pj - 2.5) * dth;
    double wc = cos(a), ws = sin(a), w[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        w[k] = ray_F<N>(L, r * wc, r * ws, wcx, wcy, rho2);
        const double cn = wc * cd - ws * sd; ws = ws * cd + wc * sd; wc = cn;
    }
    enforce_crossing(w[1], w[2], entering);
    double u, dS; bool en;
    edge_event(w[0], w[1], w[2], w[3], LD, 0.0, u, en, dS);
    U += u - 0.5; S += dS;
}

// the event noted at node pi of a radial line (direction c, s): pair (pi-2, pi-1), window nodes pi-3 .. pi
template <int N, bool LD>
UL_HD void col_event(const Lens& L, double wcx, double wcy, double rho2, double c, double s, double r0, double dr,
                     int pi, bool entering, double& U2, double& S)
{
    double w[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const double rk = r0 + (pi - 3 + k + 0.5) * dr;
        w[k] = ray_F<N>(L, rk * c, rk * s, wcx, wcy, rho2);
    }
    enforce_crossing(w[1], w[2], entering);
    const double r1 = r0 + (pi - 1.5) * dr;              // node pi-2
    const double rh = r1 + 0.5 * dr;                     // cell face between the pair
    const double rin = entering ? r1 + dr : r1;          // first inside node
    const double t2x = dr / ul_max(rin, 0.5 * dr);
    double u, dS; bool en;
    edge_event(w[0], w[1], w[2], w[3], LD, t2x, u, en, dS);
    double rc = en ? (r1 + dr) - u * dr : r1 + u * dr;
    rc = ul_max(rc, 0.0);
    U2 += en ? 0.5 * (rh * rh - rc * rc) : 0.5 * (rc * rc - rh * rh);
    S += dS * rc;
}

// Integrate one ring r over theta:  U = Int chi dtheta / dth,  S = Int chi sqrt(-F) dtheta / dth  (both in cells).
// Rays at th0 + (j + 1/2) dth, j = -2 .. n_th+1 (two halo rays per side feed the cubic stencil; for a
// periodic sector they are the wrapped rays). edge = true if one of the first / last two rays of a
// bounded sector is inside (the margin was too small).
template <int N, bool LD>
UL_HD void shoot_ring(const Lens& L, double wcx, double wcy, double rho2, double r, double th0, double dth,
                      int n_th, bool periodic, double& U_out, double& S_out, bool& edge)
{
    const double cd = cos(dth), sd = sin(dth);
    double t = th0 - 1.5 * dth;
    double c = cos(t), s = sin(t);
    double f1 = UL_BIG, f2 = UL_BIG;
    double U = 0.0, S = 0.0;
    edge = false;
    const int j_first = periodic ? 2 : 1;
    int npend = 0, pj0 = 0, pj1 = 0;
    unsigned pen = 0;
    auto resolve = [&](int pj, bool entering) { ring_event<N, LD>(L, wcx, wcy, rho2, r, th0, dth, cd, sd, pj, entering, U, S); };
    // per ray: count it, then note the pair (j-2, j-1) = (f1, f2) if the sign changes between them. In a periodic
    // sector pair (-1, 0) is pair (n_th-1, n_th) again: take it once.
    auto node = [&](int j, double f3) {
        if (j >= 0 && j < n_th && f3 < 0.0) {
            U += 1.0;
            if (LD) S += -f3 * ul_rsqrt(-f3);      // (x rsqrt(x): cheaper than sqrt(x) in FP64, 1-2 ulp)
            if (!periodic && (j < 2 || j >= n_th - 2)) edge = true;
        }
        if (j >= j_first && ((f1 < 0.0) != (f2 < 0.0))) {
            if (npend == 2) { resolve(pj0, (pen & 1u) != 0); pj0 = pj1; pen >>= 1; npend = 1; }
            if (npend == 0) pj0 = j; else pj1 = j;
            if (!(f1 < 0.0)) pen |= 1u << npend;
            ++npend;
        }
        f1 = f2; f2 = f3;
    };
    // two rays in flight per iteration: their lens maps are independent, which doubles the FP64 pipe's
    // instruction-level parallelism (the rotation recurrence is the only loop-carried chain)
    for (int j = -2; j <= n_th + 1; j += 2) {
        const double c2 = c * cd - s * sd, s2 = s * cd + c * sd;
        const double fa = ray_F<N>(L, r * c, r * s, wcx, wcy, rho2);
        const double fb = ray_F<N>(L, r * c2, r * s2, wcx, wcy, rho2);
        node(j, fa);
        if (j + 1 <= n_th + 1) node(j + 1, fb);
        c = c2 * cd - s2 * sd;
        s = s2 * cd + c2 * sd;
    }
    if (npend > 0) resolve(pj0, (pen & 1u) != 0);
    if (npend > 1) resolve(pj1, (pen & 2u) != 0);
    U_out = U; S_out = S;
}

// Scan line `line` of a sector: its coordinate across the lines (radius of a ring, or theta of a radial line)
// and its quadrature weight. r0, dr describe the span [r0, r0 + n_r dr]; with UL_PATCH_SINR the rings sit at Chebyshev-like radii
// r_c + h sin(phi) (midpoint rule in phi): where the span ends at the radial extremes of a convex image the
// integrand chord(r) ~ sqrt((r - r_lo)(r_hi - r)) becomes smooth in phi and the rule converges spectrally
// instead of like dr^1.5 (measured on the single-lens closed form in DESIGN.md).
UL_HD void line_node(int flags, int n_r, int line, double r0, double dr, double& r, double& w)
{
    if (flags & UL_PATCH_SINR) {
        double h = 0.5 * n_r * dr, ph = (line + 0.5) * (UL_PI / n_r);      // phi + pi/2
        double s, c; s = sin(ph); c = cos(ph);
        r = r0 + h * (1.0 - c);                                              // r_c - h cos(ph) = r_c + h sin(phi)
        w = h * s * (UL_PI / n_r);
    } else { r = r0 + (line + 0.5) * dr; w = dr; }
}

// Integrate one radial line theta over r (filled ring / disk sectors):
//   U = Int chi r dr,  S = Int chi sqrt(-F) r dr   (length^2 units). Nodes at r0 + (i + 1/2) dr, i = -2 .. n_r+1.
// A node with r < 0 is the point on the opposite side of the origin: F is smooth along the whole line, so
// the stencil stays valid; the inside run of a disk simply starts at node 0 (midpoint rule exact for r dr).
template <int N, bool LD>
UL_HD void shoot_col(const Lens& L, double wcx, double wcy, double rho2, double th, double r0, double dr,
                     int n_r, double& U_out, double& S_out, bool& edge)
{
    const double c = cos(th), s = sin(th);
    double f1 = UL_BIG, f2 = UL_BIG;
    double U = 0.0, S = 0.0, U2 = 0.0;
    edge = false;
    int npend = 0, pi0 = 0, pi1 = 0;
    unsigned pen = 0;
    auto resolve = [&](int pi, bool entering) { col_event<N, LD>(L, wcx, wcy, rho2, c, s, r0, dr, pi, entering, U2, S); };
    auto node = [&](int i, double r, double f3) {
        if (i >= 0 && i < n_r && f3 < 0.0) {
            U += r;
            if (LD) S += r * (-f3 * ul_rsqrt(-f3));
            if ((i < 2 && r0 > 0.0) || i >= n_r - 2) edge = true;
        }
        // pair (i-2, i-1) = (f1, f2); the cell face between the pair must lie at r > 0
        if (i >= 1 && ((f1 < 0.0) != (f2 < 0.0)) && (r0 + (i - 1.0) * dr > 0.0)) {
            if (npend == 2) { resolve(pi0, (pen & 1u) != 0); pi0 = pi1; pen >>= 1; npend = 1; }
            if (npend == 0) pi0 = i; else pi1 = i;
            if (!(f1 < 0.0)) pen |= 1u << npend;
            ++npend;
        }
        f1 = f2; f2 = f3;
    };
    for (int i = -2; i <= n_r + 1; i += 2) {               // two rays in flight (see shoot_ring)
        const double ra = r0 + (i + 0.5) * dr, rb = r0 + (i + 1.5) * dr;
        const double fa = ray_F<N>(L, ra * c, ra * s, wcx, wcy, rho2);
        const double fb = ray_F<N>(L, rb * c, rb * s, wcx, wcy, rho2);
        node(i, ra, fa);
        if (i + 1 <= n_r + 1) node(i + 1, rb, fb);
    }
    if (npend > 0) resolve(pi0, (pen & 1u) != 0);
    if (npend > 1) resolve(pi1, (pen & 2u) != 0);
    U_out = U * dr + U2; S_out = S * dr;
}

}  // namespace ulens
