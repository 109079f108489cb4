// ulens_dual.cuh -- forward-mode variant of the ray-shooting integrator (step a8).
//
// PAPER.md Sec. 3.5: derivatives of the magnification by forward-mode differentiation THROUGH
// the region construction and the quadrature. What is differentiated here is the discrete rule of
// ulens_core.cuh with the inside flags piecewise constant:
//   * the grid of a sector moves with the image across its scan lines: the span's two ends carry tangents
//     obtained from the extreme image-limb points by implicit differentiation of Eq. 1 (P:163-175 uses the
//     polynomial; the lens equation itself is better conditioned) -- without this the square-root behaviour
//     of the chord length at the ends of an image ruins the derivative;
//   * every ray's F = |w(z) - w_c|^2 - rho^2 has the tangent  dF_m = mot_m h + explicit_m  in direction m:
//     grid motion (mot_m = how the ray's scan line moves, h = the ray's response to it) + the explicit
//     dependence of Eq. 1 on the lens parameters + the source centre / radius;
//   * the edge position from the cubic, the uniform weight u - 1/2 and the square-root end correction
//     (Hurwitz zetas) are differentiated exactly, so the edge-motion (Reynolds boundary) term is that of the
//     rule itself and the paper's sigmoid surrogate for the Heaviside function (Eq. 9) is not needed.
//
// HOW (round 2). Every tangent of a line integral is LINEAR in the tangents of the rays that feed it:
//   dU_m = sum_rays a_ray dF_ray,m ,   dS_m = sum_rays b_ray dF_ray,m
// with weights a, b that do not depend on the direction m (for an inside ray of the limb-darkened term
// b = -1/(2 sqrt(-F)); for the four window rays of an edge event a, b are the sensitivities of the cubic's root
// and of the end correction to the window values, edge_event_adj). And dF_ray,m is itself a contraction of a few
// per-ray numbers (the "basis": h, 2(w - w_c), and per lens Re conj(E)/conj(d_i), conj(E)/conj(d_i)^2) with the
// per-configuration tangent table. So a scan line accumulates weight x basis into two small statistic sets
// (TanStat, 4 + 3 N doubles each) and contracts them with the table ONCE per line, instead of carrying NT
// tangents through every ray and through the Newton iteration of every edge event (round 1: 114 FP64
// instructions per ray and ~600 per event in 6-component dual arithmetic, 250 registers). Outside rays cost
// what they cost in the primal kernel; the number of directions (5 binary, 8 triple) only enters per line.
#pragma once
#include "ulens_core.cuh"

namespace ulens {

// Tangent directions. m = 0, 1: source centre (w_cx, w_cy); m = 2 .. NT-2: lens parameters in the geometry of
// ulens_lens_binary / ulens_lens_triple (binary: s, q; triple: s, q, q3, r3, psi); m = NT-1: rho.
#define UL_NT_MAX 8
#define UL_NT 5          // binary (and single) lens: w_cx, w_cy, s, q, rho
template <int N> struct TanDirs { static constexpr int NT = (N == 3) ? 8 : 5; };

// how the inputs of Eq. 1 / Eq. 5 move in each direction (filled on the host per configuration, upload_tangents)
struct TangentTable {
    double dwx[UL_NT_MAX], dwy[UL_NT_MAX], drho[UL_NT_MAX];
    double deps[UL_NT_MAX][3], dax[UL_NT_MAX][3], day[UL_NT_MAX][3];
};

template <int NT>
struct Dual {
    double v;
    double d[NT];
};

template <int NT> UL_HD Dual<NT> dual_const(double a) { Dual<NT> r; r.v = a; for (int k = 0; k < NT; ++k) r.d[k] = 0.0; return r; }
template <int NT> UL_HD Dual<NT> operator+(const Dual<NT>& a, const Dual<NT>& b) { Dual<NT> r; r.v = a.v + b.v; for (int k = 0; k < NT; ++k) r.d[k] = a.d[k] + b.d[k]; return r; }
template <int NT> UL_HD Dual<NT> operator-(const Dual<NT>& a, const Dual<NT>& b) { Dual<NT> r; r.v = a.v - b.v; for (int k = 0; k < NT; ++k) r.d[k] = a.d[k] - b.d[k]; return r; }
template <int NT> UL_HD Dual<NT> operator*(const Dual<NT>& a, const Dual<NT>& b) { Dual<NT> r; r.v = a.v * b.v; for (int k = 0; k < NT; ++k) r.d[k] = a.d[k] * b.v + a.v * b.d[k]; return r; }
template <int NT> UL_HD Dual<NT> operator*(const Dual<NT>& a, double b) { Dual<NT> r; r.v = a.v * b; for (int k = 0; k < NT; ++k) r.d[k] = a.d[k] * b; return r; }
template <int NT> UL_HD Dual<NT> operator/(const Dual<NT>& a, const Dual<NT>& b)
{
    Dual<NT> r; double ib = 1.0 / b.v; r.v = a.v * ib;
    for (int k = 0; k < NT; ++k) r.d[k] = (a.d[k] - r.v * b.d[k]) * ib;
    return r;
}

// ------------------------------------------------------------------------------------------------ per-ray quantities

// Eq. 1 at one ray, keeping what the tangents reuse: d_i = z - a_i, 1/|d_i|^2 (one reciprocal per ray through the
// common denominator, as ray_F), w - w_c and F. A ray on a lens gives inf/NaN -> F = +UL_BIG (outside).
template <int N>
struct RayCore {
    double dx[N], dy[N], iv[N];
    double ex, ey, F;
};

template <int N>
UL_HD void ray_core(const Lens& L, double x, double y, double wcx, double wcy, double rho2, RayCore<N>& R)
{
    double D[N];
#pragma unroll
    for (int i = 0; i < N; ++i) { R.dx[i] = x - L.ax[i]; R.dy[i] = y - L.ay[i]; D[i] = R.dx[i] * R.dx[i] + R.dy[i] * R.dy[i]; }
    if constexpr (N == 1) {
        R.iv[0] = 1.0 / D[0];
    } else if constexpr (N == 2) {
        const double inv = 1.0 / (D[0] * D[1]);
        R.iv[0] = D[1] * inv; R.iv[1] = D[0] * inv;
    } else {
        const double D01 = D[0] * D[1];
        const double inv = 1.0 / (D01 * D[2]);
        R.iv[0] = D[1] * D[2] * inv; R.iv[1] = D[0] * D[2] * inv; R.iv[2] = D01 * inv;
    }
    double ex = x - wcx, ey = y - wcy;
#pragma unroll
    for (int i = 0; i < N; ++i) { const double e = L.eps[i] * R.iv[i]; ex -= e * R.dx[i]; ey -= e * R.dy[i]; }
    R.ex = ex; R.ey = ey;
    R.F = fmin(ex * ex + ey * ey - rho2, UL_BIG);      // fmin returns the non-NaN operand
}

// The numbers dF_m is contracted from (E = 2 (w - w_c), p_i = 1/conj(d_i), q_i = 1/conj(d_i)^2, g = sum eps_i q_i):
//   dF_m = mot_m h - dw_cx,m ex2 - dw_cy,m ey2 - 2 rho drho_m - sum_i [ deps_i,m cp_i + eps_i (dax_i,m cqr_i + day_i,m cqi_i) ]
//   h    = Re(conj(E) (e + g conj(e))),  e = unit displacement of the ray when its scan line moves:
//          ring (COL = false): the ring's radius moves, e = (c, s);
//          radial line (COL = true): the line turns, e = r (-s, c);
//   cp_i = Re(conj(E) p_i),  cqr_i + i cqi_i = conj(E) q_i        (Eq. 1 differentiated: dw = dz + g conj(dz)
//          - dw_c - sum_i [ deps_i p_i + eps_i conj(da_i) q_i ];  dF = Re(conj(E) dw) - 2 rho drho)
template <int N>
struct RayBasis {
    double h, ex2, ey2;
    double cp[N], cqr[N], cqi[N];
};

template <int N, bool COL>
UL_HD void ray_basis(const Lens& L, const RayCore<N>& R, double r, double c, double s, RayBasis<N>& B)
{
    const double ex2 = 2.0 * R.ex, ey2 = 2.0 * R.ey;
    double gx = 0.0, gy = 0.0;
#pragma unroll
    for (int i = 0; i < N; ++i) {
        const double px = R.dx[i] * R.iv[i], py = R.dy[i] * R.iv[i];
        const double qx = px * px - py * py, qy = 2.0 * px * py;
        gx += L.eps[i] * qx; gy += L.eps[i] * qy;
        B.cp[i] = ex2 * px + ey2 * py;
        B.cqr[i] = ex2 * qx + ey2 * qy;
        B.cqi[i] = ex2 * qy - ey2 * qx;
    }
    if (!COL) B.h = ex2 * (c + gx * c + gy * s) + ey2 * (s + gy * c - gx * s);
    else B.h = r * (ex2 * (-s - gx * s + gy * c) + ey2 * (c - gy * s - gx * c));
    B.ex2 = ex2; B.ey2 = ey2;
    if (!(R.F < UL_BIG)) {                               // ray on a lens: counts as outside, no tangent
        B.h = B.ex2 = B.ey2 = 0.0;
#pragma unroll
        for (int i = 0; i < N; ++i) B.cp[i] = B.cqr[i] = B.cqi[i] = 0.0;
    }
}

// sum over rays of weight x basis
template <int N>
struct TanStat {
    double h, ex, ey, one;
    double cp[N], cqr[N], cqi[N];
};

template <int N>
UL_HD void stat_zero(TanStat<N>& S)
{
    S.h = S.ex = S.ey = S.one = 0.0;
#pragma unroll
    for (int i = 0; i < N; ++i) S.cp[i] = S.cqr[i] = S.cqi[i] = 0.0;
}

template <int N>
UL_HD void stat_add(TanStat<N>& S, double w, const RayBasis<N>& B)
{
    S.h += w * B.h; S.ex += w * B.ex2; S.ey += w * B.ey2; S.one += w;
#pragma unroll
    for (int i = 0; i < N; ++i) { S.cp[i] += w * B.cp[i]; S.cqr[i] += w * B.cqr[i]; S.cqi[i] += w * B.cqi[i]; }
}

// out_m = sum_rays weight dF_ray,m  for the NT directions of table T; mot = how the line moves (NT values)
template <int N, int NT>
UL_HD void stat_contract(const Lens& L, const TangentTable& T, double rho, const TanStat<N>& S, const double* mot,
                         double scale, double* out)
{
#pragma unroll
    for (int m = 0; m < NT; ++m) {
        double v = mot[m] * S.h - T.dwx[m] * S.ex - T.dwy[m] * S.ey - 2.0 * rho * T.drho[m] * S.one;
        if (N > 1) {
#pragma unroll
            for (int i = 0; i < N; ++i)
                v -= T.deps[m][i] * S.cp[i] + L.eps[i] * (T.dax[m][i] * S.cqr[i] + T.day[m][i] * S.cqi[i]);
        }
        out[m] = scale * v;
    }
}

// ------------------------------------------------------------------------------------------------ edge events

// edge_event of ulens_core.cuh together with the sensitivities of its two outputs to the four window values:
//   du = sum_k au[k] df_k,   d(dS) = sum_k aS[k] df_k.
// With p(x) = sum_k f_k l_k(x) the cubic through the window (l_k = Lagrange basis at x = -1, 0, 1, 2) and x its root
// in [0, 1]:  dx = - sum_k l_k(x) df_k / p'(x)   (implicit-function theorem: the Reynolds boundary term of P:163-175
// for the discrete rule);  d p'(x) = sum_k l_k'(x) df_k + p''(x) dx,  d p''(x) = sum_k l_k''(x) df_k + p'''(x) dx;
// u, sigma, tau and the Hurwitz-zeta end correction are smooth functions of (x, p', p'').
// (out of line: an event is rare next to the rays, and inlined at the flush site it costs the scan loops ~60 registers)
UL_HDNI void edge_event_adj(double f0, double f1, double f2, double f3, bool want_S, bool keep_sing, double t2_extra,
                            double& u, bool& entering, double& dS, double* au, double* aS)
{
    // rows: coefficient of x^0..x^3; columns: f0..f3
    const double M1[4] = {-1.0 / 3.0, -0.5, 1.0, -1.0 / 6.0};
    const double M2[4] = {0.5, -1.0, 0.5, 0.0};
    const double M3[4] = {-1.0 / 6.0, 0.5, -0.5, 1.0 / 6.0};
    const double c0 = f1;
    const double c1 = (-2.0 * f0 - 3.0 * f1 + 6.0 * f2 - f3) * (1.0 / 6.0);
    const double c2 = (f0 - 2.0 * f1 + f2) * 0.5;
    const double c3 = (-f0 + 3.0 * f1 - 3.0 * f2 + f3) * (1.0 / 6.0);
    const double idf = 1.0 / (f1 - f2);
    double x = f1 * idf;                                // linear guess, in (0,1) because the signs differ
    bool cubic_ok = true;
#pragma unroll 1
    for (int it = 0; it < 5; ++it) {
        const double p = c0 + x * (c1 + x * (c2 + x * c3));
        const double dp = c1 + x * (2.0 * c2 + 3.0 * x * c3);
        const double xn = x - p / dp;
        if (!(xn >= 0.0 && xn <= 1.0)) { cubic_ok = false; break; }
        x = xn;
    }
    double dp, d2p, dx[4], ddp[4], dd2p[4];
    if (cubic_ok) {
        dp = c1 + x * (2.0 * c2 + 3.0 * x * c3);
        d2p = 2.0 * c2 + 6.0 * x * c3;
        const double idp = -1.0 / dp;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const double l = (k == 1 ? 1.0 : 0.0) + x * (M1[k] + x * (M2[k] + x * M3[k]));
            dx[k] = l * idp;
            ddp[k] = M1[k] + x * (2.0 * M2[k] + 3.0 * x * M3[k]) + d2p * dx[k];
            dd2p[k] = 2.0 * M2[k] + 6.0 * x * M3[k] + 6.0 * c3 * dx[k];
        }
    } else {                                            // G13 fallback: linear interpolation
        x = f1 * idf;
        dp = f2 - f1; d2p = 0.0;
        dx[0] = dx[3] = 0.0; dx[1] = -f2 * idf * idf; dx[2] = f1 * idf * idf;
        ddp[0] = ddp[3] = 0.0; ddp[1] = -1.0; ddp[2] = 1.0;
        dd2p[0] = dd2p[1] = dd2p[2] = dd2p[3] = 0.0;
    }
    entering = !(f1 < 0.0);                             // node 1 outside, node 2 inside
    u = entering ? 1.0 - x : x;
    const double sg = entering ? -1.0 : 1.0;
#pragma unroll
    for (int k = 0; k < 4; ++k) { au[k] = sg * dx[k]; aS[k] = 0.0; }
    dS = 0.0;
    if (want_S) {
        const double sigma = sg * dp;                   // slope of -F away from the edge, per cell
        const double tau = -0.5 * d2p;
        if (sigma > 0.0) {
            const double ss = sqrt(sigma);
            double z12, dz12, z32, dz32;
            zeta_m12_du(u, keep_sing, z12, dz12);
            zeta_m32_du(u, z32, dz32);
            const double t2 = tau / (2.0 * sigma) + (entering ? t2_extra : -t2_extra);
            const bool use32 = fabs(t2) < 0.5;
            const double zz = z12 + (use32 ? t2 * z32 : 0.0);
            dS = -ss * zz;
            // partial derivatives of corr = ss (z12(u) + t2 z32(u))
            const double c_sig = 0.5 * zz / ss - (use32 ? ss * z32 * tau / (2.0 * sigma * sigma) : 0.0);
            const double c_tau = use32 ? ss * z32 / (2.0 * sigma) : 0.0;
            const double c_u = ss * (dz12 + (use32 ? t2 * dz32 : 0.0));
#pragma unroll
            for (int k = 0; k < 4; ++k) aS[k] = -(c_sig * sg * ddp[k] - 0.5 * c_tau * dd2p[k] + c_u * au[k]);
        }
    }
}

// A node whose -F is below this fraction of rho^2 sits on the edge to rounding (the sector grids are anchored at limb
// points, i.e. at exact edge points, so this happens ~1e-5 per source point, not ~1e-10): d sqrt(-F) does not exist there.
#define UL_DUAL_SING_FLOOR 1e-10

// Edge events in the tangent loops are DEFERRED as in the primal loops (ulens_core.cuh shoot_ring): the loop notes the node
// of a sign change (two slots), the events are resolved in two extra passes after the rays, where the lanes of the warp
// are together again, from the four window rays recomputed at the noted node.
// (enforce_crossing, ulens_core.cuh, keeps the loop's classification of the pair authoritative for the recomputed window)

// ------------------------------------------------------------------------------------------------ scan lines

// shoot_ring of ulens_core.cuh with tangent statistics. U, S: the line sums (in cells); SU, SS: sum of weight x basis
// for U and for S (contract with stat_contract, mot = the ring radius' tangents). theta grid frozen.
template <int N, bool LD>
UL_HD void shoot_ring_t(const Lens& L, double wcx, double wcy, double rho2, double r, double th0, double dth,
                        int n_th, bool periodic, double& U_out, double& S_out, TanStat<N>& SU, TanStat<N>& SS, bool& edge)
{
    const double cd = cos(dth), sd = sin(dth);
    const double t = th0 - 1.5 * dth;
    double c = cos(t), s = sin(t);
    double f1 = UL_BIG, f2 = UL_BIG;
    double U = 0.0, S = 0.0;
    stat_zero(SU); stat_zero(SS);
    edge = false;
    const int j_first = periodic ? 2 : 1;
    int npend = 0, pj0 = 0, pj1 = 0;
    unsigned penb = 0;
    auto flush = [&](int pj, bool pen) {
        {
            // window nodes pj-3 .. pj at angles th0 + (k + 1/2) dth
            const double a = th0 + (pj - 2.5) * dth;
            double wc = cos(a), ws = sin(a);
            double w[4];
            RayCore<N> R;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                ray_core<N>(L, r * wc, r * ws, wcx, wcy, rho2, R);
                w[k] = R.F;
                const double cn = wc * cd - ws * sd; ws = ws * cd + wc * sd; wc = cn;
            }
            const bool keep = -w[pen ? 2 : 1] > UL_DUAL_SING_FLOOR * rho2;     // the loop's rule for the first inside node
            enforce_crossing(w[1], w[2], pen);
            double u, dS, au[4], aS[4]; bool en;
            edge_event_adj(w[0], w[1], w[2], w[3], LD, keep, 0.0, u, en, dS, au, aS);
            U += u - 0.5; S += dS;
            wc = cos(a); ws = sin(a);
#pragma unroll 1
            for (int k = 0; k < 4; ++k) {
                RayBasis<N> B;
                ray_core<N>(L, r * wc, r * ws, wcx, wcy, rho2, R);
                ray_basis<N, false>(L, R, r, wc, ws, B);
                stat_add(SU, au[k], B);
                if (LD) stat_add(SS, aS[k], B);
                const double cn = wc * cd - ws * sd; ws = ws * cd + wc * sd; wc = cn;
            }
        }
    };
    // (the loop runs up to two passes beyond the rays: they resolve the noted events -- one flush site in the code)
    for (int j = -2; j <= n_th + 3; ++j) {
        const bool last = j > n_th + 1;
        RayCore<N> R;
        ray_core<N>(L, r * c, r * s, wcx, wcy, rho2, R);
        const double f3 = last ? UL_BIG : R.F;
        if (j >= 0 && j < n_th && f3 < 0.0) {
            U += 1.0;
            if (LD) {
                // sqrt(-F) and its derivative -dF / (2 sqrt(-F)) from one reciprocal square root (no division). A node
                // (numerically) ON the edge has no such derivative: its weight and its counterpart in the end correction
                // (zeta_m12_du) are dropped together
                const double rs = ul_rsqrt(-f3);
                S += -f3 * rs;
                RayBasis<N> B;
                ray_basis<N, false>(L, R, r, c, s, B);
                stat_add(SS, (-f3 > UL_DUAL_SING_FLOOR * rho2) ? -0.5 * rs : 0.0, B);
            }
            if (!periodic && (j < 2 || j >= n_th - 2)) edge = true;
        }
        const bool ev = !last && j >= j_first && ((f1 < 0.0) != (f2 < 0.0));
        // a noted event is resolved after the rays (the two extra passes), or on the spot when a third one arrives
        if (npend > 0 && (last || (ev && npend == 2))) {
            flush(pj0, (penb & 1u) != 0);
            pj0 = pj1; penb >>= 1; --npend;
        }
        if (ev) {
            if (npend == 0) pj0 = j; else pj1 = j;
            if (!(f1 < 0.0)) penb |= 1u << npend;
            ++npend;
        }
        f1 = f2; f2 = f3;
        const double cn = c * cd - s * sd;
        s = s * cd + c * sd;
        c = cn;
    }
    U_out = U; S_out = S;
}

// shoot_col of ulens_core.cuh with tangent statistics: radial line at angle th (c = cos th, s = sin th), nodes
// r0 + (i + 1/2) dr FROZEN along the line; the line itself turns (mot = theta's tangents). U_out, S_out in
// length^2 units; the S statistics still want the factor dr (apply it as `scale` in stat_contract), the U ones do not.
template <int N, bool LD>
UL_HD void shoot_col_t(const Lens& L, double wcx, double wcy, double rho2, double c, double s, double r0, double dr,
                       int n_r, double& U_out, double& S_out, TanStat<N>& SU, TanStat<N>& SS, bool& edge)
{
    double f1 = UL_BIG, f2 = UL_BIG;
    double U = 0.0, S = 0.0, U2 = 0.0;
    stat_zero(SU); stat_zero(SS);
    edge = false;
    int npend = 0, pi0 = 0, pi1 = 0;
    unsigned penb = 0;
    auto flush = [&](int pi, bool pen) {
        {
            double w[4];
            RayCore<N> R;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const double rk = r0 + dr * (pi - 3 + k + 0.5);
                ray_core<N>(L, rk * c, rk * s, wcx, wcy, rho2, R);
                w[k] = R.F;
            }
            const bool keep = -w[pen ? 2 : 1] > UL_DUAL_SING_FLOOR * rho2;
            enforce_crossing(w[1], w[2], pen);
            const double r1 = r0 + dr * (pi - 1.5);       // node pi - 2
            const double rh = r1 + 0.5 * dr;              // cell face between the pair
            const double rin = pen ? r1 + dr : r1;        // first inside node
            const double t2x = dr / ul_max(rin, 0.5 * dr);
            double u, dS, au[4], aS[4]; bool en;
            edge_event_adj(w[0], w[1], w[2], w[3], LD, keep, t2x, u, en, dS, au, aS);
            double rc = en ? (r1 + dr) - u * dr : r1 + u * dr;
            const bool rc_free = rc > 0.0;
            rc = ul_max(rc, 0.0);
            U2 += en ? 0.5 * (rh * rh - rc * rc) : 0.5 * (rc * rc - rh * rh);
            S += dS * rc;
            // d rc = -/+ dr du;  d U2 = rc dr du (either way);  d (dS rc) = rc d(dS) + dS d rc
            const double drc = rc_free ? (en ? -dr : dr) : 0.0;
#pragma unroll 1
            for (int k = 0; k < 4; ++k) {
                const double rk = r0 + dr * (pi - 3 + k + 0.5);
                RayBasis<N> B;
                ray_core<N>(L, rk * c, rk * s, wcx, wcy, rho2, R);
                ray_basis<N, true>(L, R, rk, c, s, B);
                stat_add(SU, rc_free ? rc * dr * au[k] : 0.0, B);
                if (LD) stat_add(SS, rc * aS[k] + dS * drc * au[k], B);          // (the caller scales the S set by dr)
            }
        }
    };
    for (int i = -2; i <= n_r + 3; ++i) {                 // (last two passes: resolve the noted events)
        const bool last = i > n_r + 1;
        const double r = r0 + dr * (i + 0.5);
        RayCore<N> R;
        ray_core<N>(L, r * c, r * s, wcx, wcy, rho2, R);
        const double f3 = last ? UL_BIG : R.F;
        if (i >= 0 && i < n_r && f3 < 0.0) {
            U += r;
            if (LD) {
                const double rs = ul_rsqrt(-f3);
                S += r * (-f3 * rs);
                RayBasis<N> B;
                ray_basis<N, true>(L, R, r, c, s, B);
                stat_add(SS, (-f3 > UL_DUAL_SING_FLOOR * rho2) ? -0.5 * r * rs : 0.0, B);
            }
            if ((i < 2 && r0 > 0.0) || i >= n_r - 2) edge = true;
        }
        // pair (i-2, i-1) = (f1, f2); the cell face between the pair must lie at r > 0
        const bool ev = !last && i >= 1 && ((f1 < 0.0) != (f2 < 0.0)) && (r0 + dr * (i - 1.0) > 0.0);
        if (npend > 0 && (last || (ev && npend == 2))) {
            flush(pi0, (penb & 1u) != 0);
            pi0 = pi1; penb >>= 1; --npend;
        }
        if (ev) {
            if (npend == 0) pi0 = i; else pi1 = i;
            if (!(f1 < 0.0)) penb |= 1u << npend;
            ++npend;
        }
        f1 = f2; f2 = f3;
    }
    U_out = U * dr + U2; S_out = S * dr;
}

// line_node of ulens_core.cuh for a span [x0, x0 + n dx] that moves with the parameters
template <int NT>
UL_HD void line_node_d(int flags, int n, int line, const Dual<NT>& x0, const Dual<NT>& dx, Dual<NT>& x, Dual<NT>& w)
{
    if (flags & UL_PATCH_SINR) {
        double ph = (line + 0.5) * (UL_PI / n), sn = sin(ph), cs = cos(ph);
        Dual<NT> h = dx * (0.5 * n);
        x = x0 + h * (1.0 - cs);
        w = h * (sn * (UL_PI / n));
    } else { x = x0 + dx * (line + 0.5); w = dx; }
}

// d z / d p_m of an image point z of the limb point w_c + rho e^{i phi}: Eq. 1 differentiated at fixed phi,
// dz + g conj(dz) = b_m,  b_m = dw_c + drho e^{i phi} + sum_i [ deps_i / conj(d_i) + eps_i conj(da_i) / conj(d_i)^2 ]
// => dz = (b - g conj(b)) / (1 - |g|^2)   (P:163-175 by the implicit-function theorem, here on Eq. 1 itself).
// Returns d|z|/dp_m in out[m] (and d arg z/dp_m in out_theta[m]); the tangents are capped (they only have to
// follow the edge).
template <int N, int NT>
UL_HD void limb_point_rdot(const Lens& L, const TangentTable& T, double zx, double zy, double phi, double* out,
                           double* out_theta = nullptr)
{
    double gx = 0.0, gy = 0.0, px[N], py[N], qx[N], qy[N];
#pragma unroll
    for (int i = 0; i < N; ++i) {
        double dx = zx - L.ax[i], dy = zy - L.ay[i];
        double inv = 1.0 / (dx * dx + dy * dy);
        px[i] = dx * inv; py[i] = dy * inv;
        qx[i] = px[i] * px[i] - py[i] * py[i]; qy[i] = 2.0 * px[i] * py[i];
        gx += L.eps[i] * qx[i]; gy += L.eps[i] * qy[i];
    }
    double det = 1.0 - (gx * gx + gy * gy);
    double rr = sqrt(zx * zx + zy * zy);
    double cp = cos(phi), sp = sin(phi);
#pragma unroll 1
    for (int k = 0; k < NT; ++k) {
        double bx = T.dwx[k] + T.drho[k] * cp, by = T.dwy[k] + T.drho[k] * sp;
#pragma unroll
        for (int i = 0; i < N; ++i) {
            bx += T.deps[k][i] * px[i]; by += T.deps[k][i] * py[i];
            // eps_i conj(da_i) / conj(d_i)^2 = eps_i (dax - i day)(qx + i qy)
            bx += L.eps[i] * (T.dax[k][i] * qx[i] + T.day[k][i] * qy[i]);
            by += L.eps[i] * (T.dax[k][i] * qy[i] - T.day[k][i] * qx[i]);
        }
        // g conj(b)
        double hx = gx * bx + gy * by, hy = gy * bx - gx * by;
        double dzx = (bx - hx) / det, dzy = (by - hy) / det;
        double v = rr > 0.0 ? (zx * dzx + zy * dzy) / rr : 0.0;
        if (!(fabs(v) < 1e3)) v = 0.0;                            // on a critical curve: give up following
        if (out) out[k] = v;
        if (out_theta) {
            double tv = rr > 0.0 ? (zx * dzy - zy * dzx) / (rr * rr) : 0.0;
            if (!(fabs(tv) < 1e3)) tv = 0.0;
            out_theta[k] = tv;
        }
    }
}

}  // namespace ulens
