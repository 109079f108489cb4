// ulens_dual.cuh -- forward-mode (dual-number) variant of the ray-shooting integrator (step a8).
//
// PAPER.md Sec. 3.5: derivatives of the magnification by forward-mode differentiation THROUGH
// the region construction and the quadrature. What is differentiated here is the discrete rule of
// ulens_core.cuh with the inside flags piecewise constant:
//   * the radial grid of a sector moves with the image: r0 and dr carry tangents obtained from the extreme
//     image-limb points by implicit differentiation of Eq. 1 (P:163-175 uses the polynomial; the lens
//     equation itself is better conditioned) -- without this the square-root behaviour of the chord
//     length at the radial ends of an image ruins the derivative;
//   * every ray carries dF/dp_k for the NT = 5 intrinsic directions p = (w_cx, w_cy, s, q, rho): grid motion
//     + explicit dependence of Eq. 1 on the lens parameters + the source centre / radius;
//   * the edge position from the cubic, the uniform weight u - 1/2 and the square-root end correction
//     (Hurwitz zetas) are evaluated in dual arithmetic, so the edge-motion (Reynolds boundary) term is exact
//     for the rule and the paper's sigmoid surrogate for the Heaviside function (Eq. 9) is not needed.
#pragma once
#include "ulens_core.cuh"

namespace ulens {

#define UL_NT 5          // tangent directions: w_cx, w_cy, s, q, rho

// how the inputs of Eq. 1 / Eq. 5 move in each direction (filled on the host per configuration by
// upload_tangents, whose structure -- which entries can be non-zero -- ray_F_dual relies on)
struct TangentTable {
    double dwx[UL_NT], dwy[UL_NT], drho[UL_NT];
    double deps[UL_NT][3], dax[UL_NT][3], day[UL_NT][3];
};

struct D5 {
    double v;
    double d[UL_NT];
};

UL_HD D5 d5_const(double a) { D5 r; r.v = a; for (int k = 0; k < UL_NT; ++k) r.d[k] = 0.0; return r; }
UL_HD D5 operator+(const D5& a, const D5& b) { D5 r; r.v = a.v + b.v; for (int k = 0; k < UL_NT; ++k) r.d[k] = a.d[k] + b.d[k]; return r; }
UL_HD D5 operator-(const D5& a, const D5& b) { D5 r; r.v = a.v - b.v; for (int k = 0; k < UL_NT; ++k) r.d[k] = a.d[k] - b.d[k]; return r; }
UL_HD D5 operator-(const D5& a) { D5 r; r.v = -a.v; for (int k = 0; k < UL_NT; ++k) r.d[k] = -a.d[k]; return r; }
UL_HD D5 operator+(const D5& a, double b) { D5 r = a; r.v += b; return r; }
UL_HD D5 operator-(const D5& a, double b) { D5 r = a; r.v -= b; return r; }
UL_HD D5 operator+(double b, const D5& a) { D5 r = a; r.v += b; return r; }
UL_HD D5 operator-(double b, const D5& a) { D5 r; r.v = b - a.v; for (int k = 0; k < UL_NT; ++k) r.d[k] = -a.d[k]; return r; }
UL_HD D5 operator*(const D5& a, const D5& b) { D5 r; r.v = a.v * b.v; for (int k = 0; k < UL_NT; ++k) r.d[k] = a.d[k] * b.v + a.v * b.d[k]; return r; }
UL_HD D5 operator*(const D5& a, double b) { D5 r; r.v = a.v * b; for (int k = 0; k < UL_NT; ++k) r.d[k] = a.d[k] * b; return r; }
UL_HD D5 operator*(double b, const D5& a) { return a * b; }
UL_HD D5 operator/(const D5& a, const D5& b)
{
    D5 r; double ib = 1.0 / b.v; r.v = a.v * ib;
    for (int k = 0; k < UL_NT; ++k) r.d[k] = (a.d[k] - r.v * b.d[k]) * ib;
    return r;
}
UL_HD D5 d5_sqrt(const D5& a)
{
    D5 r; r.v = sqrt(a.v); double h = 0.5 / r.v;
    for (int k = 0; k < UL_NT; ++k) r.d[k] = a.d[k] * h;
    return r;
}
UL_HD D5& operator+=(D5& a, const D5& b) { a.v += b.v; for (int k = 0; k < UL_NT; ++k) a.d[k] += b.d[k]; return a; }

// zeta(-1/2, u), zeta(-3/2, u) of ulens_core.cuh in dual arithmetic (same coefficients, same fit)
UL_HD D5 zeta_m12_d(const D5& u)
{
    const double c[10] = {-0.207886224314425946, -0.730177387536053191, -0.326542433690562406,
                          0.0837832566266219698, -0.0435998186937335486, 0.0271396135617846347,
                          -0.0165300041688832568, 0.00823252937110980637, -0.00274063185833692022,
                          0.000434876090612478912};
    double p = c[9], dp = 0.0;
    for (int i = 8; i >= 0; --i) { dp = dp * u.v + p; p = p * u.v + c[i]; }
    D5 r; double su = sqrt(u.v);
    r.v = su + p;
    // d sqrt(u)/du is singular at u = 0 (a node exactly on the edge: the rule is not differentiable there): dropped
    double g = (u.v > 1e-8 ? 0.5 / su : 0.0) + dp;
    for (int k = 0; k < UL_NT; ++k) r.d[k] = g * u.d[k];
    return r;
}
UL_HD D5 zeta_m32_d(const D5& u)
{
    const double c[10] = {-0.0254852020522020475, -0.311829304876540199, -0.547634035662697937,
                          -0.163258961591498412, 0.0313415948971861593, -0.0127998326381573904,
                          0.00616325441161647825, -0.00268571587959467142, 0.000828839924548779593,
                          -0.0001258385180165005};
    double p = c[9], dp = 0.0;
    for (int i = 8; i >= 0; --i) { dp = dp * u.v + p; p = p * u.v + c[i]; }
    D5 r; double su = sqrt(u.v);
    r.v = u.v * su + p;
    double g = 1.5 * su + dp;
    for (int k = 0; k < UL_NT; ++k) r.d[k] = g * u.d[k];
    return r;
}

// F(z) = |w(z) - w_c|^2 - rho^2 with its tangents. The ray sits at z = r (c, s), r = r.v with tangent r.d[k]
// (co-moving grid); along a radial scan line c, s are constants, along a ring they rotate -- either way
// dz_k = r.d[k] (c, s). Explicit dependences: -d w_c, -d eps_i / conj(z - a_i), -eps_i conj(d a_i) / conj(z - a_i)^2
// and, through the moving ray, dw = dz + g conj(dz) (Eq. 1 differentiated; g = sum eps_i / conj(z - a_i)^2).
template <int N>
UL_HD D5 ray_F_dual(const Lens& L, const TangentTable& T, const D5& r, double c, double s, double wcx, double wcy,
                    double rho, const double* thdot = nullptr)
{
    // The five directions have a fixed structure (upload_tangents in ulens_api.cu is the only writer of T):
    //   k = 0, 1  source centre: dw_c = 1, i            k = 4  rho
    //   k = 2     s: real displacements da_i = T.dax[2][i]
    //   k = 3     q: d eps_i = T.deps[3][i] and real displacements da_i = T.dax[3][i]
    // so per ray: g once, the moving-ray response h = e + g conj(e) once (e = unit vector of the line), and two
    // explicit lens-parameter terms; every tangent is then one FMA on top of the value's reciprocals.
    const double x = r.v * c, y = r.v * s;
    double ex = x - wcx, ey = y - wcy;
    double gx = 0.0, gy = 0.0, s2x = 0.0, s2y = 0.0, s3x = 0.0, s3y = 0.0;
#pragma unroll
    for (int i = 0; i < N; ++i) {
        double dx = x - L.ax[i], dy = y - L.ay[i];
        double inv = 1.0 / (dx * dx + dy * dy);
        double px = dx * inv, py = dy * inv;                      // 1/conj(d) = d/|d|^2
        double qx = px * px - py * py, qy = 2.0 * px * py;        // 1/conj(d)^2
        ex -= L.eps[i] * px; ey -= L.eps[i] * py;
        gx += L.eps[i] * qx; gy += L.eps[i] * qy;
        if (N > 1) {
            // - d eps_i / conj(d_i)  -  eps_i conj(d a_i) / conj(d_i)^2     (Eq. 1 differentiated at fixed z)
            const double e2 = L.eps[i] * T.dax[2][i], e3 = L.eps[i] * T.dax[3][i];
            s2x -= e2 * qx; s2y -= e2 * qy;
            s3x -= T.deps[3][i] * px + e3 * qx; s3y -= T.deps[3][i] * py + e3 * qy;
        }
    }
    D5 F;
    F.v = ex * ex + ey * ey - rho * rho;
    const double ex2 = 2.0 * ex, ey2 = 2.0 * ey;
    // dz = a (c, s): dz + g conj(dz) = a h
    const double H = ex2 * (c + gx * c + gy * s) + ey2 * (s + gy * c - gx * s);
    const double expl[UL_NT] = {-ex2, -ey2, ex2 * s2x + ey2 * s2y, ex2 * s3x + ey2 * s3y, -2.0 * rho};
#pragma unroll
    for (int k = 0; k < UL_NT; ++k) F.d[k] = r.d[k] * H + expl[k];
    if (thdot) {                                                  // the scan line itself turns: dz += r thdot (-s, c)
        const double Hp = r.v * (ex2 * (-s - gx * s + gy * c) + ey2 * (c - gy * s - gx * c));
#pragma unroll
        for (int k = 0; k < UL_NT; ++k) F.d[k] += thdot[k] * Hp;
    }
    if (!(F.v < UL_BIG)) { F = d5_const(UL_BIG); }               // ray on a lens: outside, never NaN
    return F;
}

// edge_event of ulens_core.cuh in dual arithmetic: u and dS carry the tangents of the edge position
// (implicit differentiation of the cubic's root comes for free from Newton's iteration on dual numbers).
UL_HD void edge_event_d(const D5& f0, const D5& f1, const D5& f2, const D5& f3, bool want_S, double t2_extra,
                        D5& u, bool& entering, D5& dS)
{
    D5 c0 = f1;
    D5 c1 = (f0 * -2.0 - f1 * 3.0 + f2 * 6.0 - f3) * (1.0 / 6.0);
    D5 c2 = (f0 - f1 * 2.0 + f2) * 0.5;
    D5 c3 = (f1 * 3.0 - f0 - f2 * 3.0 + f3) * (1.0 / 6.0);
    D5 x = f1 / (f1 - f2);
    D5 xl = x;
    bool cubic_ok = true;
#pragma unroll 1
    for (int it = 0; it < 5; ++it) {
        D5 p = c0 + x * (c1 + x * (c2 + x * c3));
        D5 dp = c1 + x * (c2 * 2.0 + x * c3 * 3.0);
        D5 xn = x - p / dp;
        if (!(xn.v >= 0.0 && xn.v <= 1.0)) { cubic_ok = false; break; }
        x = xn;
    }
    D5 dp, d2p;
    if (cubic_ok) {
        dp = c1 + x * (c2 * 2.0 + x * c3 * 3.0);
        d2p = c2 * 2.0 + x * c3 * 6.0;
    } else {
        x = xl;
        dp = f2 - f1; d2p = d5_const(0.0);
    }
    entering = !(f1.v < 0.0);
    u = entering ? (1.0 - x) : x;
    dS = d5_const(0.0);
    if (want_S) {
        D5 sigma = entering ? -dp : dp;
        D5 tau = d2p * -0.5;
        if (sigma.v > 0.0) {
            D5 ss = d5_sqrt(sigma);
            D5 corr = ss * zeta_m12_d(u);
            D5 t2 = tau / (sigma * 2.0) + (entering ? t2_extra : -t2_extra);
            if (fabs(t2.v) < 0.5) corr += ss * t2 * zeta_m32_d(u);
            dS = -corr;
        }
    }
}

// Edge events in the dual loops are DEFERRED and BATCHED. An event costs ~600 instructions in D5 arithmetic and each
// of the 32 lines of a work unit meets the image edge at its own node: evaluated on the spot, 1-2 lanes were
// active in edge_event_d and the events took two thirds of the kernel (ncu: 15 of 32 lanes active on average).
// Now the loop keeps only the VALUES of the 4-node window; a lane that sees a sign change remembers the node
// index, and the warp evaluates all pending events together -- at the latest UL_DEFER_D nodes later, or when one of the lanes meets its next crossing --
// recomputing the four window rays with their tangents (4 ray_F_dual, also batched).
#ifndef UL_DEFER_D
#define UL_DEFER_D 32
#endif

// The recomputed window may differ from the loop's values in the last bit (another rounding path), which can flip
// the sign of a node sitting exactly on the edge: the loop's classification (entering: node 1 outside, node 2
// inside) is authoritative, a disagreeing node is moved onto the edge.
UL_HD void enforce_crossing(D5& w1, D5& w2, bool entering)
{
    if (entering) { if (w1.v < 0.0) w1.v = 0.0; if (!(w2.v < 0.0)) w2.v = -1e-9 * fabs(w1.v) - 1e-300; }
    else { if (!(w1.v < 0.0)) w1.v = -1e-9 * fabs(w2.v) - 1e-300; if (w2.v < 0.0) w2.v = 0.0; }
}

// shoot_ring of ulens_core.cuh with tangents. r = ring radius (dual); theta grid frozen.
template <int N, bool LD>
UL_HD void shoot_ring_d(const Lens& L, const TangentTable& T, double wcx, double wcy, double rho, const D5& r,
                        double th0, double dth, int n_th, bool periodic, D5& U_out, D5& S_out, bool& edge)
{
    double cd = cos(dth), sd = sin(dth);
    double t = th0 - 1.5 * dth;
    double c = cos(t), s = sin(t);
    double f0 = UL_BIG, f1 = UL_BIG, f2 = UL_BIG;
    D5 U = d5_const(0.0), S = d5_const(0.0);
    edge = false;
    const int j_first = periodic ? 2 : 1;
    bool pend = false, pen = false; int pj = 0;
    auto flush = [&]() {
        if (pend) {
            // window nodes pj-3 .. pj at angles th0 + (k + 1/2) dth
            double a = th0 + (pj - 2.5) * dth, wc = cos(a), ws = sin(a);
            D5 w[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                w[k] = ray_F_dual<N>(L, T, r, wc, ws, wcx, wcy, rho);
                double cn = wc * cd - ws * sd; ws = ws * cd + wc * sd; wc = cn;
            }
#ifdef UL_DEBUG_FLUSH
            printf("ring flush pj %d pen %d w %.6g %.6g %.6g %.6g  loop f1 f2 ? r %.12g\n", pj, (int)pen, w[0].v, w[1].v, w[2].v, w[3].v, r.v);
#endif
            enforce_crossing(w[1], w[2], pen);
            D5 u, dS; bool en;
            edge_event_d(w[0], w[1], w[2], w[3], LD, 0.0, u, en, dS);
#ifdef UL_DEBUG_FLUSH
            printf("   u %.6g du0 %.6g dS %.6g dS0 %.6g\n", u.v, u.d[0], dS.v, dS.d[0]);
#endif
            U += u - 0.5; S += dS;
            pend = false;
        }
    };
    for (int j = -2; j <= n_th + 1; ++j) {
        D5 f3 = ray_F_dual<N>(L, T, r, c, s, wcx, wcy, rho);
        if (j >= 0 && j < n_th && f3.v < 0.0) {
            U.v += 1.0;
            if (LD) S += d5_sqrt(-f3);
            if (!periodic && (j < 2 || j >= n_th - 2)) edge = true;
        }
        const bool ev = j >= j_first && ((f1 < 0.0) != (f2 < 0.0));
        // flush for the whole warp when a pending event is old enough or its lane meets its next crossing
        if (UL_WARP_ANY(pend && (ev || j - pj >= UL_DEFER_D))) flush();
        if (ev) { pj = j; pend = true; pen = !(f1 < 0.0); }
        f0 = f1; f1 = f2; f2 = f3.v;
        double cn = c * cd - s * sd;
        s = s * cd + c * sd;
        c = cn;
    }
    flush();
    (void)f0;
    U_out = U; S_out = S;
}

// shoot_col of ulens_core.cuh with tangents: radial line at fixed theta, nodes r0 + (i + 1/2) dr with dual r0, dr.
template <int N, bool LD>
UL_HD void shoot_col_d(const Lens& L, const TangentTable& T, double wcx, double wcy, double rho, const D5& th,
                       const D5& r0, const D5& dr, int n_r, D5& U_out, D5& S_out, bool& edge)
{
    double c = cos(th.v), s = sin(th.v);
    double f0 = UL_BIG, f1 = UL_BIG, f2 = UL_BIG;
    D5 U = d5_const(0.0), S = d5_const(0.0), U2 = d5_const(0.0);
    edge = false;
    bool pend = false, pen = false; int pi = 0;
    auto flush = [&]() {
        if (pend) {
            D5 w[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) w[k] = ray_F_dual<N>(L, T, r0 + dr * (pi - 3 + k + 0.5), c, s, wcx, wcy, rho, th.d);
            enforce_crossing(w[1], w[2], pen);
            D5 r1 = r0 + dr * (pi - 1.5);
            D5 rh = r1 + dr * 0.5;
            D5 u, dS; bool en;
            bool ent = pen;
            D5 rin = ent ? r1 + dr : r1;
            double t2x = dr.v / ul_max(rin.v, 0.5 * dr.v);
            edge_event_d(w[0], w[1], w[2], w[3], LD, t2x, u, en, dS);
            D5 rc = en ? (r1 + dr) - u * dr : r1 + u * dr;
            if (rc.v < 0.0) rc = d5_const(0.0);
            U2 += en ? (rh * rh - rc * rc) * 0.5 : (rc * rc - rh * rh) * 0.5;
            S += dS * rc;
            pend = false;
        }
    };
    for (int i = -2; i <= n_r + 1; ++i) {
        D5 r = r0 + dr * (i + 0.5);
        D5 f3 = ray_F_dual<N>(L, T, r, c, s, wcx, wcy, rho, th.d);
        if (i >= 0 && i < n_r && f3.v < 0.0) {
            U += r;
            if (LD) S += r * d5_sqrt(-f3);
            if ((i < 2 && r0.v > 0.0) || i >= n_r - 2) edge = true;
        }
        // pair (i-2, i-1) = (f1, f2); the cell face between the pair must lie at r > 0
        const bool ev = i >= 1 && ((f1 < 0.0) != (f2 < 0.0)) && (r0.v + dr.v * (i - 1.0) > 0.0);
        if (UL_WARP_ANY(pend && (ev || i - pi >= UL_DEFER_D))) flush();
        if (ev) { pi = i; pend = true; pen = !(f1 < 0.0); }
        f0 = f1; f1 = f2; f2 = f3.v;
    }
    flush();
    (void)f0;
    U_out = U * dr + U2; S_out = S * dr;
}

// line_node of ulens_core.cuh for a span [x0, x0 + n dx] that moves with the parameters
UL_HD void line_node_d(int flags, int n, int line, const D5& x0, const D5& dx, D5& x, D5& w)
{
    if (flags & UL_PATCH_SINR) {
        double ph = (line + 0.5) * (UL_PI / n), sn = sin(ph), cs = cos(ph);
        D5 h = dx * (0.5 * n);
        x = x0 + h * (1.0 - cs);
        w = h * (sn * (UL_PI / n));
    } else { x = x0 + dx * (line + 0.5); w = dx; }
}

// d z / d p_k of an image point z of the limb point w_c + rho e^{i phi}: Eq. 1 differentiated at fixed phi,
// dz + g conj(dz) = b_k,  b_k = dw_c + drho e^{i phi} + sum_i [ deps_i / conj(d_i) + eps_i conj(da_i) / conj(d_i)^2 ]
// => dz = (b - g conj(b)) / (1 - |g|^2)   (P:163-175 by the implicit-function theorem, here on Eq. 1 itself).
// Returns d|z|/dp_k in out[k]; the tangents are capped (they only have to follow the edge).
template <int N>
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
#pragma unroll
    for (int k = 0; k < UL_NT; ++k) {
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
