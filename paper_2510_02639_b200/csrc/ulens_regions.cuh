// ulens_regions.cuh -- image-region (sector) builder, second half: polar (r, theta) boxes of the image-limb
// arcs -> 1-D interval grouping in r and theta -> sectors with margins and a ray grid sized from the local
// image scale.   PAPER.md Sec. 3.2; readings G2, G8 in DESIGN.md.
//
// The first half (Eq. 8 limb sampling, warm-started Ehrlich-Aberth, Eq.-1 polish, one box per image arc) is
// k_limb in ulens_limb.cuh: a CTA per source point, a group of N^2+1 lanes per limb arc, one lane per root.
// This file holds the box helpers both halves use and the per-point sector construction (k_sectors, one
// THREAD per source point; plain C++, so tests/host_logic.cpp runs it on the CPU):
//   boxes -> disjoint r-groups (interval union); inside each r-group its member boxes -> periodic theta-groups;
//   every occupied (r-group, theta-group) cell becomes one sector ("all combinations of radial and
//   angular bins ... empty sectors are discarded, periodic ones merged"), refined to the min/max of its
//   members plus a margin, with n_r x n_theta from the local image scale.
#pragma once
#include "ulens_core.cuh"
#include "ulens_dual.cuh"

namespace ulens {

struct SubBox {
    double r_lo, r_hi;      // r_lo > r_hi: empty
    double t_lo, t_hi;      // unwrapped theta interval, t_lo in [-pi, pi), t_hi - t_lo <= 2 pi
    double hr, ht;          // smallest local half-extent (projection) of the image in r / along theta: scan-line spacing
    double cr, ct;          // smallest local half-chord of the image along r / along theta: node spacing on a line
};

#ifndef UL_EA_LIMB_TOL2
#define UL_EA_LIMB_TOL2 1e-8    // squared relative step at which a limb root is settled (the Eq.-1 polish follows)
#endif
#define UL_MAXP 12          // sector cap per point ("capped based on the maximum expected number of images")
#define UL_MAXG 16          // groups per axis
#define UL_MAXG_TMP 64      // ... while the boxes are still arriving: disjoint groups form first and are bridged later

struct RegionParams {
    int n_limb;             // multiple of 32
    int n_r, n_theta;       // rays per image half-extent
    int max_nr, max_nth;    // caps per sector
    int max_units_pt;       // cap on 32-ring units per point
};

// dual variant only: the box's own image-limb points of smallest / largest |z| and their limb angles
struct BoxExt {
    double lo_r, lo_x, lo_y, lo_ph;
    double hi_r, hi_x, hi_y, hi_ph;
    double tlo_t, tlo_x, tlo_y, tlo_ph;     // smallest / largest unwrapped theta along the arc
    double thi_t, thi_x, thi_y, thi_ph;
};

// dual variant only: how a sector's radial bounds move (d r_lo / d p_k, d r_hi / d p_k)
struct PatchTan {
    double rlo_dot[UL_NT_MAX], rhi_dot[UL_NT_MAX];
    double tlo_dot[UL_NT_MAX], thi_dot[UL_NT_MAX];
};

// boxes per source point in the k_limb -> k_sectors buffer: one per (arc, root slot) plus room for arcs that split
template <int N> struct BoxCap { static constexpr int value = (N == 1) ? 96 : (N == 2) ? 192 : 384; };

UL_HD double wrap_pi(double a)      // to (-pi, pi]
{
    if (a > UL_PI) a -= 2.0 * UL_PI;
    else if (a <= -UL_PI) a += 2.0 * UL_PI;
    return a;
}

// add an image-limb point to a slot box (polar coordinates about the origin, G8)
UL_HDNI void box_add(SubBox& b, double& t_cur, double r, double th, double hr, double ht, double cr, double ct, bool advance)
{
    if (b.r_lo > b.r_hi) {               // first point
        b.r_lo = b.r_hi = r; b.t_lo = b.t_hi = th; b.hr = hr; b.ht = ht; b.cr = cr; b.ct = ct; t_cur = th;
        return;
    }
    double d = th - t_cur;
    d -= 2.0 * UL_PI * rint(d / (2.0 * UL_PI));       // nearest equivalent angle: continuous along the boundary
    double t = t_cur + d;
    b.r_lo = ul_min(b.r_lo, r); b.r_hi = ul_max(b.r_hi, r);
    b.t_lo = ul_min(b.t_lo, t); b.t_hi = ul_max(b.t_hi, t);
    b.hr = ul_min(b.hr, hr); b.ht = ul_min(b.ht, ht); b.cr = ul_min(b.cr, cr); b.ct = ul_min(b.ct, ct);
    if (advance) t_cur = t;
}

// extreme of the parabola through three consecutive boundary samples (x = limb angle, y = r or theta), if the
// middle sample is a local extreme: the image boundary bulges beyond its samples by ~ (step)^2 / 8 x curvature,
// which matters now that the sector margins are tight
UL_HDNI bool parabola_vertex(double x0, double y0, double x1, double y1, double x2, double y2, double& yv)
{
    if (!((y1 >= y0 && y1 >= y2) || (y1 <= y0 && y1 <= y2))) return false;
    double h0 = x1 - x0, h1 = x2 - x1;
    if (!(h0 > 0.0 && h1 > 0.0)) return false;
    double s0 = (y1 - y0) / h0, s1 = (y2 - y1) / h1;
    double a = (s1 - s0) / (h0 + h1);
    if (a == 0.0) return false;
    double slope1 = s0 + a * h0;                         // derivative at x1
    double dx = -slope1 / (2.0 * a);
    if (!(dx >= -h0 && dx <= h1)) return false;
    yv = y1 - slope1 * slope1 / (4.0 * a);
    return true;
}

// local image scale at an image point z with g = sum eps_i/conj(z-a_i)^2: the image of a small disk of
// radius rho is an ellipse with semi-axes rho/(1+|g|) (along arg(g)/2) and rho/|1-|g|| (perpendicular);
// hr, ht = its half-extents (projections) along the radial / azimuthal direction at z; cr, ct = its
// half-chords through the centre along those directions.
// (single precision: the extents only size the ray grid and the box margins)
UL_HDNI void local_extents(double zx, double zy, double gx, double gy, double rho, double& hr, double& ht,
                         double& cr, double& ct)
{
    const float fgx = (float)gx, fgy = (float)gy, fzx = (float)zx, fzy = (float)zy, frho = (float)rho;
    const float ga = sqrtf(fgx * fgx + fgy * fgy);
    const float m = frho / (1.0f + ga);
    const float den = fabsf((float)(1.0 - sqrt(gx * gx + gy * gy)));     // 1 - |g| in double: |g| -> 1 on a critical curve
    const float M = den > 1e-6f ? frho / den : frho * 1e6f;
    const float z2 = fzx * fzx + fzy * fzy;
    float c2 = 0.0f;                                     // cos(2 phi), phi = angle(major axis) - angle(radial)
    if (ga > 1e-30f && z2 > 1e-30f) {
        // Re(g conj(z)^2) / (|g||z|^2) = cos(arg g - 2 theta);  major axis at arg(g)/2 + pi/2
        const float re = fgx * (fzx * fzx - fzy * fzy) + fgy * (2.0f * fzx * fzy);
        c2 = -re / (ga * z2);
        c2 = c2 > 1.0f ? 1.0f : (c2 < -1.0f ? -1.0f : c2);
    }
    const float cc = 0.5f * (1.0f + c2), ss = 0.5f * (1.0f - c2);
    const float M2 = M * M, m2 = m * m;
    hr = (double)sqrtf(M2 * cc + m2 * ss);
    ht = (double)sqrtf(M2 * ss + m2 * cc);
    cr = (double)(1.0f / sqrtf(cc / M2 + ss / m2));
    ct = (double)(1.0f / sqrtf(ss / M2 + cc / m2));
}

// margins applied to every box before grouping: a quarter of the local minor scale in both directions
// plus 2 % of the box itself (boundary bulge between limb samples)
UL_HD void box_expanded(const SubBox& b, double& rl, double& rh, double& tl, double& th)
{
    double m = ul_min(b.cr, b.ct);
    // radial margin: TIGHT (0.5 % of the local width + 0.04 % of the box). The rings of a sector are placed
    // at Chebyshev-like radii r_c + h sin(phi) (emit_patch), which removes the square-root behaviour of the
    // chord length at the radial ends of an image only if the sector ends where the image ends.
    double mr = 0.02 * (0.25 * m + 0.02 * (b.r_hi - b.r_lo));
    double rmid = ul_max(0.5 * (b.r_lo + b.r_hi), 1e-300);
    double mt = 0.02 * (0.25 * m / rmid + 0.02 * (b.t_hi - b.t_lo));   // tight, as in r
    mt = ul_min(mt, 0.5);
    rl = ul_max(b.r_lo - mr, 0.0); rh = b.r_hi + mr;
    tl = b.t_lo - mt; th = b.t_hi + mt;
}

// dual variant: tangents of a sector's radial bounds from its extreme image-limb points
template <int N>
UL_HD void patch_tangents(const Lens& L, const TangentTable& T, const BoxExt& x, bool from_origin, PatchTan& out)
{
    constexpr int NT = TanDirs<N>::NT;
    for (int k = 0; k < UL_NT_MAX; ++k) { out.rlo_dot[k] = 0.0; out.rhi_dot[k] = 0.0; out.tlo_dot[k] = 0.0; out.thi_dot[k] = 0.0; }
    if (x.hi_r < 0.0) return;                           // no own point (links only): frozen
    if (!from_origin) limb_point_rdot<N, NT>(L, T, x.lo_x, x.lo_y, x.lo_ph, out.rlo_dot);
    limb_point_rdot<N, NT>(L, T, x.hi_x, x.hi_y, x.hi_ph, out.rhi_dot);
    if (x.thi_t > -1e299 && !from_origin) {             // theta ends (used by sectors scanned along radial lines)
        limb_point_rdot<N, NT>(L, T, x.tlo_x, x.tlo_y, x.tlo_ph, nullptr, out.tlo_dot);
        limb_point_rdot<N, NT>(L, T, x.thi_x, x.thi_y, x.thi_ph, nullptr, out.thi_dot);
    }
}

// Forward-mode runs: a sector bound moves like the image's extreme point (envelope theorem: d r_max / dp is dr/dp at
// fixed limb angle, taken AT the extreme), and the ray grid must follow the image closely -- the quadrature error is a
// function of where the edge falls between the scan lines, and its derivative is not small. The extreme among the limb
// SAMPLES is off by up to half a sample spacing, which leaves a first-order error in the bound's tangent (measured on
// C4: dA/du0, dA/drho, dA/dalpha converged like 1/n_limb). So the sampled extreme of |z| (which = 0) or arg z
// (which = 1) is moved along the limb to the true one (kind = +1: maximum, -1: minimum): secant iteration on d/dphi of
// the quantity, the image z(phi) followed by Newton on Eq. 1 (dz/dphi by the implicit-function theorem, as
// limb_point_rdot). dph: the local sample spacing at most; the search stays within it. Returns false (nothing changed)
// if the image is lost, the search leaves the range, or the result is less extreme than the sample.
template <int N>
UL_HD bool refine_extreme(const Lens& L, double wcx, double wcy, double rho, int which, int kind, double dph,
                          double& x, double& y, double& ph, bool from_sample = true)
{
    // f = d(|z| or arg z)/dphi up to a positive factor
    auto slope = [&](double phi, double& zx, double& zy, double& f) -> bool {
        const double sn = sin(phi), cs = cos(phi);
        double detJ, resid, gx, gy;
        if (!polish_image_ni<N>(L, wcx + rho * cs, wcy + rho * sn, zx, zy, 8, 1e-11, detJ, resid, gx, gy)) return false;
        const double bx = -rho * sn, by = rho * cs;                       // dw/dphi
        const double vx = bx - (gx * bx + gy * by), vy = by - (gy * bx - gx * by);      // det J dz/dphi
        f = (which == 0 ? zx * vx + zy * vy : zx * vy - zy * vx) / detJ;
        return f == f && fabs(f) < 1e300;
    };
    double x0 = x, y0 = y, p0 = ph, f0;
    if (!slope(p0, x0, y0, f0)) return false;
    if (f0 == 0.0) return false;
    // second point on the side the slope points to
    double p1 = p0 + ((kind * f0 > 0.0) ? 0.25 : -0.25) * dph, x1 = x0, y1 = y0, f1;
    if (!slope(p1, x1, y1, f1)) return false;
    for (int it = 0; it < 4; ++it) {
        const double df = f1 - f0;
        if (!(fabs(df) > 0.0)) break;
        const double pn = p1 - f1 * (p1 - p0) / df;
        if (!(fabs(pn - ph) <= dph)) return false;
        p0 = p1; f0 = f1; x0 = x1; y0 = y1;
        p1 = pn;
        if (!slope(p1, x1, y1, f1)) return false;
        if (fabs(p1 - p0) < 1e-6 * dph) break;            // the tangent's error is first order in this
    }
    const double mv2 = (x1 - x) * (x1 - x) + (y1 - y) * (y1 - y);
    if (!(mv2 <= 0.01 * ul_max(x * x + y * y, 0.04))) return false;       // jumped to another image
    if (from_sample) {                                   // (a start that is only a prediction may lie beyond the true extreme)
        if (which == 0) { if (kind * (sqrt(x1 * x1 + y1 * y1) - sqrt(x * x + y * y)) < 0.0) return false; }
        else { if (kind * (x * y1 - y * x1) < 0.0) return false; }         // sign of the turn from the sample to the result
    }
    x = x1; y = y1; ph = p1;
    return true;
}

// "more extreme" with a total order: boxes arrive in any order, and two boxes that share a limb point (the end of one arc is the
// start of the next) can hold the same extreme value to the last bit with coordinates that differ in theirs
UL_HD bool ext_before(double v, double ph, double x, double v0, double ph0, double x0)
{
    return v < v0 || (v == v0 && (ph < ph0 || (ph == ph0 && x < x0)));
}

// Quiet points: the image around a centre image z_c is close to the Jacobian ellipse z_c + rho (e^{i phi} - g e^{-i phi}) / D,
// D = 1 - |g|^2, whose extremes along the radial direction n = z_c/|z_c| and across it are known in closed form:
//   Re(conj(n) dz) D / rho = Re((conj(n) - n conj(g)) e^{i phi}),   Im(conj(n) dz) D / rho = Im((conj(n) + n conj(g)) e^{i phi}).
// From those limb angles the four TRUE extremes of the image are found by refine_extreme (Newton on Eq. 1 along the limb).
// With them a sector ends exactly where its image ends, which is what the sin-spaced lines across it want: the bounds from
// the limb samples are good to ~1e-3 of the image and carry a safety margin of 0.5 %, and that offset -- not the number of
// lines -- is what limits the rule on a smooth image. Returns false (nothing usable) if any of the four is not found.
template <int N>
UL_HD bool quiet_image_extremes(const Lens& L, double wcx, double wcy, double rho, double zcx, double zcy, BoxExt& x)
{
    double fx, fy, gx, gy, dm2;
    lens_resid<N>(L, zcx, zcy, wcx, wcy, fx, fy, gx, gy, dm2);
    const double D = 1.0 - (gx * gx + gy * gy);
    const double rc = sqrt(zcx * zcx + zcy * zcy);
    if (!(fabs(D) > 1e-3) || !(rc > 0.0)) return false;
    const double nx = zcx / rc, ny = zcy / rc;
    // n conj(g)
    const double ngx = nx * gx + ny * gy, ngy = ny * gx - nx * gy;
    // radial: q_r = conj(n) - n conj(g);  azimuthal: q_t = conj(n) + n conj(g)
    const double qrx = nx - ngx, qry = -ny - ngy, qtx = nx + ngx, qty = -ny + ngy;
    const double sgn = D > 0.0 ? 1.0 : -1.0;
    const double ph_r = -atan2(qry, qrx), ph_t = 0.5 * UL_PI - atan2(qty, qtx);
    bool ok = true;
    for (int e = 0; e < 4 && ok; ++e) {
        const int which = e >> 1, kind = (e & 1) ? -1 : +1;                 // r max, r min, theta max, theta min
        double ph = (which == 0 ? ph_r : ph_t) + ((kind * sgn > 0.0) ? 0.0 : UL_PI);
        const double c = cos(ph), sn = sin(ph);
        // dz = rho (e^{i phi} - g e^{-i phi}) / D
        double px = zcx + rho * (c - (gx * c + gy * sn)) / D, py = zcy + rho * (sn - (gy * c - gx * sn)) / D;
        ok = refine_extreme<N>(L, wcx, wcy, rho, which, kind, 0.6, px, py, ph, false);
        if (!ok) break;
        const double r = sqrt(px * px + py * py);
        if (e == 0) { x.hi_r = r; x.hi_x = px; x.hi_y = py; x.hi_ph = ph; }
        else if (e == 1) { x.lo_r = r; x.lo_x = px; x.lo_y = py; x.lo_ph = ph; }
        else if (e == 2) { x.thi_t = atan2(py, px); x.thi_x = px; x.thi_y = py; x.thi_ph = ph; }
        else { x.tlo_t = atan2(py, px); x.tlo_x = px; x.tlo_y = py; x.tlo_ph = ph; }
    }
    return ok;
}

// the extreme own points of a sector (sampled) -> the true extremes of the image boundary
template <int N>
UL_HD void refine_sector_extremes(const Lens& L, double wcx, double wcy, double rho, double dph, bool from_origin, BoxExt& x)
{
    if (x.hi_r < 0.0) return;
    if (!from_origin) refine_extreme<N>(L, wcx, wcy, rho, 0, -1, dph, x.lo_x, x.lo_y, x.lo_ph);
    refine_extreme<N>(L, wcx, wcy, rho, 0, +1, dph, x.hi_x, x.hi_y, x.hi_ph);
    if (x.thi_t > -1e299 && !from_origin) {
        refine_extreme<N>(L, wcx, wcy, rho, 1, -1, dph, x.tlo_x, x.tlo_y, x.tlo_ph);
        refine_extreme<N>(L, wcx, wcy, rho, 1, +1, dph, x.thi_x, x.thi_y, x.thi_ph);
    }
}

// ---------------------------------------------------------------------------------------------- phase C
// One sector -> its ray grid (Sec. 3.3 "fixed-resolution polar grid"; spacing from the local image scale).
// Scan lines (one per lane, 32 per work unit) are rings scanned along theta for a bounded sector and radial
// lines scanned along r for a filled ring / disk, whose boundary runs along theta.
//   [rl, rh] x [tl, th]   tight bounds of the member boxes (already expanded by the box margin)
//   hr, ht / cr, ct       smallest projected half-extent / half-chord of the image along r / theta
//   gap_*                 free space to the neighbouring group on each side: margins never use more than
//                         45 % of it, so sectors stay disjoint
UL_HD void emit_patch(Patch& out, const RegionParams& P, int point, double rl, double rh, double tl, double th,
                      double hr_, double ht_, double cr_, double ct_, bool periodic, bool scan_r,
                      double gap_r_lo, double gap_r_hi, double gap_t_lo, double gap_t_hi, int& units_left,
                      unsigned& status)
{
    double r_ext = rh - rl;
    double t_ext = periodic ? 2.0 * UL_PI : (th - tl);
    out.kap_lo = out.kap_hi = 0.0;
    // lines: spaced by the projected half-extent / n_r; nodes on a line: by the half-chord / n_theta
    double hr = ul_min(scan_r ? cr_ : hr_, 0.5 * r_ext);
    double ht = ul_min(scan_r ? ht_ : ct_, 0.5 * t_ext * rh);
    int per_r = scan_r ? P.n_theta : P.n_r, per_t = scan_r ? P.n_r : P.n_theta;
    double want_r = ceil(r_ext / hr * per_r);
    double want_t = ceil(t_ext * rh / ht * per_t);
    int n_r = want_r > (double)P.max_nr ? P.max_nr : (int)want_r;
    int n_th = want_t > (double)P.max_nth ? P.max_nth : (int)want_t;
    if (want_r > (double)P.max_nr || want_t > (double)P.max_nth) status |= UL_ST_RES_CAP;
    if (n_th < 16) n_th = 16;
    if (n_r < 16) n_r = 16;
    double dth = t_ext / n_th;
    double span_t = t_ext;
    if (!periodic) {
        // 3 extra cells of margin per side (cubic stencil + empty border rays)
        // ALONG the scan lines a generous margin costs only a few nodes: 3 cells for the cubic stencil + 5 % of
        // the span; ACROSS the lines the sector must end where the image ends (sin-spaced lines): no margin
        double e_lo = ul_min(3.0 * dth + 0.05 * t_ext, 0.45 * gap_t_lo), e_hi = ul_min(3.0 * dth + 0.05 * t_ext, 0.45 * gap_t_hi);
        if (scan_r) { e_lo = ul_min(0.002 * t_ext, 0.45 * gap_t_lo); e_hi = ul_min(0.002 * t_ext, 0.45 * gap_t_hi); }   // tips thinner than a parabola
        if (scan_r) { out.kap_lo = e_lo / t_ext; out.kap_hi = e_hi / t_ext; }
        tl -= e_lo;
        span_t = t_ext + e_lo + e_hi;
        const double span = span_t;
        n_th = (int)ceil(span / dth);
        if (n_th > P.max_nth) { n_th = P.max_nth; status |= UL_ST_RES_CAP; }
        dth = span / n_th;
    }
    double dr = r_ext / n_r;
    double span_r;
    {
        // radial scan lines need 3 empty nodes per side for the cubic stencil; rings need none
        double e_lo = ul_min(3.0 * dr + 0.05 * r_ext, 0.45 * gap_r_lo), e_hi = ul_min(3.0 * dr + 0.05 * r_ext, 0.45 * gap_r_hi);
        if (!scan_r) { e_lo = ul_min(0.002 * r_ext, 0.45 * gap_r_lo); e_hi = ul_min(0.002 * r_ext, 0.45 * gap_r_hi); }
        if (!scan_r) { out.kap_lo = e_lo / r_ext; out.kap_hi = e_hi / r_ext; }
        if (rl <= 0.0) e_lo = 0.0;
        rl -= e_lo;
        span_r = r_ext + e_lo + e_hi;
        n_r = (int)ceil(span_r / dr);
        if (n_r > P.max_nr) { n_r = P.max_nr; status |= UL_ST_RES_CAP; }
    }
    // the line count is a multiple of 32 (one lane per line)
    int n_units;
    if (scan_r) { n_th = (n_th + 31) & ~31; n_units = n_th / 32; }
    else { n_r = (n_r + 31) & ~31; n_units = n_r / 32; }
    if (n_units > units_left) {                          // per-point unit budget
        status |= UL_ST_RES_CAP;
        n_units = units_left > 1 ? units_left : 1;
        if (scan_r) n_th = 32 * n_units; else n_r = 32 * n_units;
    }
    units_left -= n_units;
    if (units_left < 0) units_left = 0;
    dth = (periodic ? 2.0 * UL_PI : span_t) / n_th;    // the line count was rounded to a multiple of 32
    dr = span_r / n_r;
    out.r0 = rl; out.dr = dr; out.th0 = tl; out.dth = dth; out.n_r = n_r; out.n_th = n_th;
    out.point = point; out.unit0 = 0;
    out.flags = (periodic ? UL_PATCH_PERIODIC : 0) | (scan_r ? UL_PATCH_SCAN_R : 0) | ((scan_r && periodic) ? 0 : UL_PATCH_SINR);
    out.n_units = n_units;
}


UL_HD void ext_reset(BoxExt& x)
{
    x.lo_r = 1e300; x.hi_r = -1.0; x.lo_x = x.lo_y = x.lo_ph = x.hi_x = x.hi_y = x.hi_ph = 0.0;
    x.tlo_t = 1e300; x.thi_t = -1e300; x.tlo_x = x.tlo_y = x.tlo_ph = x.thi_x = x.thi_y = x.thi_ph = 0.0;
}

// union of intervals, order independent: insert [lo, hi] into the list of disjoint groups (room for UL_MAXG_TMP), merging
// every group it touches; at that cap the interval joins the nearest group instead of opening a new one (the only
// order-dependent step: 64 disjoint groups at once have not been seen). interval_reduce brings the final, sorted list
// down to UL_MAXG by closing the narrowest gaps.
UL_HD bool interval_absorb(double* g_lo, double* g_hi, int& ng, double lo, double hi)
{
    int first = -1;                                      // the group that has absorbed [lo, hi] so far
    for (bool changed = true; changed;) {
        changed = false;
        for (int g = 0; g < ng; ++g) {
            if (g == first || lo > g_hi[g] || hi < g_lo[g]) continue;
            if (first < 0) { first = g; g_lo[g] = ul_min(g_lo[g], lo); g_hi[g] = ul_max(g_hi[g], hi); }
            else {
                g_lo[first] = ul_min(g_lo[first], g_lo[g]); g_hi[first] = ul_max(g_hi[first], g_hi[g]);
                --ng; g_lo[g] = g_lo[ng]; g_hi[g] = g_hi[ng];
                if (first == ng) first = g;
            }
            lo = g_lo[first]; hi = g_hi[first];
            changed = true;                              // the grown group may touch groups already passed
            break;
        }
    }
    return first >= 0;
}
UL_HD void interval_insert(double* g_lo, double* g_hi, int& ng, double lo, double hi)
{
    if (interval_absorb(g_lo, g_hi, ng, lo, hi)) return;
    if (ng < UL_MAXG_TMP) { g_lo[ng] = lo; g_hi[ng] = hi; ++ng; return; }
    // at the cap: join the nearest group, then absorb whatever the grown group touches
    int best = 0; double bd = 1e300;
    for (int g = 0; g < ng; ++g) { double d = lo > g_hi[g] ? lo - g_hi[g] : g_lo[g] - hi; if (d < bd) { bd = d; best = g; } }
    lo = ul_min(g_lo[best], lo); hi = ul_max(g_hi[best], hi);
    --ng; g_lo[best] = g_lo[ng]; g_hi[best] = g_hi[ng];
    if (!interval_absorb(g_lo, g_hi, ng, lo, hi)) { g_lo[ng] = lo; g_hi[ng] = hi; ++ng; }
}

UL_HD void interval_sort(double* g_lo, double* g_hi, int ng)
{
    for (int a = 1; a < ng; ++a) {
        double lo = g_lo[a], hi = g_hi[a]; int b = a - 1;
        while (b >= 0 && g_lo[b] > lo) { g_lo[b + 1] = g_lo[b]; g_hi[b + 1] = g_hi[b]; --b; }
        g_lo[b + 1] = lo; g_hi[b + 1] = hi;
    }
}

UL_HD void interval_reduce(double* g_lo, double* g_hi, int& ng, int cap)
{
    while (ng > cap) {                                   // (sorted list) close the narrowest gap
        int best = 0; double bd = 1e300;
        for (int g = 0; g + 1 < ng; ++g) { const double d = g_lo[g + 1] - g_hi[g]; if (d < bd) { bd = d; best = g; } }
        g_hi[best] = ul_max(g_hi[best], g_hi[best + 1]);
        for (int k = best + 1; k + 1 < ng; ++k) { g_lo[k] = g_lo[k + 1]; g_hi[k] = g_hi[k + 1]; }
        --ng;
    }
}

// a gap much narrower than the groups on both sides is the neck between two arcs of one image (an image
// pair about to merge on a critical curve): one group, so that the sector ends where the image ends
UL_HD void interval_merge_necks(double* g_lo, double* g_hi, int& ng)
{
    for (int g = 0; g + 1 < ng;) {
        double gap = g_lo[g + 1] - g_hi[g];
        if (gap < 0.05 * ul_min(g_hi[g] - g_lo[g], g_hi[g + 1] - g_lo[g + 1])) {
            g_hi[g] = ul_max(g_hi[g], g_hi[g + 1]);
            for (int k = g + 1; k + 1 < ng; ++k) { g_lo[k] = g_lo[k + 1]; g_hi[k] = g_hi[k + 1]; }
            --ng;
        } else ++g;
    }
}

// Returns the number of sectors (0 if no image-limb point was found).
// The paper's "1-D binning in r and theta, all combinations, empty ones dropped" as interval unions:
// boxes -> disjoint r-groups; inside each r-group its member boxes -> periodic theta-groups; every
// (r-group, theta-group) is one sector with the tight bounds of its members.
// The boxes only follow image BOUNDARIES. A circle r = const that lies in a gap between two r-groups (or
// inside the innermost one) meets no boundary, so it is entirely inside or entirely outside the image:
// one ray on it decides. Where it is inside (ring-like image around the origin, or a disk that contains
// the origin) the gap is filled: the groups on both sides merge into one full-ring sector.
//   box [nb], ext [nb] or nullptr (forward-mode run: the boxes' extreme own points); patch / ptan [UL_MAXP] out;
//   dph_limb: spacing of this point's limb samples (forward-mode run: how far a true extreme can lie from the sampled one);
//   Pquiet, czr / czi / cmask: a quiet point (k_quiet) and the images of its centre: a sector that holds exactly one of them ends
//   at the true extremes of that image (quiet_image_extremes) and takes the coarser ray grid *Pquiet; any other sector of the
//   point keeps its bounds from the limb samples and the full grid P.
template <int N>
UL_HDN int sectors_from_boxes(const SubBox* box, const BoxExt* ext, int nb, const RegionParams& P, int point, const Lens& L,
                              double wcx, double wcy, double rho, unsigned& status, const TangentTable* TT, Patch* patch,
                              PatchTan* ptan, double dph_limb = 2.0 * UL_PI / 512, const RegionParams* Pquiet = nullptr,
                              const double* czr = nullptr, const double* czi = nullptr, unsigned cmask = 0)
{
    if (nb == 0) { status |= UL_ST_NO_IMAGE; return 0; }

    // ---- r groups
    double gr_lo[UL_MAXG_TMP], gr_hi[UL_MAXG_TMP];
    int ngr = 0;
    for (int i = 0; i < nb; ++i) {
        double rl, rh, tl, th;
        box_expanded(box[i], rl, rh, tl, th);
        interval_insert(gr_lo, gr_hi, ngr, rl, rh);
    }
    interval_sort(gr_lo, gr_hi, ngr);
    interval_merge_necks(gr_lo, gr_hi, ngr);
    interval_reduce(gr_lo, gr_hi, ngr, UL_MAXG);
    // ---- fill gaps whose circles are inside the image
    bool ring_group[UL_MAXG];
    {
        int m = 0;                                       // groups after merging
        for (int g = 0; g < ngr; ++g) {
            double lo_edge = (g == 0) ? 0.0 : gr_hi[g - 1];
            bool fill = false;
            if (gr_lo[g] > lo_edge) {
                double rm = 0.5 * (lo_edge + gr_lo[g]);
                fill = ray_F<N>(L, rm * 0.9553364891256060, rm * 0.2955202066613396, wcx, wcy, rho * rho) < 0.0;   // theta = 0.3
            }
            if (g == 0) {
                gr_lo[0] = fill ? 0.0 : gr_lo[0]; ring_group[0] = fill; m = 1;
            } else if (fill) {
                gr_hi[m - 1] = gr_hi[g]; ring_group[m - 1] = true;
            } else {
                gr_lo[m] = gr_lo[g]; gr_hi[m] = gr_hi[g]; ring_group[m] = false; ++m;
            }
        }
        ngr = m;
    }

    int np = 0;
    int units_left = P.max_units_pt;
    bool capped = false;
    for (int a = 0; a < ngr && !capped; ++a) {
        const double gap_r_lo = (a == 0) ? gr_lo[0] : gr_lo[a] - gr_hi[a - 1];
        const double gap_r_hi = (a == ngr - 1) ? 1e300 : gr_lo[a + 1] - gr_hi[a];
        if (ring_group[a]) {
            // filled ring / disk: one full-ring sector scanned along radial lines
            double hr = 1e300, ht = 1e300, cr = 1e300, ct = 1e300;
            BoxExt xlo; ext_reset(xlo);                  // full ring: theta frozen
            for (int i = 0; i < nb; ++i) {
                const SubBox& b = box[i];
                double rl, rh, tl, th;
                box_expanded(b, rl, rh, tl, th);
                if (!(rl >= gr_lo[a] && rl <= gr_hi[a])) continue;
                hr = ul_min(hr, b.hr); ht = ul_min(ht, b.ht); cr = ul_min(cr, b.cr); ct = ul_min(ct, b.ct);
                if (ext) {
                    const BoxExt& e = ext[i];
                    if (ext_before(e.lo_r, e.lo_ph, e.lo_x, xlo.lo_r, xlo.lo_ph, xlo.lo_x)) { xlo.lo_r = e.lo_r; xlo.lo_x = e.lo_x; xlo.lo_y = e.lo_y; xlo.lo_ph = e.lo_ph; }
                    if (ext_before(-e.hi_r, e.hi_ph, e.hi_x, -xlo.hi_r, xlo.hi_ph, xlo.hi_x)) { xlo.hi_r = e.hi_r; xlo.hi_x = e.hi_x; xlo.hi_y = e.hi_y; xlo.hi_ph = e.hi_ph; }
                }
            }
            if (np == UL_MAXP) { capped = true; break; }
            if (ext && TT) {
                refine_sector_extremes<N>(L, wcx, wcy, rho, dph_limb, gr_lo[a] <= 0.0, xlo);
                patch_tangents<N>(L, *TT, xlo, gr_lo[a] <= 0.0, ptan[np]);
            }
            emit_patch(patch[np++], P, point, gr_lo[a], gr_hi[a], -UL_PI, UL_PI, hr, ht, cr, ct, true, true,
                       gap_r_lo, gap_r_hi, 0.0, 0.0, units_left, status);
            continue;
        }
        // ---- theta groups of this r-group's members: intervals on the circle, t_lo in [-pi, pi), span <= 2 pi
        double gt_lo[UL_MAXG_TMP], gt_hi[UL_MAXG_TMP];
        int ngt = 0;
        bool full_ring = false;
        for (int i = 0; i < nb && !full_ring; ++i) {
            double rl, rh, tl, th;
            box_expanded(box[i], rl, rh, tl, th);
            if (!(rl >= gr_lo[a] && rl <= gr_hi[a])) continue;
            // merge with every group it touches, in whichever turn of the circle they meet
            for (int g = 0; g < ngt;) {
                int k = 2;
                if (!(tl > gt_hi[g] || th < gt_lo[g])) k = 0;
                else if (!(tl + 2.0 * UL_PI > gt_hi[g] || th + 2.0 * UL_PI < gt_lo[g])) k = 1;
                else if (!(tl - 2.0 * UL_PI > gt_hi[g] || th - 2.0 * UL_PI < gt_lo[g])) k = -1;
                if (k != 2) {
                    tl = ul_min(tl + 2.0 * UL_PI * k, gt_lo[g]); th = ul_max(th + 2.0 * UL_PI * k, gt_hi[g]);
                    gt_lo[g] = gt_lo[ngt - 1]; gt_hi[g] = gt_hi[ngt - 1]; --ngt;
                    g = 0;                               // the grown interval may now touch earlier groups
                } else ++g;
            }
            if (th - tl >= 2.0 * UL_PI) { full_ring = true; break; }
            const double sh = 2.0 * UL_PI * floor((tl + UL_PI) / (2.0 * UL_PI));      // t_lo back to [-pi, pi)
            tl -= sh; th -= sh;
            if (ngt < UL_MAXG_TMP) { gt_lo[ngt] = tl; gt_hi[ngt] = th; ++ngt; }
            else { full_ring = true; }                   // more disjoint arcs at once than there is room for: one ring
        }
        if (!full_ring) {
            interval_sort(gt_lo, gt_hi, ngt);
            interval_merge_necks(gt_lo, gt_hi, ngt);
            // the neck between the last and the first group, across the cut at -pi / +pi
            if (ngt > 1) {
                double gap = gt_lo[0] + 2.0 * UL_PI - gt_hi[ngt - 1];
                if (gap < 0.05 * ul_min(gt_hi[0] - gt_lo[0], gt_hi[ngt - 1] - gt_lo[ngt - 1])) {
                    gt_hi[ngt - 1] = gt_hi[0] + 2.0 * UL_PI;
                    for (int k = 0; k + 1 < ngt; ++k) { gt_lo[k] = gt_lo[k + 1]; gt_hi[k] = gt_hi[k + 1]; }
                    --ngt;
                }
            }
            for (int g = 0; g < ngt; ++g) if (gt_hi[g] - gt_lo[g] >= 2.0 * UL_PI - 1e-12) full_ring = true;
            if (ngt > UL_MAXG) full_ring = true;         // more arcs than sectors: one ring around them all
        }
        if (full_ring) { gt_lo[0] = -UL_PI; gt_hi[0] = UL_PI; ngt = 1; }
        // ---- tight bounds of each theta-group's members
        double c_rl[UL_MAXG], c_rh[UL_MAXG], c_tl[UL_MAXG], c_th[UL_MAXG], c_hr[UL_MAXG], c_ht[UL_MAXG], c_cr[UL_MAXG], c_ct[UL_MAXG];
        BoxExt c_ext[UL_MAXG];                           // forward-mode run: the cells' extreme own points
        for (int g = 0; g < ngt; ++g) { c_rl[g] = 1e300; c_rh[g] = -1e300; c_tl[g] = 1e300; c_th[g] = -1e300; c_hr[g] = c_ht[g] = c_cr[g] = c_ct[g] = 1e300; }
        if (ext) for (int g = 0; g < ngt; ++g) ext_reset(c_ext[g]);
        for (int i = 0; i < nb; ++i) {
            const SubBox& b = box[i];
            double rl, rh, tl, th;
            box_expanded(b, rl, rh, tl, th);
            if (!(rl >= gr_lo[a] && rl <= gr_hi[a])) continue;
            int c = 0;
            if (full_ring) { tl = -UL_PI; th = UL_PI; }
            else {
                // the group (and the turn of the circle) this box's lower end lies in -- or lies nearest to: a group's
                // ends went through +- 2 pi shifts while it was merged, so a member can miss it by a rounding error
                double bd = 1e300; int bk = 0;
                for (int g = 0; g < ngt; ++g) {
#pragma unroll
                    for (int k = -1; k <= 1; ++k) {
                        const double t = tl + 2.0 * UL_PI * k;
                        const double d = ul_max(ul_max(gt_lo[g] - t, t - gt_hi[g]), 0.0);
                        if (d < bd) { bd = d; c = g; bk = k; }
                    }
                }
                tl += 2.0 * UL_PI * bk; th += 2.0 * UL_PI * bk;
            }
            c_rl[c] = ul_min(c_rl[c], rl); c_rh[c] = ul_max(c_rh[c], rh);
            c_tl[c] = ul_min(c_tl[c], tl); c_th[c] = ul_max(c_th[c], th);
            c_hr[c] = ul_min(c_hr[c], b.hr); c_ht[c] = ul_min(c_ht[c], b.ht);
            c_cr[c] = ul_min(c_cr[c], b.cr); c_ct[c] = ul_min(c_ct[c], b.ct);
            if (ext) {
                const BoxExt& e = ext[i];
                BoxExt& x = c_ext[c];
                if (ext_before(e.lo_r, e.lo_ph, e.lo_x, x.lo_r, x.lo_ph, x.lo_x)) { x.lo_r = e.lo_r; x.lo_x = e.lo_x; x.lo_y = e.lo_y; x.lo_ph = e.lo_ph; }
                if (ext_before(-e.hi_r, e.hi_ph, e.hi_x, -x.hi_r, x.hi_ph, x.hi_x)) { x.hi_r = e.hi_r; x.hi_x = e.hi_x; x.hi_y = e.hi_y; x.hi_ph = e.hi_ph; }
                // theta ends in the cell's own unwrapping: this box's interval is [tl, th] after the shifts above
                if (ext_before(tl, e.tlo_ph, e.tlo_x, x.tlo_t, x.tlo_ph, x.tlo_x)) { x.tlo_t = tl; x.tlo_x = e.tlo_x; x.tlo_y = e.tlo_y; x.tlo_ph = e.tlo_ph; }
                if (ext_before(-th, e.thi_ph, e.thi_x, -x.thi_t, x.thi_ph, x.thi_x)) { x.thi_t = th; x.thi_x = e.thi_x; x.thi_y = e.thi_y; x.thi_ph = e.thi_ph; }
            }
        }
        // ---- quiet point: a cell that holds exactly one image of the centre ends at that image's true extremes
        bool c_exact[UL_MAXG];
        for (int c = 0; c < ngt; ++c) c_exact[c] = false;
        if (Pquiet && czr && !full_ring) {
            constexpr int DEG = N * N + 1;
            for (int c = 0; c < ngt; ++c) {
                if (c_rl[c] > c_rh[c] || !(c_rl[c] > 0.0)) continue;
                int cnt = 0, kk = -1;
                for (int k = 0; k < DEG; ++k) {
                    if (!((cmask >> k) & 1u)) continue;
                    const double r = sqrt(czr[k] * czr[k] + czi[k] * czi[k]);
                    if (!(r >= c_rl[c] && r <= c_rh[c])) continue;
                    double t = atan2(czi[k], czr[k]);
                    t += 2.0 * UL_PI * floor((0.5 * (c_tl[c] + c_th[c]) - t) / (2.0 * UL_PI) + 0.5);     // the turn nearest to the cell
                    if (t >= c_tl[c] && t <= c_th[c]) { ++cnt; kk = k; }
                }
                if (cnt != 1) continue;
                BoxExt x; ext_reset(x);
                if (!quiet_image_extremes<N>(L, wcx, wcy, rho, czr[kk], czi[kk], x)) continue;
                const double mid = 0.5 * (c_tl[c] + c_th[c]);
                x.tlo_t += 2.0 * UL_PI * floor((mid - x.tlo_t) / (2.0 * UL_PI) + 0.5);
                x.thi_t += 2.0 * UL_PI * floor((mid - x.thi_t) / (2.0 * UL_PI) + 0.5);
                // the true extremes must agree with what the limb samples bounded (else: not the image this cell holds)
                const double er = 0.1 * (c_rh[c] - c_rl[c]), et = 0.1 * (c_th[c] - c_tl[c]);
                if (!(x.lo_r < x.hi_r && x.tlo_t < x.thi_t && x.lo_r >= c_rl[c] - er && x.lo_r <= c_rl[c] + er &&
                      x.hi_r >= c_rh[c] - er && x.hi_r <= c_rh[c] + er && x.tlo_t >= c_tl[c] - et && x.tlo_t <= c_tl[c] + et &&
                      x.thi_t >= c_th[c] - et && x.thi_t <= c_th[c] + et)) continue;
                const double mr = 2e-4 * (x.hi_r - x.lo_r), mt = 2e-4 * (x.thi_t - x.tlo_t);
                c_rl[c] = ul_max(x.lo_r - mr, 0.0); c_rh[c] = x.hi_r + mr; c_tl[c] = x.tlo_t - mt; c_th[c] = x.thi_t + mt;
                c_exact[c] = true;
                if (ext) c_ext[c] = x;
            }
        }
        for (int c = 0; c < ngt; ++c) {
            if (c_rl[c] > c_rh[c]) continue;
            // free space to the neighbouring cells, from the cells' TIGHT bounds (minima / maxima of member values: the same
            // whatever order the boxes arrived in; the group bounds gt_* went through +- 2 pi shifts while they were merged
            // and carry order-dependent rounding in their last bits)
            double gap_lo, gap_hi;
            if (ngt == 1) { gap_lo = gap_hi = 2.0 * UL_PI - (c_th[0] - c_tl[0]); }
            else {
                int cp = (c + ngt - 1) % ngt, cn = (c + 1) % ngt;
                while (c_rl[cp] > c_rh[cp] && cp != c) cp = (cp + ngt - 1) % ngt;          // (skip cells without members)
                while (c_rl[cn] > c_rh[cn] && cn != c) cn = (cn + 1) % ngt;
                gap_lo = c_tl[c] - c_th[cp];
                gap_hi = c_tl[cn] - c_th[c];
                // neighbouring cells live in their own turns of the circle
                gap_lo -= 2.0 * UL_PI * floor(gap_lo / (2.0 * UL_PI));
                gap_hi -= 2.0 * UL_PI * floor(gap_hi / (2.0 * UL_PI));
                if (cp == c) gap_lo = gap_hi = 2.0 * UL_PI - (c_th[c] - c_tl[c]);
            }
            if (np == UL_MAXP) { capped = true; break; }
            // Scan lines run ACROSS the long axis of the sector. Images near the Einstein ring are arcs that
            // hug a circle r = const: along rings their chord length jumps from zero to the full arc within
            // a tiny step in r, while radial lines cut the arc once each and the line integral varies smoothly
            // with theta up to the two tips, which the sin-spaced lines (UL_PATCH_SINR) take care of. A sector
            // that closes on itself in theta has no tips at all (spectral convergence).
            const bool scan_r = full_ring || ((c_th[c] - c_tl[c]) * c_rh[c] > (c_rh[c] - c_rl[c]));
            if (ext && TT) {
                if (!c_exact[c]) refine_sector_extremes<N>(L, wcx, wcy, rho, dph_limb, false, c_ext[c]);
                patch_tangents<N>(L, *TT, c_ext[c], false, ptan[np]);
            }
            emit_patch(patch[np++], c_exact[c] ? *Pquiet : P, point, c_rl[c], c_rh[c], c_tl[c], c_th[c], c_hr[c], c_ht[c], c_cr[c], c_ct[c],
                       full_ring, scan_r, gap_r_lo, gap_r_hi, gap_lo, gap_hi, units_left, status);
        }
    }
    if (capped) {
        // more sectors than the cap: one full-ring sector around everything (never drop an image)
        status |= UL_ST_PATCH_CAP;
        double rl = 1e300, rh = 0.0, hr = 1e300, ht = 1e300, cr = 1e300, ct = 1e300;
        for (int i = 0; i < nb; ++i) {
            const SubBox& b = box[i];
            double a1, a2, a3, a4; box_expanded(b, a1, a2, a3, a4);
            rl = ul_min(rl, a1); rh = ul_max(rh, a2); hr = ul_min(hr, b.hr); ht = ul_min(ht, b.ht); cr = ul_min(cr, b.cr); ct = ul_min(ct, b.ct);
        }
        np = 0; units_left = P.max_units_pt;
        if (ptan) for (int k = 0; k < UL_NT_MAX; ++k) { ptan[0].rlo_dot[k] = 0.0; ptan[0].rhi_dot[k] = 0.0; ptan[0].tlo_dot[k] = 0.0; ptan[0].thi_dot[k] = 0.0; }
        emit_patch(patch[np++], P, point, rl, rh, -UL_PI, UL_PI, hr, ht, cr, ct, true, false, rl, 1e300, 0.0, 0.0,
                   units_left, status);
    }
    return np;
}

}  // namespace ulens
