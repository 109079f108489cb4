// ulens_regions.cuh -- image-region (sector) builder: Eq. 8 limb sampling -> image-limb points ->
// polar (r, theta) boxes -> 1-D interval grouping in r and theta -> sectors with margins and a ray
// grid sized from the local image scale.   PAPER.md Sec. 3.2; readings G2, G8 in DESIGN.md.
//
// One warp builds the sectors of one source point. The work is written as phases that take the lane
// index explicitly, so the same code is also callable lane by lane from a host logic test:
//   phase A (32 lanes)  each lane follows n_limb/32 consecutive limb points (warm-started EA, Eq. 7),
//                       validates / polishes every root on Eq. 1 and keeps, per root slot, the polar
//                       bounding box of the image-limb points it saw (a piece of an image boundary);
//                       slots whose validity flips between consecutive limb points (image pairs created
//                       or destroyed on a caustic) are linked so that their boxes overlap.
//   phase B (32 lanes)  rank-sort the boxes by lower r and by lower theta.
//   phase C (lane 0)    sweep the sorted intervals -> r-groups, theta-groups (periodic); every occupied
//                       (r-group, theta-group) cell becomes one sector ("all combinations of radial and
//                       angular bins ... empty sectors are discarded, periodic ones merged"), refined to the
//                       min/max of its members plus a margin, with n_r x n_theta from the local image scale.
#pragma once
#include "ulens_core.cuh"

namespace ulens {

struct SubBox {
    double r_lo, r_hi;      // r_lo > r_hi: empty
    double t_lo, t_hi;      // unwrapped theta interval, t_lo in [-pi, pi), t_hi - t_lo <= 2 pi
    double hr, ht;          // smallest local half-extent (projection) of the image in r / along theta: scan-line spacing
    double cr, ct;          // smallest local half-chord of the image along r / along theta: node spacing on a line
};

#define UL_MAXP 12          // sector cap per point ("capped based on the maximum expected number of images")
#define UL_MAXG 16          // groups per axis

struct RegionParams {
    int n_limb;             // multiple of 32
    int n_r, n_theta;       // rays per image half-extent
    int max_nr, max_nth;    // caps per sector
    int max_units_pt;       // cap on 32-ring units per point
};

template <int DEG>
struct RegionWork {
    SubBox box[32 * DEG];
    short order_r[32 * DEG], order_t[32 * DEG];
    int n_sorted;
    unsigned status;
    int n_patch;
    Patch patch[UL_MAXP];
};

UL_HD double wrap_pi(double a)      // to (-pi, pi]
{
    if (a > UL_PI) a -= 2.0 * UL_PI;
    else if (a <= -UL_PI) a += 2.0 * UL_PI;
    return a;
}

// add an image-limb point to a slot box (polar coordinates about the origin, G8)
UL_HD void box_add(SubBox& b, double& t_cur, double r, double th, double hr, double ht, double cr, double ct, bool advance)
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

// local image scale at an image point z with g = sum eps_i/conj(z-a_i)^2: the image of a small disk of
// radius rho is an ellipse with semi-axes rho/(1+|g|) (along arg(g)/2) and rho/|1-|g|| (perpendicular);
// hr, ht = its half-extents (projections) along the radial / azimuthal direction at z; cr, ct = its
// half-chords through the centre along those directions.
UL_HD void local_extents(double zx, double zy, double gx, double gy, double rho, double& hr, double& ht,
                         double& cr, double& ct)
{
    double ga = sqrt(gx * gx + gy * gy);
    double m = rho / (1.0 + ga);
    double den = fabs(1.0 - ga);
    double M = den > 1e-6 ? rho / den : rho * 1e6;
    double z2 = zx * zx + zy * zy;
    double c2 = 0.0;                                    // cos(2 phi), phi = angle(major axis) - angle(radial)
    if (ga > 1e-300 && z2 > 1e-300) {
        // Re(g conj(z)^2) / (|g||z|^2) = cos(arg g - 2 theta);  major axis at arg(g)/2 + pi/2
        double re = gx * (zx * zx - zy * zy) + gy * (2.0 * zx * zy);
        c2 = -re / (ga * z2);
    }
    double cc = 0.5 * (1.0 + c2), ss = 0.5 * (1.0 - c2);
    hr = sqrt(M * M * cc + m * m * ss);
    ht = sqrt(M * M * ss + m * m * cc);
    cr = 1.0 / sqrt(cc / (M * M) + ss / (m * m));
    ct = 1.0 / sqrt(ss / (M * M) + cc / (m * m));
}

// ---------------------------------------------------------------------------------------------- phase A
template <int N>
UL_HDN void regions_phaseA(int lane, const Lens& L, const LensPoly& T, double wcx, double wcy, double rho,
                           const RegionParams& P, RegionWork<N * N + 1>& W, unsigned& status, int& n_solves)
{
    constexpr int DEG = N * N + 1;
    const int chunk = P.n_limb / 32;
    SubBox* B = &W.box[lane * DEG];
    double t_cur[DEG];
    double zr[DEG], zi[DEG], ozr[DEG], ozi[DEG], pvx[DEG], pvy[DEG];
    double br[DEG + 1], bi[DEG + 1];
    unsigned valid_prev = 0;
#pragma unroll
    for (int j = 0; j < DEG; ++j) { B[j].r_lo = 1.0; B[j].r_hi = -1.0; B[j].t_lo = B[j].t_hi = 0.0; B[j].hr = B[j].ht = B[j].cr = B[j].ct = 1e300; t_cur[j] = 0.0; pvx[j] = pvy[j] = 0.0; }

    const double dphi = 2.0 * UL_PI / P.n_limb;
    for (int s = 0; s <= chunk; ++s) {
        int k = lane * chunk + s;                       // limb index; k = n_limb wraps to 0 (same point)
        double ph = dphi * k;
        double wx = wcx + rho * cos(ph), wy = wcy + rho * sin(ph);      // Eq. 8 (G2)
        poly_coeffs<N>(L, T, wx, wy, br, bi);
        // limb solves only have to land in the basin of the Eq.-1 polish: relative step 1e-7
        int it;
        bool cold = (s == 0);
        if (s == 0) { ea_init<DEG>(br, bi, zr, zi); it = ea_iterate<DEG>(br, bi, zr, zi, 64, 1e-14); }
        else {
#pragma unroll
            for (int j = 0; j < DEG; ++j) { ozr[j] = zr[j]; ozi[j] = zi[j]; }
            it = ea_iterate<DEG>(br, bi, zr, zi, 24, 1e-14);
            if (it > 24) { cold = true; ea_init<DEG>(br, bi, zr, zi); it = ea_iterate<DEG>(br, bi, zr, zi, 64, 1e-14); if (it <= 64) it = 1; }
            match_roots<DEG>(ozr, ozi, zr, zi);          // slot j keeps following the same root
        }
        ++n_solves;
        if ((s == 0 && it > 64) || (s > 0 && it > 24)) status |= UL_ST_EA_NOCONV;
        (void)cold;

        unsigned valid = 0;
        double px[DEG], py[DEG], hrr[DEG], htt[DEG], crr[DEG], ctt[DEG];
#pragma unroll
        for (int j = 0; j < DEG; ++j) {
            double zx = zr[j], zy = zi[j], detJ, resid, gx, gy;
            // distance of the EA root to the nearest lens bounds how far the polish may move it
            double dm2 = 1e300;
#pragma unroll
            for (int i = 0; i < N; ++i) { double dx = zx - L.ax[i], dy = zy - L.ay[i]; dm2 = ul_min(dm2, dx * dx + dy * dy); }
            bool ok = polish_image<N>(L, wx, wy, zx, zy, 4, 1e-9, detJ, resid, gx, gy);
            double mv2 = (zx - zr[j]) * (zx - zr[j]) + (zy - zi[j]) * (zy - zi[j]);
            ok = ok && (mv2 <= 0.01 * dm2);
            px[j] = zx; py[j] = zy;
            if (ok) {
                valid |= 1u << j;
                zr[j] = zx; zi[j] = zy;                 // polished image = better warm start
                local_extents(zx, zy, gx, gy, rho, hrr[j], htt[j], crr[j], ctt[j]);
            } else { hrr[j] = htt[j] = crr[j] = ctt[j] = 1e300; }
        }
        // own points
#pragma unroll
        for (int j = 0; j < DEG; ++j)
            if (valid & (1u << j))
                box_add(B[j], t_cur[j], sqrt(px[j] * px[j] + py[j] * py[j]), atan2(py[j], px[j]), hrr[j], htt[j], crr[j], ctt[j], true);
        // links: a slot that switched off (its last point) or on (its first point) between s-1 and s is one
        // half of an image pair destroyed / created on a critical curve somewhere between the two partners'
        // end points: each partner's box takes the other's end point, so that the pair's boxes overlap.
        // Partner = the nearest other switching slot, if closer than 0.5 (unrelated flips are not linked).
        if (s > 0) {
            unsigned off = valid_prev & ~valid, on = valid & ~valid_prev;
            unsigned grp = off | on;
            if (grp && (grp & (grp - 1))) {             // at least two members
                double ex[DEG], ey[DEG];
#pragma unroll
                for (int a = 0; a < DEG; ++a) { ex[a] = (off & (1u << a)) ? pvx[a] : px[a]; ey[a] = (off & (1u << a)) ? pvy[a] : py[a]; }
#pragma unroll
                for (int a = 0; a < DEG; ++a) {
                    if (!(grp & (1u << a))) continue;
                    int nb = -1; double bd = 0.25;
#pragma unroll
                    for (int b = 0; b < DEG; ++b) {
                        if (b == a || !(grp & (1u << b))) continue;
                        double dx = ex[a] - ex[b], dy = ey[a] - ey[b];
                        double d = dx * dx + dy * dy;
                        if (d < bd) { bd = d; nb = b; }
                    }
                    if (nb >= 0) {
                        double ra = sqrt(ex[a] * ex[a] + ey[a] * ey[a]), ta = atan2(ey[a], ex[a]);
                        double rb = sqrt(ex[nb] * ex[nb] + ey[nb] * ey[nb]), tb = atan2(ey[nb], ex[nb]);
                        box_add(B[nb], t_cur[nb], ra, ta, 1e300, 1e300, 1e300, 1e300, false);
                        box_add(B[a], t_cur[a], rb, tb, 1e300, 1e300, 1e300, 1e300, false);
                    }
                }
            }
        }
#pragma unroll
        for (int j = 0; j < DEG; ++j) { pvx[j] = px[j]; pvy[j] = py[j]; }
        valid_prev = valid;
    }
    // normalise theta intervals: t_lo in [-pi, pi)
#pragma unroll
    for (int j = 0; j < DEG; ++j) {
        if (B[j].r_lo > B[j].r_hi) continue;
        double sh = 2.0 * UL_PI * floor((B[j].t_lo + UL_PI) / (2.0 * UL_PI));
        B[j].t_lo -= sh; B[j].t_hi -= sh;
        if (B[j].t_hi - B[j].t_lo > 2.0 * UL_PI) B[j].t_hi = B[j].t_lo + 2.0 * UL_PI;
    }
}

// margins applied to every box before grouping: a quarter of the local minor scale in both directions
// plus 2 % of the box itself (boundary bulge between limb samples)
UL_HD void box_expanded(const SubBox& b, double& rl, double& rh, double& tl, double& th)
{
    double m = ul_min(b.cr, b.ct);
    double mr = 0.25 * m + 0.02 * (b.r_hi - b.r_lo);
    double rmid = ul_max(0.5 * (b.r_lo + b.r_hi), 1e-300);
    double mt = 0.25 * m / rmid + 0.02 * (b.t_hi - b.t_lo);
    mt = ul_min(mt, 0.5);
    rl = ul_max(b.r_lo - mr, 0.0); rh = b.r_hi + mr;
    tl = b.t_lo - mt; th = b.t_hi + mt;
}

// ---------------------------------------------------------------------------------------------- phase B
template <int DEG>
UL_HDN void regions_phaseB(int lane, RegionWork<DEG>& W)
{
    const int n = 32 * DEG;
    for (int i = lane; i < n; i += 32) {
        const SubBox& b = W.box[i];
        if (b.r_lo > b.r_hi) continue;
        double rl, rh, tl, th;
        box_expanded(b, rl, rh, tl, th);
        int rank_r = 0, rank_t = 0;
        for (int j = 0; j < n; ++j) {
            const SubBox& c = W.box[j];
            if (c.r_lo > c.r_hi || j == i) continue;
            double rl2, rh2, tl2, th2;
            box_expanded(c, rl2, rh2, tl2, th2);
            rank_r += (rl2 < rl) || (rl2 == rl && j < i);
            rank_t += (tl2 < tl) || (tl2 == tl && j < i);
        }
        W.order_r[rank_r] = (short)i;
        W.order_t[rank_t] = (short)i;
    }
}

// ---------------------------------------------------------------------------------------------- phase C
// Returns the number of sectors (0 if no image-limb point was found).
// The boxes only follow image BOUNDARIES. A circle r = const that lies in a gap between two r-groups (or
// inside the innermost one) meets no boundary, so it is entirely inside or entirely outside the image:
// one ray on it decides. Where it is inside (ring-like image around the origin, or a disk that contains
// the origin) the gap is filled: the groups on both sides merge into one full-ring sector.
template <int N>
UL_HDN int regions_phaseC(RegionWork<N * N + 1>& W, const RegionParams& P, int point, const Lens& L, double wcx,
                          double wcy, double rho, unsigned& status)
{
    constexpr int DEG = N * N + 1;
    const int n = 32 * DEG;
    int nb = 0;
    for (int i = 0; i < n; ++i) nb += !(W.box[i].r_lo > W.box[i].r_hi);
    W.n_sorted = nb;
    W.n_patch = 0;
    if (nb == 0) { status |= UL_ST_NO_IMAGE; return 0; }

    // ---- r groups
    double gr_lo[UL_MAXG], gr_hi[UL_MAXG];
    int ngr = 0;
    {
        double cur_hi = -1.0;
        for (int q = 0; q < nb; ++q) {
            double rl, rh, tl, th;
            box_expanded(W.box[W.order_r[q]], rl, rh, tl, th);
            if (ngr == 0 || (rl > cur_hi && ngr < UL_MAXG)) { gr_lo[ngr] = rl; gr_hi[ngr] = rh; cur_hi = rh; ++ngr; }
            else { cur_hi = ul_max(cur_hi, rh); gr_hi[ngr - 1] = cur_hi; }
        }
    }
    // ---- fill gaps whose circles are inside the image
    bool ring_group[UL_MAXG];
    {
        int m = 0;                                       // groups after merging
        bool fill_prev = false;
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
            fill_prev = fill;
        }
        (void)fill_prev;
        ngr = m;
    }
    // ---- theta groups (periodic)
    double gt_lo[UL_MAXG], gt_hi[UL_MAXG];
    int ngt = 0;
    {
        double cur_hi = -1e300;
        for (int q = 0; q < nb; ++q) {
            double rl, rh, tl, th;
            box_expanded(W.box[W.order_t[q]], rl, rh, tl, th);
            if (ngt == 0 || (tl > cur_hi && ngt < UL_MAXG)) { gt_lo[ngt] = tl; gt_hi[ngt] = th; cur_hi = th; ++ngt; }
            else { cur_hi = ul_max(cur_hi, th); gt_hi[ngt - 1] = cur_hi; }
        }
        // wrap: the group reaching furthest past +pi swallows the leading groups it covers
        for (;;) {
            if (ngt <= 1) break;
            int im = 0;
            for (int g = 1; g < ngt; ++g) if (gt_hi[g] > gt_hi[im]) im = g;
            if (im == 0 || gt_hi[im] - 2.0 * UL_PI < gt_lo[0]) break;
            // merge group 0 into group im (shifted by 2 pi), drop group 0
            gt_hi[im] = ul_max(gt_hi[im], gt_hi[0] + 2.0 * UL_PI);
            for (int g = 1; g < ngt; ++g) { gt_lo[g - 1] = gt_lo[g]; gt_hi[g - 1] = gt_hi[g]; }
            --ngt;
        }
        for (int g = 0; g < ngt; ++g) if (gt_hi[g] - gt_lo[g] >= 2.0 * UL_PI) { gt_lo[0] = -UL_PI; gt_hi[0] = UL_PI; ngt = 1; break; }
    }
    const bool full_ring_only = (ngt == 1 && gt_hi[0] - gt_lo[0] >= 2.0 * UL_PI - 1e-12);

    // ---- occupied cells -> sectors (tight bbox of the members, expanded)
    signed char cell[UL_MAXG][UL_MAXG];
    for (int a = 0; a < UL_MAXG; ++a) for (int b = 0; b < UL_MAXG; ++b) cell[a][b] = -1;
    double p_rl[UL_MAXP], p_rh[UL_MAXP], p_tl[UL_MAXP], p_th[UL_MAXP], p_hr[UL_MAXP], p_ht[UL_MAXP], p_cr[UL_MAXP], p_ct[UL_MAXP];
    int p_gr[UL_MAXP], p_gt[UL_MAXP];
    int np = 0;
    bool capped = false;
    for (int i = 0; i < n; ++i) {
        const SubBox& b = W.box[i];
        if (b.r_lo > b.r_hi) continue;
        double rl, rh, tl, th;
        box_expanded(b, rl, rh, tl, th);
        int a = 0;
        for (int g = 0; g < ngr; ++g) if (rl >= gr_lo[g] && rl <= gr_hi[g]) { a = g; break; }
        int c = 0;
        if (ring_group[a]) { rl = gr_lo[a]; rh = gr_hi[a]; }
        if (full_ring_only || ring_group[a]) { tl = -UL_PI; th = UL_PI; }
        else {
            bool found = false;
            for (int g = 0; g < ngt && !found; ++g) {
                if (tl >= gt_lo[g] && tl <= gt_hi[g]) { c = g; found = true; }
                else if (tl + 2.0 * UL_PI >= gt_lo[g] && tl + 2.0 * UL_PI <= gt_hi[g]) { c = g; tl += 2.0 * UL_PI; th += 2.0 * UL_PI; found = true; }
            }
        }
        int p = cell[a][c];
        if (p < 0) {
            if (np == UL_MAXP) { capped = true; p = UL_MAXP - 1; }
            else {
                p = np++; cell[a][c] = (signed char)p;
                p_rl[p] = rl; p_rh[p] = rh; p_tl[p] = tl; p_th[p] = th; p_hr[p] = b.hr; p_ht[p] = b.ht; p_cr[p] = b.cr; p_ct[p] = b.ct; p_gr[p] = a; p_gt[p] = c;
                continue;
            }
        }
        p_rl[p] = ul_min(p_rl[p], rl); p_rh[p] = ul_max(p_rh[p], rh);
        p_tl[p] = ul_min(p_tl[p], tl); p_th[p] = ul_max(p_th[p], th);
        p_hr[p] = ul_min(p_hr[p], b.hr); p_ht[p] = ul_min(p_ht[p], b.ht);
        p_cr[p] = ul_min(p_cr[p], b.cr); p_ct[p] = ul_min(p_ct[p], b.ct);
    }
    if (capped) {
        // more sectors than the cap: one sector around everything (never drop an image)
        status |= UL_ST_PATCH_CAP;
        double rl = 1e300, rh = 0.0, hr = 1e300, ht = 1e300, cr = 1e300, ct = 1e300;
        for (int i = 0; i < n; ++i) {
            const SubBox& b = W.box[i];
            if (b.r_lo > b.r_hi) continue;
            double a1, a2, a3, a4; box_expanded(b, a1, a2, a3, a4);
            rl = ul_min(rl, a1); rh = ul_max(rh, a2); hr = ul_min(hr, b.hr); ht = ul_min(ht, b.ht); cr = ul_min(cr, b.cr); ct = ul_min(ct, b.ct);
        }
        np = 1; p_rl[0] = rl; p_rh[0] = rh; p_tl[0] = -UL_PI; p_th[0] = UL_PI; p_hr[0] = hr; p_ht[0] = ht; p_cr[0] = cr; p_ct[0] = ct; p_gr[0] = 0; p_gt[0] = 0;
        ngr = 1; gr_lo[0] = rl; gr_hi[0] = rh; ngt = 1; gt_lo[0] = -UL_PI; gt_hi[0] = UL_PI;
    }

    // ---- grid per sector. Scan lines (one per lane, 32 per work unit) are rings scanned along theta for a
    // bounded sector (Sec. 3.3) and radial lines scanned along r for a filled ring / disk, whose boundary
    // runs along theta: there the line integral is a smooth periodic function of theta.
    int units_left = P.max_units_pt;
    for (int p = 0; p < np; ++p) {
        Patch& out = W.patch[p];
        bool periodic = (p_th[p] - p_tl[p] >= 2.0 * UL_PI - 1e-12);
        bool scan_r = periodic && ring_group[p_gr[p]];
        double r_ext = p_rh[p] - p_rl[p];
        double t_ext = periodic ? 2.0 * UL_PI : (p_th[p] - p_tl[p]);
        // lines: spaced by the projected half-extent / n_r; nodes on a line: by the half-chord / n_theta
        double hr = ul_min(scan_r ? p_cr[p] : p_hr[p], 0.5 * r_ext);
        double ht = ul_min(scan_r ? p_ht[p] : p_ct[p], 0.5 * t_ext * p_rh[p]);
        int per_r = scan_r ? P.n_theta : P.n_r, per_t = scan_r ? P.n_r : P.n_theta;
        double want_r = ceil(r_ext / hr * per_r);
        double want_t = ceil(t_ext * p_rh[p] / ht * per_t);
        int n_r = want_r > (double)P.max_nr ? P.max_nr : (int)want_r;
        int n_th = want_t > (double)P.max_nth ? P.max_nth : (int)want_t;
        if (want_r > (double)P.max_nr || want_t > (double)P.max_nth) status |= UL_ST_RES_CAP;
        if (n_th < 16) n_th = 16;
        if (n_r < 16) n_r = 16;
        double dth = t_ext / n_th;
        double tl = p_tl[p];
        if (!periodic) {
            // 3 extra cells of margin per side (cubic stencil + empty border rays), but never more than
            // 45 % of the gap to the neighbouring theta-group so that sectors stay disjoint
            int c = p_gt[p];
            double gap_lo, gap_hi;
            if (ngt == 1) { gap_lo = gap_hi = 2.0 * UL_PI - (gt_hi[0] - gt_lo[0]); }
            else {
                int cp = (c + ngt - 1) % ngt, cn = (c + 1) % ngt;
                gap_lo = gt_lo[c] - gt_hi[cp]; if (c == 0) gap_lo += 2.0 * UL_PI;
                gap_hi = gt_lo[cn] - gt_hi[c]; if (c == ngt - 1) gap_hi += 2.0 * UL_PI;
                // a group shifted by the wrap merge may sit a full turn away
                gap_lo -= 2.0 * UL_PI * floor(gap_lo / (2.0 * UL_PI));
                gap_hi -= 2.0 * UL_PI * floor(gap_hi / (2.0 * UL_PI));
            }
            double e_lo = ul_min(3.0 * dth, 0.45 * gap_lo), e_hi = ul_min(3.0 * dth, 0.45 * gap_hi);
            tl -= e_lo;
            double span = t_ext + e_lo + e_hi;
            n_th = (int)ceil(span / dth);
            if (n_th > P.max_nth) { n_th = P.max_nth; status |= UL_ST_RES_CAP; }
            dth = span / n_th;
        }
        // r: 3 extra cells of margin per side within 45 % of the gap to the neighbouring r-group
        double dr = r_ext / n_r;
        double rl = p_rl[p];
        double span_r = r_ext;
        {
            int a = p_gr[p];
            double gap_lo = (a == 0) ? gr_lo[0] : gr_lo[a] - gr_hi[a - 1];
            double gap_hi = (a == ngr - 1) ? 1e300 : gr_lo[a + 1] - gr_hi[a];
            double e_lo = ul_min(3.0 * dr, 0.45 * gap_lo), e_hi = ul_min(3.0 * dr, 0.45 * gap_hi);
            if (p_rl[p] <= 0.0) e_lo = 0.0;
            rl -= e_lo;
            span_r = r_ext + e_lo + e_hi;
            n_r = (int)ceil(span_r / dr);
            if (n_r > P.max_nr) { n_r = P.max_nr; status |= UL_ST_RES_CAP; }
        }
        // the line count is a multiple of 32 (one lane per line)
        int n_units;
        if (scan_r) { n_th = (n_th + 31) & ~31; n_units = n_th / 32; }
        else { n_r = (n_r + 31) & ~31; n_units = n_r / 32; }
        if (n_units > units_left) {                      // per-point unit budget
            status |= UL_ST_RES_CAP;
            n_units = units_left > 1 ? units_left : 1;
            if (scan_r) n_th = 32 * n_units; else n_r = 32 * n_units;
        }
        units_left -= n_units;
        if (units_left < 0) units_left = 0;
        if (periodic) dth = 2.0 * UL_PI / n_th;
        dr = span_r / n_r;
        out.r0 = rl; out.dr = dr; out.th0 = tl; out.dth = dth; out.n_r = n_r; out.n_th = n_th;
        out.point = point; out.unit0 = 0;
        out.flags = (periodic ? UL_PATCH_PERIODIC : 0) | (scan_r ? UL_PATCH_SCAN_R : 0);
        out.n_units = n_units;
    }
    W.n_patch = np;
    return np;
}

}  // namespace ulens
