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

template <int DEG>
struct RegionWork {
    BoxExt* ext;            // [32 * DEG] or nullptr (primal run)
    PatchTan ptan[UL_MAXP];
    SubBox box[32 * DEG];
    double key_r[32 * DEG], key_t[32 * DEG];   // lower r / lower theta of the expanded boxes (sort keys; empty: 1e300)
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
UL_HDNI void local_extents(double zx, double zy, double gx, double gy, double rho, double& hr, double& ht,
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
                           const RegionParams& P, RegionWork<N * N + 1>& W, unsigned& status, int& n_solves,
                           const double* czr, const double* czi, unsigned cmask)
{
    constexpr int DEG = N * N + 1;
    const int chunk = P.n_limb / 32;
    SubBox* B = &W.box[lane * DEG];
    double t_cur[DEG];              // per BOX: unwrapped theta of its last point
    double lastx[DEG], lasty[DEG];  // per BOX: its last point
    int bmap[DEG];                  // slot -> the box that slot's current arc writes to
    double h_ph[DEG][2], h_r[DEG][2], h_t[DEG][2];   // per BOX: its last two own points (limb angle, r, theta)
    int h_n[DEG];
#pragma unroll
    for (int j = 0; j < DEG; ++j) { bmap[j] = -1; lastx[j] = lasty[j] = 0.0; h_n[j] = 0; }
    double zr[DEG], zi[DEG], ozr[DEG], ozi[DEG], pvx[DEG], pvy[DEG];
    double br[DEG + 1], bi[DEG + 1];
    unsigned valid_prev = 0, faint_prev = 0;
    BoxExt* E = W.ext ? &W.ext[lane * DEG] : nullptr;
    if (E) for (int j = 0; j < DEG; ++j) { E[j].lo_r = 1e300; E[j].hi_r = -1.0; E[j].lo_x = E[j].lo_y = E[j].lo_ph = E[j].hi_x = E[j].hi_y = E[j].hi_ph = 0.0;
        E[j].tlo_t = 1e300; E[j].thi_t = -1e300; E[j].tlo_x = E[j].tlo_y = E[j].tlo_ph = E[j].thi_x = E[j].thi_y = E[j].thi_ph = 0.0; }
#pragma unroll
    for (int j = 0; j < DEG; ++j) { B[j].r_lo = 1.0; B[j].r_hi = -1.0; B[j].t_lo = B[j].t_hi = 0.0; B[j].hr = B[j].ht = B[j].cr = B[j].ct = 1e300; t_cur[j] = 0.0; pvx[j] = pvy[j] = 0.0; }

    // The lane walks its arc of the limb, phi in [phi0, phi0 + chunk dphi], with an ADAPTIVE step: the base
    // step is dphi = 2 pi / n_limb (Eq. 8); a step is halved and retried (down to dphi / 4096) when an image
    // moved by more than ~4 % of its distance from the origin -- where the limb passes close to a lens or to a
    // cusp the image boundary races along a long arc within a fraction of dphi and uniform limb sampling
    // would leave most of that arc unsampled -- and (down to dphi / 8) when the set of images
    // changed, which localises the creation / destruction of an image pair on a caustic.
    // light lenses (eps_a < 1e-2) whose planetary caustic -- centred on w_a = a_a - sum_{b != a} eps_b/conj(a_a - a_b),
    // a few sqrt(eps_a) across -- the source overlaps or nearly so
    unsigned near_light = 0;
    if (N == 3) {
#pragma unroll
        for (int a = 0; a < N; ++a) {
            if (!(L.eps[a] < 1e-2)) continue;
            double tx = L.ax[a] - wcx, ty = L.ay[a] - wcy;
#pragma unroll
            for (int b = 0; b < N; ++b) {
                if (b == a) continue;
                double dx = L.ax[a] - L.ax[b], dy = L.ay[a] - L.ay[b];
                double i2 = L.eps[b] / (dx * dx + dy * dy);
                tx -= dx * i2; ty -= dy * i2;
            }
            const double R = 8.0 * sqrt(L.eps[a]) + 2.0 * rho;
            if (tx * tx + ty * ty < R * R) near_light |= 1u << a;
        }
    }
    const double dphi = 2.0 * UL_PI / P.n_limb;
    const double ph0 = dphi * (lane * chunk), ph_end = dphi * (lane * chunk + chunk);
    double ph = ph0, step = dphi;
    bool first = true;
    int guard = 0;
    while (first || ph < ph_end - 1e-9 * dphi) {
        const int s = first ? 0 : 1;
        double st_try = step;
        if (ph + st_try > ph_end - 1e-9 * dphi) st_try = ph_end - ph;      // land exactly on the arc's end
        const double ph_new = first ? ph0 : ph + st_try;
        double wx = wcx + rho * cos(ph_new), wy = wcy + rho * sin(ph_new);      // Eq. 8 (G2)
        poly_coeffs_ni<N>(L, T, wx, wy, br, bi);
        // limb solves only have to land in the basin of the Eq.-1 polish: relative step 1e-7.
        // Warm start from the previous limb point (cap 24); cold restart from the Cauchy circle (cap 64) for the
        // arc's first point or when the warm solve hits its cap. One call site each (code size).
        int it;
        bool cold = first;
        // Triple lens: continuation first. A slot that held an image at the previous limb point follows it by
        // damped Newton on Eq. 1 itself (exact, and independent of the conditioning of the degree-10 polynomial,
        // SURVEY 7-2). Those roots are then FROZEN in the simultaneous iteration -- they still repel the others
        // (implicit deflation, Eq. 7) -- so Ehrlich-Aberth only has to move the roots that are not images, which
        // is where image pairs are born. Measured on C3: 11 % faster step, 30 % fewer rays (no sectors from
        // noisy roots next to the light lenses), fewer flagged points; for degree 5 the warm-started EA is
        // already as cheap and the plain order is 6 % faster, so N <= 2 keeps it.
        unsigned frozen = 0;
        double c_det[DEG], c_gx[DEG], c_gy[DEG];
        if (!first) {
#pragma unroll
            for (int j = 0; j < DEG; ++j) { ozr[j] = zr[j]; ozi[j] = zi[j]; }
        }
        if (N == 3 && !first) {
#pragma unroll 1
            for (int j = 0; j < DEG; ++j) {
                if (!(valid_prev & (1u << j))) continue;
                double zx = pvx[j], zy = pvy[j], detJ, resid, gx, gy;
                bool ok = polish_image_ni<N>(L, wx, wy, zx, zy, 10, 1e-9, detJ, resid, gx, gy);
                double jx = zx - pvx[j], jy = zy - pvy[j];
                ok = ok && (jx * jx + jy * jy <= 0.0016 * ul_max(zx * zx + zy * zy, 0.04));
                if (ok) {
#pragma unroll 1
                    for (int q = 0; q < j; ++q) {          // two slots running into one image: the pair merges
                        if (!(frozen & (1u << q))) continue;
                        double ddx = zx - zr[q], ddy = zy - zi[q];
                        if (ddx * ddx + ddy * ddy < 1e-10 * ul_max(1.0, zx * zx + zy * zy)) ok = false;
                    }
                }
                if (ok) { zr[j] = zx; zi[j] = zy; frozen |= 1u << j; c_det[j] = detJ; c_gx[j] = gx; c_gy[j] = gy; }
            }
        }
#pragma unroll 1
        for (;;) {
            if (cold) { ea_init_ni<DEG>(br, bi, zr, zi); frozen = 0; }
            it = ea_iterate_ni<DEG>(br, bi, zr, zi, cold ? 64 : 24, UL_EA_LIMB_TOL2, frozen);
            if (cold || it <= 24) break;
            cold = true;
        }
        if (!first) {
            if (cold && it <= 64) it = 1;
            match_roots<DEG>(ozr, ozi, zr, zi, frozen);  // slot j keeps following the same root
        }
        ++n_solves;
        const bool noconv = (first && it > 64) || (!first && it > 24);

        unsigned valid = 0, faint = 0;
        double px[DEG], py[DEG], hrr[DEG], htt[DEG], crr[DEG], ctt[DEG];
#pragma unroll 1
        for (int j = 0; j < DEG; ++j) {
            double zx = zr[j], zy = zi[j], detJ, resid, gx, gy;
            bool ok;
            if (frozen & (1u << j)) {                    // continued image: already exact
                ok = true; detJ = c_det[j]; gx = c_gx[j]; gy = c_gy[j];
            } else {
            // distance of the EA root to the nearest lens bounds how far the polish may move it
            double dm2 = 1e300;
#pragma unroll
            for (int i = 0; i < N; ++i) { double dx = zx - L.ax[i], dy = zy - L.ay[i]; dm2 = ul_min(dm2, dx * dx + dy * dy); }
            // (0.04: the acceptance test below allows a total move of 10 % of that distance, so a first step
            // beyond 20 % is rejected either way -- after one iteration instead of six)
            ok = polish_image_ni<N>(L, wx, wy, zx, zy, 6, 1e-9, detJ, resid, gx, gy, 0.04);
            // along the limb a slot must follow ONE image continuously: a polish that carries the EA root
            // further than 10 % of its distance to the nearest lens has jumped to some other image
            double mv2 = (zx - zr[j]) * (zx - zr[j]) + (zy - zi[j]) * (zy - zi[j]);
            ok = ok && (mv2 <= 0.01 * dm2);
            }
            // continuation: a slot that held an image at the previous limb point and lost it (EA cannot
            // resolve the root clusters next to a light lens in double) is re-polished from that image
            if (!ok && (valid_prev & (1u << j)) && (N < 3 || cold)) {
                zx = pvx[j]; zy = pvy[j];
                ok = polish_image_ni<N>(L, wx, wy, zx, zy, 10, 1e-9, detJ, resid, gx, gy);
                double jx = zx - pvx[j], jy = zy - pvy[j];
                ok = ok && (jx * jx + jy * jy <= 0.0016 * ul_max(zx * zx + zy * zy, 0.04));
            }
            // two slots on one image: the later one is not an image of its own
            if (ok) {
#pragma unroll
                for (int q = 0; q < DEG; ++q) {
                    if (q >= j || !(valid & (1u << q))) continue;
                    double ddx = zx - px[q], ddy = zy - py[q];
                    if (ddx * ddx + ddy * ddy < 1e-10 * ul_max(1.0, zx * zx + zy * zy)) ok = false;
                }
            }
            px[j] = zx; py[j] = zy;
            if (ok) {
                valid |= 1u << j;
                zr[j] = zx; zi[j] = zy;                 // polished image = better warm start
                local_extents(zx, zy, gx, gy, rho, hrr[j], htt[j], crr[j], ctt[j]);
                // an image of magnification 1/|det J| < 1e-7 (the one sitting on top of a light lens) is
                // tracked but gets no sector: at most N of them, i.e. < 3e-7 of A >= 1
                if (fabs(detJ) > 1e7) faint |= 1u << j;
            } else { hrr[j] = htt[j] = crr[j] = ctt[j] = 1e300; }
        }
        if (first) {
            // seed the arc's first point from the images of the source CENTRE (step a2, found with an
            // unrestricted polish, duplicates removed, faint images seeded): damped Newton on Eq. 1 for this
            // limb point from each of them. Whatever it converges to is an image of the limb point; if no
            // slot holds it yet it takes a free one.
#pragma unroll 1
            for (int m = 0; m < DEG; ++m) {
                if (!(cmask & (1u << m))) continue;
                double zx = czr[m], zy = czi[m], detJ, resid, gx, gy;
                if (!polish_image_ni<N>(L, wx, wy, zx, zy, 12, 1e-9, detJ, resid, gx, gy)) continue;
                bool dup = false;
                int free_slot = -1;
#pragma unroll
                for (int q = 0; q < DEG; ++q) {
                    if (valid & (1u << q)) {
                        double ddx = zx - px[q], ddy = zy - py[q];
                        if (ddx * ddx + ddy * ddy < 1e-10 * ul_max(1.0, zx * zx + zy * zy)) dup = true;
                    } else if (free_slot < 0) free_slot = q;
                }
                if (dup || free_slot < 0) continue;
                const int q = free_slot;
                valid |= 1u << q; px[q] = zx; py[q] = zy; zr[q] = zx; zi[q] = zy;
                local_extents(zx, zy, gx, gy, rho, hrr[q], htt[q], crr[q], ctt[q]);
                if (fabs(detJ) > 1e7) faint |= 1u << q;
            }
        }
        if (N == 3) {
            // Wrong image parity at this limb point: images next to a light lens are hidden in the root cluster
            // EA cannot resolve (see centre_images). Seed Eq. 1 from that lens's Einstein ring; whatever converges to
            // an image no slot holds yet takes a free slot and is tracked by continuation from here on.
            int nv = 0;
#pragma unroll
            for (int j = 0; j < DEG; ++j) nv += (valid >> j) & 1u;
            const bool bad_parity = (((nv - (N + 1)) & 1) != 0 || nv < N + 1);
            // A missing PAIR leaves the parity right. Where the source sits on the planetary caustic of a light lens
            // (near_light, below) the ring is therefore seeded at every limb point.
            if (bad_parity || near_light) {
#pragma unroll 1
                for (int a = 0; a < N; ++a) {
                    if (!(L.eps[a] < 1e-2)) continue;
                    if (!bad_parity && !(near_light & (1u << a))) continue;
                    const double re = sqrt(L.eps[a]);
#pragma unroll 1
                    // all 8 directions at the arc's first point and on a wrong parity; otherwise the even and the odd
                    // four on alternate limb points (an image, once found, is tracked by continuation)
                    const int k_step = (first || bad_parity) ? 1 : 2, k_0 = (first || bad_parity) ? 0 : (n_solves & 1);
                    for (int k = k_0; k < 8; k += k_step) {
                        double zx = L.ax[a] + re * UL_RING8_X(k), zy = L.ay[a] + re * UL_RING8_Y(k), detJ, resid, gx, gy;
                        if (!polish_image_ni<N>(L, wx, wy, zx, zy, 12, 1e-9, detJ, resid, gx, gy)) continue;
                        bool dup = false;
                        int free_slot = -1;
#pragma unroll 1
                        for (int q = 0; q < DEG; ++q) {
                            if (valid & (1u << q)) {
                                double ddx = zx - px[q], ddy = zy - py[q];
                                if (ddx * ddx + ddy * ddy < 1e-10 * ul_max(1.0, zx * zx + zy * zy)) dup = true;
                            } else if (free_slot < 0) free_slot = q;
                        }
                        if (dup || free_slot < 0) continue;
                        const int q = free_slot;
                        valid |= 1u << q; px[q] = zx; py[q] = zy; zr[q] = zx; zi[q] = zy;
                        local_extents(zx, zy, gx, gy, rho, hrr[q], htt[q], crr[q], ctt[q]);
                        if (fabs(detJ) > 1e7) faint |= 1u << q;
                    }
                }
            }
        }
        if (!first && ++guard < 4096) {
            // largest image displacement over this step, relative to the image's distance from the origin
            bool too_far = false;
#pragma unroll
            for (int j = 0; j < DEG; ++j) {
                if (!(valid & valid_prev & ~faint & (1u << j))) continue;
                double dx = px[j] - pvx[j], dy = py[j] - pvy[j];
                double z2 = px[j] * px[j] + py[j] * py[j];
                if (dx * dx + dy * dy > 0.0016 * ul_max(z2, 0.04)) too_far = true;
            }
            const bool flipped = (valid != valid_prev);
            if ((too_far && st_try > dphi * (1.0 / 4096.0)) || (flipped && st_try > dphi * 0.126)) {
#pragma unroll
                for (int j = 0; j < DEG; ++j) { zr[j] = ozr[j]; zi[j] = ozi[j]; }
                step = 0.5 * st_try;
                continue;                                 // retry from the previous point with half the step
            }
        }
        if (noconv) status |= UL_ST_EA_NOCONV;
        // own points
#pragma unroll 1
        for (int j = 0; j < DEG; ++j) {
            if (!(valid & ~faint & (1u << j))) continue;
            // A box holds ONE arc. If this slot's image is nowhere near the last point of its box (the slot
            // swapped identity with another root, or lost its image and found a different one), its new
            // arc goes to an unused box of this lane if there is one.
            int bi = bmap[j];
            const double far2 = 0.0036 * ul_max(px[j] * px[j] + py[j] * py[j], 0.04);
            if (bi >= 0) {
                double dx = px[j] - lastx[bi], dy = py[j] - lasty[bi];
                if (dx * dx + dy * dy > far2) bi = -1;
            }
            if (bi < 0) {
                // an empty box no slot writes to; failing that, the box whose last point is nearest
                double bd = 1e300; int nearest = 0;
                for (int b = 0; b < DEG && bi < 0; ++b) {
                    bool in_use = false;
                    for (int q = 0; q < DEG; ++q) in_use = in_use || (q != j && bmap[q] == b);
                    if (B[b].r_lo > B[b].r_hi) { if (!in_use) bi = b; continue; }
                    double dx = px[j] - lastx[b], dy = py[j] - lasty[b], d = dx * dx + dy * dy;
                    if (d < bd) { bd = d; nearest = b; }
                }
                if (bi < 0) bi = nearest;
                bmap[j] = bi;
                h_n[bi] = 0;                             // a new arc starts: forget the old arc's samples
            }
            box_add(B[bi], t_cur[bi], sqrt(px[j] * px[j] + py[j] * py[j]), atan2(py[j], px[j]), hrr[j], htt[j], crr[j], ctt[j], true);
            lastx[bi] = px[j]; lasty[bi] = py[j];
            {
                // bulge of the boundary between samples: vertex of the parabola through the last three
                const double rr = sqrt(px[j] * px[j] + py[j] * py[j]), tt = t_cur[bi];
                if (h_n[bi] >= 2) {
                    double yv;
                    if (parabola_vertex(h_ph[bi][0], h_r[bi][0], h_ph[bi][1], h_r[bi][1], ph_new, rr, yv)) {
                        B[bi].r_lo = ul_min(B[bi].r_lo, ul_max(yv, 0.0)); B[bi].r_hi = ul_max(B[bi].r_hi, yv);
                    }
                    if (parabola_vertex(h_ph[bi][0], h_t[bi][0], h_ph[bi][1], h_t[bi][1], ph_new, tt, yv)) {
                        B[bi].t_lo = ul_min(B[bi].t_lo, yv); B[bi].t_hi = ul_max(B[bi].t_hi, yv);
                    }
                }
                h_ph[bi][0] = h_ph[bi][1]; h_r[bi][0] = h_r[bi][1]; h_t[bi][0] = h_t[bi][1];
                h_ph[bi][1] = ph_new; h_r[bi][1] = rr; h_t[bi][1] = tt;
                if (h_n[bi] < 2) ++h_n[bi];
            }
            if (E) {
                double rr = sqrt(px[j] * px[j] + py[j] * py[j]);
                if (rr < E[bi].lo_r) { E[bi].lo_r = rr; E[bi].lo_x = px[j]; E[bi].lo_y = py[j]; E[bi].lo_ph = ph_new; }
                if (rr > E[bi].hi_r) { E[bi].hi_r = rr; E[bi].hi_x = px[j]; E[bi].hi_y = py[j]; E[bi].hi_ph = ph_new; }
                if (t_cur[bi] < E[bi].tlo_t) { E[bi].tlo_t = t_cur[bi]; E[bi].tlo_x = px[j]; E[bi].tlo_y = py[j]; E[bi].tlo_ph = ph_new; }
                if (t_cur[bi] > E[bi].thi_t) { E[bi].thi_t = t_cur[bi]; E[bi].thi_x = px[j]; E[bi].thi_y = py[j]; E[bi].thi_ph = ph_new; }
            }
        }
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
#pragma unroll 1
                for (int a = 0; a < DEG; ++a) {
                    if (!(grp & ~(faint | faint_prev) & (1u << a))) continue;
                    int nb = -1; double bd = 0.25;
#pragma unroll 1
                    for (int b = 0; b < DEG; ++b) {
                        if (b == a || !(grp & ~(faint | faint_prev) & (1u << b))) continue;
                        double dx = ex[a] - ex[b], dy = ey[a] - ey[b];
                        double d = dx * dx + dy * dy;
                        if (d < bd) { bd = d; nb = b; }
                    }
                    if (nb >= 0) {
                        double ra = sqrt(ex[a] * ex[a] + ey[a] * ey[a]), ta = atan2(ey[a], ex[a]);
                        double rb = sqrt(ex[nb] * ex[nb] + ey[nb] * ey[nb]), tb = atan2(ey[nb], ex[nb]);
                        if (bmap[nb] >= 0) box_add(B[bmap[nb]], t_cur[bmap[nb]], ra, ta, 1e300, 1e300, 1e300, 1e300, false);
                        if (bmap[a] >= 0) box_add(B[bmap[a]], t_cur[bmap[a]], rb, tb, 1e300, 1e300, 1e300, 1e300, false);
                    }
                }
            }
        }
#pragma unroll
        for (int j = 0; j < DEG; ++j) { pvx[j] = px[j]; pvy[j] = py[j]; }
        valid_prev = valid; faint_prev = faint;
        if (!first) { ph = ph_new; step = ul_min(2.0 * st_try, dphi); }
        first = false;
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

// ---------------------------------------------------------------------------------------------- phase B
template <int DEG>
UL_HDN void regions_phaseB_keys(int lane, RegionWork<DEG>& W)
{
    const int n = 32 * DEG;
    for (int i = lane; i < n; i += 32) {
        const SubBox& b = W.box[i];
        double rl = 1e300, rh, tl = 1e300, th;
        if (!(b.r_lo > b.r_hi)) box_expanded(b, rl, rh, tl, th);
        W.key_r[i] = rl; W.key_t[i] = tl;
    }
}

// rank sort on the cached keys (call regions_phaseB_keys first, then synchronise the warp)
template <int DEG>
UL_HDN void regions_phaseB(int lane, RegionWork<DEG>& W)
{
    const int n = 32 * DEG;
    for (int i = lane; i < n; i += 32) {
        const double rl = W.key_r[i], tl = W.key_t[i];
        if (rl >= 1e300) continue;
        int rank_r = 0, rank_t = 0;
        for (int j = 0; j < n; ++j) {
            const double rl2 = W.key_r[j], tl2 = W.key_t[j];
            if (rl2 >= 1e300 || j == i) continue;
            rank_r += (rl2 < rl) || (rl2 == rl && j < i);
            rank_t += (tl2 < tl) || (tl2 == tl && j < i);
        }
        W.order_r[rank_r] = (short)i;
        W.order_t[rank_t] = (short)i;
    }
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

// Returns the number of sectors (0 if no image-limb point was found).
// The paper's "1-D binning in r and theta, all combinations, empty ones dropped" as interval sweeps:
// boxes -> disjoint r-groups; inside each r-group its member boxes -> periodic theta-groups; every
// (r-group, theta-group) is one sector with the tight bounds of its members.
// The boxes only follow image BOUNDARIES. A circle r = const that lies in a gap between two r-groups (or
// inside the innermost one) meets no boundary, so it is entirely inside or entirely outside the image:
// one ray on it decides. Where it is inside (ring-like image around the origin, or a disk that contains
// the origin) the gap is filled: the groups on both sides merge into one full-ring sector.
template <int N>
UL_HDN int regions_phaseC(RegionWork<N * N + 1>& W, const RegionParams& P, int point, const Lens& L, double wcx,
                          double wcy, double rho, unsigned& status, const TangentTable* TT = nullptr)
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
    // a gap much narrower than the groups on both sides is the neck between two arcs of one image (an image
    // pair about to merge on a critical curve): one group, so that the sector ends where the image ends
    for (int g = 0; g + 1 < ngr;) {
        double gap = gr_lo[g + 1] - gr_hi[g];
        if (gap < 0.05 * ul_min(gr_hi[g] - gr_lo[g], gr_hi[g + 1] - gr_lo[g + 1])) {
            gr_hi[g] = gr_hi[g + 1];
            for (int k = g + 1; k + 1 < ngr; ++k) { gr_lo[k] = gr_lo[k + 1]; gr_hi[k] = gr_hi[k + 1]; }
            --ngr;
        } else ++g;
    }
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
            BoxExt xlo; xlo.lo_r = 1e300; xlo.hi_r = -1.0; xlo.lo_x = xlo.lo_y = xlo.lo_ph = xlo.hi_x = xlo.hi_y = xlo.hi_ph = 0.0;
            xlo.tlo_t = 1e300; xlo.thi_t = -1e300; xlo.tlo_x = xlo.tlo_y = xlo.tlo_ph = xlo.thi_x = xlo.thi_y = xlo.thi_ph = 0.0;   // full ring: theta frozen
            for (int i = 0; i < n; ++i) {
                const SubBox& b = W.box[i];
                if (b.r_lo > b.r_hi) continue;
                double rl, rh, tl, th;
                box_expanded(b, rl, rh, tl, th);
                if (!(rl >= gr_lo[a] && rl <= gr_hi[a])) continue;
                hr = ul_min(hr, b.hr); ht = ul_min(ht, b.ht); cr = ul_min(cr, b.cr); ct = ul_min(ct, b.ct);
                if (W.ext) {
                    const BoxExt& e = W.ext[i];
                    if (e.lo_r < xlo.lo_r) { xlo.lo_r = e.lo_r; xlo.lo_x = e.lo_x; xlo.lo_y = e.lo_y; xlo.lo_ph = e.lo_ph; }
                    if (e.hi_r > xlo.hi_r) { xlo.hi_r = e.hi_r; xlo.hi_x = e.hi_x; xlo.hi_y = e.hi_y; xlo.hi_ph = e.hi_ph; }
                }
            }
            if (np == UL_MAXP) { capped = true; break; }
            if (W.ext && TT) patch_tangents<N>(L, *TT, xlo, gr_lo[a] <= 0.0, W.ptan[np]);
            emit_patch(W.patch[np++], P, point, gr_lo[a], gr_hi[a], -UL_PI, UL_PI, hr, ht, cr, ct, true, true,
                       gap_r_lo, gap_r_hi, 0.0, 0.0, units_left, status);
            continue;
        }
        // ---- theta groups of this r-group's members (periodic)
        double gt_lo[UL_MAXG], gt_hi[UL_MAXG];
        int ngt = 0;
        {
            double cur_hi = -1e300;
            for (int q = 0; q < nb; ++q) {
                double rl, rh, tl, th;
                box_expanded(W.box[W.order_t[q]], rl, rh, tl, th);
                if (!(rl >= gr_lo[a] && rl <= gr_hi[a])) continue;
                if (ngt == 0 || (tl > cur_hi && ngt < UL_MAXG)) { gt_lo[ngt] = tl; gt_hi[ngt] = th; cur_hi = th; ++ngt; }
                else { cur_hi = ul_max(cur_hi, th); gt_hi[ngt - 1] = cur_hi; }
            }
            for (int g = 0; g + 1 < ngt;) {               // necks, as for r
                double gap = gt_lo[g + 1] - gt_hi[g];
                if (gap < 0.05 * ul_min(gt_hi[g] - gt_lo[g], gt_hi[g + 1] - gt_lo[g + 1])) {
                    gt_hi[g] = gt_hi[g + 1];
                    for (int k = g + 1; k + 1 < ngt; ++k) { gt_lo[k] = gt_lo[k + 1]; gt_hi[k] = gt_hi[k + 1]; }
                    --ngt;
                } else ++g;
            }
            // wrap: the group reaching furthest past +pi swallows the leading groups it covers
            for (;;) {
                if (ngt <= 1) break;
                int im = 0;
                for (int g = 1; g < ngt; ++g) if (gt_hi[g] > gt_hi[im]) im = g;
                if (im == 0 || gt_hi[im] - 2.0 * UL_PI < gt_lo[0]) break;
                gt_hi[im] = ul_max(gt_hi[im], gt_hi[0] + 2.0 * UL_PI);
                for (int g = 1; g < ngt; ++g) { gt_lo[g - 1] = gt_lo[g]; gt_hi[g - 1] = gt_hi[g]; }
                --ngt;
            }
            for (int g = 0; g < ngt; ++g) if (gt_hi[g] - gt_lo[g] >= 2.0 * UL_PI) { gt_lo[0] = -UL_PI; gt_hi[0] = UL_PI; ngt = 1; break; }
        }
        const bool full_ring = (ngt == 1 && gt_hi[0] - gt_lo[0] >= 2.0 * UL_PI - 1e-12);
        // ---- tight bounds of each theta-group's members
        double c_rl[UL_MAXG], c_rh[UL_MAXG], c_tl[UL_MAXG], c_th[UL_MAXG], c_hr[UL_MAXG], c_ht[UL_MAXG], c_cr[UL_MAXG], c_ct[UL_MAXG];
        BoxExt c_ext[UL_MAXG];
        for (int g = 0; g < ngt; ++g) { c_ext[g].lo_r = 1e300; c_ext[g].hi_r = -1.0; c_ext[g].lo_x = c_ext[g].lo_y = c_ext[g].lo_ph = c_ext[g].hi_x = c_ext[g].hi_y = c_ext[g].hi_ph = 0.0;
            c_ext[g].tlo_t = 1e300; c_ext[g].thi_t = -1e300; c_ext[g].tlo_x = c_ext[g].tlo_y = c_ext[g].tlo_ph = c_ext[g].thi_x = c_ext[g].thi_y = c_ext[g].thi_ph = 0.0; }
        for (int g = 0; g < ngt; ++g) { c_rl[g] = 1e300; c_rh[g] = -1e300; c_tl[g] = 1e300; c_th[g] = -1e300; c_hr[g] = c_ht[g] = c_cr[g] = c_ct[g] = 1e300; }
        for (int i = 0; i < n; ++i) {
            const SubBox& b = W.box[i];
            if (b.r_lo > b.r_hi) continue;
            double rl, rh, tl, th;
            box_expanded(b, rl, rh, tl, th);
            if (!(rl >= gr_lo[a] && rl <= gr_hi[a])) continue;
            int c = 0;
            if (full_ring) { tl = -UL_PI; th = UL_PI; }
            else {
                for (int g = 0; g < ngt; ++g) {
                    if (tl >= gt_lo[g] && tl <= gt_hi[g]) { c = g; break; }
                    if (tl + 2.0 * UL_PI >= gt_lo[g] && tl + 2.0 * UL_PI <= gt_hi[g]) { c = g; tl += 2.0 * UL_PI; th += 2.0 * UL_PI; break; }
                }
            }
            c_rl[c] = ul_min(c_rl[c], rl); c_rh[c] = ul_max(c_rh[c], rh);
            c_tl[c] = ul_min(c_tl[c], tl); c_th[c] = ul_max(c_th[c], th);
            c_hr[c] = ul_min(c_hr[c], b.hr); c_ht[c] = ul_min(c_ht[c], b.ht);
            c_cr[c] = ul_min(c_cr[c], b.cr); c_ct[c] = ul_min(c_ct[c], b.ct);
            if (W.ext) {
                const BoxExt& e = W.ext[i];
                BoxExt& x = c_ext[c];
                if (e.lo_r < x.lo_r) { x.lo_r = e.lo_r; x.lo_x = e.lo_x; x.lo_y = e.lo_y; x.lo_ph = e.lo_ph; }
                if (e.hi_r > x.hi_r) { x.hi_r = e.hi_r; x.hi_x = e.hi_x; x.hi_y = e.hi_y; x.hi_ph = e.hi_ph; }
                // theta ends in the cell's own unwrapping: this box's interval is [tl, th] after the shifts above
                if (tl < x.tlo_t) { x.tlo_t = tl; x.tlo_x = e.tlo_x; x.tlo_y = e.tlo_y; x.tlo_ph = e.tlo_ph; }
                if (th > x.thi_t) { x.thi_t = th; x.thi_x = e.thi_x; x.thi_y = e.thi_y; x.thi_ph = e.thi_ph; }
            }
        }
        for (int c = 0; c < ngt; ++c) {
            if (c_rl[c] > c_rh[c]) continue;
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
            if (np == UL_MAXP) { capped = true; break; }
            // Scan lines run ACROSS the long axis of the sector. Images near the Einstein ring are arcs that
            // hug a circle r = const: along rings their chord length jumps from zero to the full arc within
            // a tiny step in r, while radial lines cut the arc once each and the line integral varies smoothly
            // with theta up to the two tips, which the sin-spaced lines (UL_PATCH_SINR) take care of. A sector
            // that closes on itself in theta has no tips at all (spectral convergence).
            const bool scan_r = full_ring || ((c_th[c] - c_tl[c]) * c_rh[c] > (c_rh[c] - c_rl[c]));
            if (W.ext && TT) patch_tangents<N>(L, *TT, c_ext[c], false, W.ptan[np]);
            emit_patch(W.patch[np++], P, point, c_rl[c], c_rh[c], c_tl[c], c_th[c], c_hr[c], c_ht[c], c_cr[c], c_ct[c],
                       full_ring, scan_r, gap_r_lo, gap_r_hi, gap_lo, gap_hi, units_left, status);
        }
    }
    if (capped) {
        // more sectors than the cap: one full-ring sector around everything (never drop an image)
        status |= UL_ST_PATCH_CAP;
        double rl = 1e300, rh = 0.0, hr = 1e300, ht = 1e300, cr = 1e300, ct = 1e300;
        for (int i = 0; i < n; ++i) {
            const SubBox& b = W.box[i];
            if (b.r_lo > b.r_hi) continue;
            double a1, a2, a3, a4; box_expanded(b, a1, a2, a3, a4);
            rl = ul_min(rl, a1); rh = ul_max(rh, a2); hr = ul_min(hr, b.hr); ht = ul_min(ht, b.ht); cr = ul_min(cr, b.cr); ct = ul_min(ct, b.ct);
        }
        np = 0; units_left = P.max_units_pt;
        for (int k = 0; k < UL_NT_MAX; ++k) { W.ptan[0].rlo_dot[k] = 0.0; W.ptan[0].rhi_dot[k] = 0.0; W.ptan[0].tlo_dot[k] = 0.0; W.ptan[0].thi_dot[k] = 0.0; }
        emit_patch(W.patch[np++], P, point, rl, rh, -UL_PI, UL_PI, hr, ht, cr, ct, true, false, rl, 1e300, 0.0, 0.0,
                   units_left, status);
    }
    W.n_patch = np;
    return np;
}

}  // namespace ulens
