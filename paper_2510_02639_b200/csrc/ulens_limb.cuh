// ulens_limb.cuh -- image-region builder, first half (steps a3 and the box part of a4): Eq. 8 limb sampling ->
// warm-started Ehrlich-Aberth (Eq. 7) -> validation / polish on Eq. 1 -> one polar (r, theta) box per image
// arc.   PAPER.md Sec. 3.2; readings G2, G6-G8 in DESIGN.md.  Device code only (warp collectives).
//
// Parallel layout (round 2; round 1 ran one LANE per limb arc with ~1.5 KB of per-lane state in local memory:
// 250 registers, 8 warps per SM, 6 % of the FP64 pipe):
//   the limb of a source point is cut into NARC arcs of consecutive limb points; an arc is followed by a GROUP of
//   DEG = N^2+1 lanes, ONE LANE PER ROOT of the lens polynomial; a warp holds GPW groups, and the WARPS = NARC / GPW warps
//   of a point run independently of each other (no barrier: a first version with one CTA per point spent a quarter
//   of its stall samples waiting at the CTA's final barrier for its slowest warp). Everything indexed by root slot in the
//   paper's algorithm is then a per-lane scalar in registers: the root, the image it polishes to, the previous
//   image (warm start / continuation), the box of the arc this slot is drawing. What couples the roots goes
//   through the group: the polynomial coefficients (lane l computes b_l; shared memory), the Aberth repulsion sum
//   (the other roots, shared memory; all roots move at once -- Jacobi order instead of round 1's Gauss-Seidel),
//   convergence / validity votes (ballots). 6 groups share a warp for the binary lens, 3 for the triple lens.
//   A finished box is appended to the point's box list in global memory; k_sectors (ulens_regions.cuh) turns the
//   list into sectors, one thread per point.
// The algorithm along an arc is round 1's, step for step: adaptive limb step (halved and retried when an image
// moved by more than 4 % of its distance from the origin, or when the image set changed), cold restart when the
// warm solve hits its cap, continuation of lost images on Eq. 1, continuation-first for the triple lens, seeds
// from the centre's images at an arc's first point and from the Einstein ring of a light third body, links
// between the boxes of an image pair created / destroyed on a caustic, parabola vertex for the bulge between
// samples.
#pragma once
#include "ulens_core.cuh"
#include "ulens_dual.cuh"
#include "ulens_regions.cuh"

namespace ulens {

template <int N>
struct LimbGeom {
    static constexpr int DEG = N * N + 1;
    static constexpr int GPW = 32 / DEG;                 // groups (arcs) per warp: 16, 6, 3
    static constexpr int NARC = (N == 1) ? 32 : 30;      // arcs per source point
    static constexpr int WARPS = NARC / GPW;             // 2, 5, 10
    static constexpr int THREADS = 32 * WARPS;
};

// shared memory of ONE WARP (its GPW arcs); the warps of a CTA are independent of each other
template <int N>
struct LimbShared {
    double2 coef[LimbGeom<N>::GPW][N * N + 2];           // b_0 .. b_DEG of the arc's current limb point
    double2 z[LimbGeom<N>::GPW][N * N + 1];              // the roots during the simultaneous iteration
};

#define UL_FULL 0xffffffffu

// P and P' at z from the group's coefficients
template <int DEG>
__device__ __forceinline__ void horner_sh(const double2* c, double x, double y, double& pr, double& pi, double& dr, double& di)
{
    pr = c[DEG].x; pi = c[DEG].y; dr = 0.0; di = 0.0;
#pragma unroll
    for (int l = DEG - 1; l >= 0; --l) {
        const double2 b = c[l];
        double t = dr * x - di * y + pr;
        di = dr * y + di * x + pi;
        dr = t;
        t = pr * x - pi * y + b.x;
        pi = pr * y + pi * x + b.y;
        pr = t;
    }
}

// Cauchy-circle start of slot j (G6), from the group's coefficients
template <int DEG>
__device__ __forceinline__ void ea_init_sh(const double2* c, int j, double& zr, double& zi)
{
    const double ln2 = c[DEG].x * c[DEG].x + c[DEG].y * c[DEG].y;
    double m2 = 0.0;
#pragma unroll
    for (int l = 0; l < DEG; ++l) m2 = ul_max(m2, c[l].x * c[l].x + c[l].y * c[l].y);
    double R = ul_min(1.0 + sqrt(m2 / ln2), 8.0);
    const double qx = (c[DEG - 1].x * c[DEG].x + c[DEG - 1].y * c[DEG].y) / ln2;
    const double qy = (c[DEG - 1].y * c[DEG].x - c[DEG - 1].x * c[DEG].y) / ln2;
    double cx = -qx / DEG, cy = -qy / DEG;
    if (!(cx * cx + cy * cy < 16.0)) { cx = 0.0; cy = 0.0; }
    double sn, cs;
    sincos(0.4 + 2.0 * UL_PI * j / DEG, &sn, &cs);
    zr = cx + R * cs; zi = cy + R * sn;
}

// Ehrlich-Aberth (Eq. 7, Newton form G6) with one lane per root, all roots of a group updated at once from the
// others' previous positions. `run`: this lane's group takes part; `frozen`: this lane's root is already exact
// (it still repels the others). Stop rule per root as ea_iterate (ulens_core.cuh). Returns the group's iteration
// count, cap + 1 if a root was still moving at the cap (uniform within a group). All 32 lanes must call.
template <int DEG>
__device__ __forceinline__ int ea_coop(bool run, bool frozen, const double2* coef, double2* zs, int j, unsigned gmask,
                                       double& zr, double& zi, int cap, double tol2)
{
    bool done = !run || frozen;
    bool bad = false;
    double prev_s2 = 1e300, prev_den = 1.0;             // the previous step as (|step|^2, |z|^2): rel = s2 / den without dividing
    int its = 0;
    if (run) zs[j] = make_double2(zr, zi);
    __syncwarp();
    for (int it = 1; it <= cap; ++it) {
        const unsigned nd = __ballot_sync(UL_FULL, !done);
        if (nd == 0) break;
        const bool grp_running = (nd & gmask) != 0;
        if (grp_running) its = it;
        double nzr = zr, nzi = zi;
        if (!done) {
            double pr, pi, dr, di;
            horner_sh<DEG>(coef, zr, zi, pr, pi, dr, di);
            const double p2 = pr * pr + pi * pi;
            if (p2 == 0.0) done = true;
            else {
                const double d2 = dr * dr + di * di;
                double nx, ny;
                if (d2 > 0.0) { const double id = 1.0 / d2; nx = (pr * dr + pi * di) * id; ny = (pi * dr - pr * di) * id; }
                else { nx = 1e-3; ny = 1e-3; }
                double sx = 0.0, sy = 0.0;
#pragma unroll
                for (int jj = 0; jj < DEG; ++jj) {
                    if (jj == j) continue;
                    const double2 o = zs[jj];
                    const double ux = zr - o.x, uy = zi - o.y;
                    const double u2 = ux * ux + uy * uy;
                    if (u2 > 0.0) { const double iu = 1.0 / u2; sx += ux * iu; sy -= uy * iu; }
                }
                const double ax = 1.0 - (nx * sx - ny * sy), ay = -(nx * sy + ny * sx);
                const double a2 = ax * ax + ay * ay;
                double stx, sty;
                if (a2 > 1e-300) { const double ia = 1.0 / a2; stx = (nx * ax + ny * ay) * ia; sty = (ny * ax - nx * ay) * ia; }
                else { stx = nx; sty = ny; }
                nzr = zr - stx; nzi = zi - sty;
                const double s2 = stx * stx + sty * sty, den = nzr * nzr + nzi * nzi + 1e-12;
                if (!(s2 == s2) || !(den == den)) bad = true;
                // rel < tol2  ||  (rel < 1e-6 && rel > 0.5 prev),  rel = s2 / den
                if (s2 < tol2 * den || (s2 < 1e-6 * den && s2 * prev_den > 0.5 * prev_s2 * den)) done = true;
                prev_s2 = s2; prev_den = den;
            }
        }
        __syncwarp();                                    // everyone has read the old positions
        if (run && !frozen && (nzr != zr || nzi != zi)) { zr = nzr; zi = nzi; zs[j] = make_double2(zr, zi); }
        __syncwarp();
    }
    const unsigned nd = __ballot_sync(UL_FULL, !done), bd = __ballot_sync(UL_FULL, bad);
    if ((nd & gmask) || (bd & gmask)) its = cap + 1;
    return its;
}

// Per-lane state of the box a root slot is drawing
struct ArcBox {
    SubBox B;
    double t_cur, lastx, lasty;          // unwrapped theta of / position of the box's last own point
    double h_ph[2], h_r[2], h_t[2];      // its last two own points (limb angle, r, theta): parabola vertex
    int h_n;
    bool open;
};

__device__ __forceinline__ void arcbox_start(ArcBox& a)
{
    a.B.r_lo = 1.0; a.B.r_hi = -1.0; a.B.t_lo = a.B.t_hi = 0.0; a.B.hr = a.B.ht = a.B.cr = a.B.ct = 1e300;
    a.t_cur = 0.0; a.lastx = a.lasty = 0.0; a.h_n = 0; a.open = true;
}

// append a finished box to the point's list (theta interval normalised to t_lo in [-pi, pi), span <= 2 pi)
template <bool DUAL>
__device__ __forceinline__ void arcbox_flush(ArcBox& a, const BoxExt& E, int* n_box, int cap, SubBox* boxes, BoxExt* exts,
                                             unsigned& status)
{
    if (!a.open) return;
    a.open = false;
    if (a.B.r_lo > a.B.r_hi) return;
    const double sh = 2.0 * UL_PI * floor((a.B.t_lo + UL_PI) / (2.0 * UL_PI));
    a.B.t_lo -= sh; a.B.t_hi -= sh;
    if (a.B.t_hi - a.B.t_lo > 2.0 * UL_PI) a.B.t_hi = a.B.t_lo + 2.0 * UL_PI;
    const int idx = atomicAdd(n_box, 1);
    if (idx < cap) {
        boxes[idx] = a.B;
        if (DUAL) exts[idx] = E;
    } else status |= UL_ST_PATCH_CAP;                     // list full: the arc is dropped, the point is flagged
}

// One candidate image per lane (cand_ok, cx, cy with its det J and g) is offered to the group, slot by slot: a
// candidate that is not an image the group already holds takes the lowest free slot, and is tracked from here on.
template <int N, int NC>
__device__ __forceinline__ void adopt_candidates(bool run, int j, int gbase, unsigned gmask, double rho,
                                                 bool cand_ok, double cx, double cy, double cdet, double cgx, double cgy,
                                                 bool& valid, bool& faint, double& px, double& py, double& zr, double& zi,
                                                 double& hr, double& ht, double& cr, double& ct)
{
    constexpr int DEG = N * N + 1;
#pragma unroll 1
    for (int m = 0; m < NC; ++m) {
        const int src = gbase + m;
        const bool ok_m = __shfl_sync(UL_FULL, (int)cand_ok, src) != 0;
        const double mx = __shfl_sync(UL_FULL, cx, src), my = __shfl_sync(UL_FULL, cy, src);
        const double md = __shfl_sync(UL_FULL, cdet, src), mgx = __shfl_sync(UL_FULL, cgx, src), mgy = __shfl_sync(UL_FULL, cgy, src);
        const double ddx = mx - px, ddy = my - py;
        const bool dup = valid && (ddx * ddx + ddy * ddy < 1e-10 * ul_max(1.0, mx * mx + my * my));
        const unsigned dupb = __ballot_sync(UL_FULL, dup) & gmask;
        const unsigned freeb = (~__ballot_sync(UL_FULL, valid)) & gmask;
        if (!run || !ok_m || dupb || !freeb) continue;
        if (gbase + j == __ffs(freeb) - 1) {
            valid = true; px = mx; py = my; zr = mx; zi = my;
            local_extents(mx, my, mgx, mgy, rho, hr, ht, cr, ct);
            faint = fabs(md) > 1e7;
        }
    }
    (void)DEG;
}

// The limb tracker of one warp of one source point (warp = 0 .. WARPS-1: which arcs). All 32 lanes call it.
// n_box: the point's box counter (global memory, zeroed before the launch); returns this lane's status bits and
// adds the warp's limb solves to n_solves_out.
template <int N, bool DUAL>
__device__ unsigned limb_track(LimbShared<N>& sh, int warp, const Lens& L, const LensPoly& T, double wcx, double wcy, double rho,
                               const RegionParams& P, const double* __restrict__ czr, const double* __restrict__ czi,
                               unsigned cmask, SubBox* boxes, BoxExt* exts, int* n_box, int box_cap, int& n_solves_out,
                               int n_arcs = LimbGeom<N>::NARC, int per_arc_in = 0)
{
    typedef LimbGeom<N> G;
    constexpr int DEG = G::DEG;
    const int lane = threadIdx.x & 31;
    const int gw = lane / DEG;
    const bool active = gw < G::GPW && warp * G::GPW + gw < n_arcs;
    const int gbase = active ? gw * DEG : 0;
    const int j = active ? lane - gbase : 0;
    const int arc = active ? warp * G::GPW + gw : 0;
    const unsigned gmask = active ? (((1u << DEG) - 1u) << gbase) : 0u;
    double2* coef = sh.coef[active ? gw : 0];
    double2* zs = sh.z[active ? gw : 0];

    // light lenses (eps_a < 1e-2) whose planetary caustic -- centred on w_a = a_a - sum_{b != a} eps_b/conj(a_a - a_b),
    // a few sqrt(eps_a) across -- the source overlaps or nearly so (triple lens: images hidden in a root cluster)
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

    // (quiet source points, k_quiet: the whole limb as n_arcs = GPW arcs of one warp, per_arc_in points each)
    const int per_arc = per_arc_in > 0 ? per_arc_in : max(1, (P.n_limb + G::NARC / 2) / G::NARC);
    const double dphi = 2.0 * UL_PI / (per_arc * n_arcs);
    const double ph0 = dphi * (arc * per_arc), ph_end = dphi * (arc * per_arc + per_arc);

    double zr = 0.0, zi = 0.0, ozr = 0.0, ozi = 0.0, pvx = 0.0, pvy = 0.0;
    bool vprev = false, fprev = false;
    ArcBox ab; arcbox_start(ab); ab.open = false;
    BoxExt E; ext_reset(E);
    double ph = ph0, step = dphi;
    bool first = true, arc_done = !active;
    int guard = 0, n_solves = 0;
    unsigned status = 0;

    while (__any_sync(UL_FULL, !arc_done)) {
        const bool run = !arc_done;
        double st_try = step;
        if (ph + st_try > ph_end - 1e-9 * dphi) st_try = ph_end - ph;          // land exactly on the arc's end
        const double ph_new = first ? ph0 : ph + st_try;
        double sn, cs;
        sincos(ph_new, &sn, &cs);
        const double wx = wcx + rho * cs, wy = wcy + rho * sn;                  // Eq. 8 (G2)

        // ---- Eq. 4: lane l computes b_l = S_{l-1} - w S_l - R_l (ulens_core.cuh poly_coeffs), b_DEG = S_{DEG-1}
        {
            double ex[N + 1], ey[N + 1], fx[N], fy[N];
            poly_sym<N>(L, wx, wy, ex, ey, fx, fy);
            double ar = 0.0, ai = 0.0, rr = 0.0, ri = 0.0;
#pragma unroll
            for (int k = 0; k <= N; ++k) {
                const double tr = T.tr[k][j], ti = T.ti[k][j];
                ar += ex[k] * tr - ey[k] * ti;
                ai += ex[k] * ti + ey[k] * tr;
                if (k >= 1) {
                    rr += fx[k - 1] * tr - fy[k - 1] * ti;
                    ri += fx[k - 1] * ti + fy[k - 1] * tr;
                }
            }
            double pr_ = __shfl_up_sync(UL_FULL, ar, 1), pi_ = __shfl_up_sync(UL_FULL, ai, 1);
            if (j == 0) { pr_ = 0.0; pi_ = 0.0; }
            if (run) {
                coef[j] = make_double2(pr_ - (wx * ar - wy * ai) - rr, pi_ - (wx * ai + wy * ar) - ri);
                if (j == DEG - 1) coef[DEG] = make_double2(ar, ai);
            }
        }
        __syncwarp();

        // ---- triple lens: continuation first. A slot that held an image at the previous limb point follows it by
        // damped Newton on Eq. 1 itself (exact, and independent of the conditioning of the degree-10 polynomial,
        // SURVEY 7-2); those roots are then FROZEN in the simultaneous iteration -- they still repel the others --
        // so Ehrlich-Aberth only has to move the roots that are not images, which is where image pairs are born.
        bool frozen = false;
        double c_det = 0.0, c_gx = 0.0, c_gy = 0.0;
        if (N == 3) {
            double fxx = pvx, fyy = pvy;
            if (run && !first && vprev) {
                double resid;
                bool ok = polish_image_ni<N>(L, wx, wy, fxx, fyy, 10, 1e-9, c_det, resid, c_gx, c_gy);
                const double jx = fxx - pvx, jy = fyy - pvy;
                frozen = ok && (jx * jx + jy * jy <= 0.0016 * ul_max(fxx * fxx + fyy * fyy, 0.04));
            }
            // two slots running into one image: the pair merges, the later slot lets go
            const unsigned fb = __ballot_sync(UL_FULL, frozen);
            bool dup = false;
#pragma unroll 1
            for (int q = 0; q < DEG - 1; ++q) {
                const double qx = __shfl_sync(UL_FULL, fxx, gbase + q), qy = __shfl_sync(UL_FULL, fyy, gbase + q);
                if (q < j && ((fb >> (gbase + q)) & 1u)) {
                    const double ddx = fxx - qx, ddy = fyy - qy;
                    if (ddx * ddx + ddy * ddy < 1e-10 * ul_max(1.0, fxx * fxx + fyy * fyy)) dup = true;
                }
            }
            frozen = frozen && !dup;
            if (frozen) { zr = fxx; zi = fyy; }
        }

        // ---- Eq. 7. Warm start from the previous limb point (cap 24); cold from the Cauchy circle (cap 64) for the
        // arc's first point or when the warm solve hits its cap.
        // (`first` is the same for every running group of the warp: all arcs take their first point in the same pass)
        // One call site for both passes (code size: the kernel is instruction-fetch bound): pass 0 is the warm solve
        // (cold at an arc's first point), pass 1 the cold restart of the groups whose warm solve failed.
        bool cold = first;
        int it = 0;
        bool go = run;
#pragma unroll 1
        for (int pass = 0; pass < 2; ++pass) {
            if (go && cold) { frozen = false; ea_init_sh<DEG>(coef, j, zr, zi); }
            const int cap = __any_sync(UL_FULL, go && cold) ? 64 : 24;
            const int itp = ea_coop<DEG>(go, frozen, coef, zs, j, gmask, zr, zi, cap, UL_EA_LIMB_TOL2);
            if (go) it = itp;
            go = run && !cold && it > 24;                // warm solve hit its cap: restart this group from the Cauchy circle
            if (!__any_sync(UL_FULL, go)) break;
            if (go) cold = true;
        }
        const bool noconv = run && it > (cold ? 64 : 24);
        if (run && j == 0) ++n_solves;

        // ---- keep root identities along the limb: slot j takes the new root nearest to its previous position, if
        // that assignment is a permutation (it almost always is the identity)
        if (N > 1) {
            int kstar = j;
            const unsigned fb = __ballot_sync(UL_FULL, frozen);
            if (run && !first && !frozen) {
                double bd = 1e300;
#pragma unroll
                for (int k = 0; k < DEG; ++k) {
                    if ((fb >> (gbase + k)) & 1u) continue;
                    const double2 o = zs[k];
                    const double dx = o.x - ozr, dy = o.y - ozi, d = dx * dx + dy * dy;
                    if (d < bd) { bd = d; kstar = k; }
                }
            }
            int claims = 0;
#pragma unroll
            for (int q = 0; q < DEG; ++q) claims += (__shfl_sync(UL_FULL, kstar, gbase + q) == j) ? 1 : 0;
            const unsigned notperm = __ballot_sync(UL_FULL, claims != 1) & gmask;
            if (run && !notperm && kstar != j) { const double2 o = zs[kstar]; zr = o.x; zi = o.y; }
            __syncwarp();
        }

        // ---- validate + polish on Eq. 1 (G7)
        bool ok = false;
        double px = zr, py = zi, detJ = 0.0, gx = 0.0, gy = 0.0, resid;
        if (run) {
            if (frozen) { ok = true; detJ = c_det; gx = c_gx; gy = c_gy; }
            else {
                // distance of the EA root to the nearest lens bounds how far the polish may move it
                double dm2 = 1e300;
#pragma unroll
                for (int i = 0; i < N; ++i) { double dx = zr - L.ax[i], dy = zi - L.ay[i]; dm2 = ul_min(dm2, dx * dx + dy * dy); }
                // (0.04: the acceptance test below allows a total move of 10 % of that distance, so a first step
                // beyond 20 % is rejected either way -- after one iteration instead of six)
                ok = polish_image<N>(L, wx, wy, px, py, 6, 1e-9, detJ, resid, gx, gy, 0.04, false);   // (inlined: measured 12 % faster on C4 than the out-of-line copy)
                // along the limb a slot must follow ONE image continuously: a polish that carries the EA root
                // further than 10 % of its distance to the nearest lens has jumped to some other image
                const double mv2 = (px - zr) * (px - zr) + (py - zi) * (py - zi);
                ok = ok && (mv2 <= 0.01 * dm2);
            }
            // continuation: a slot that held an image at the previous limb point and lost it (EA cannot
            // resolve the root clusters next to a light lens in double) is re-polished from that image
            if (!ok && vprev && (N < 3 || cold)) {
                px = pvx; py = pvy;
                ok = polish_image_ni<N>(L, wx, wy, px, py, 10, 1e-9, detJ, resid, gx, gy);
                const double jx = px - pvx, jy = py - pvy;
                ok = ok && (jx * jx + jy * jy <= 0.0016 * ul_max(px * px + py * py, 0.04));
            }
        }
        // two slots on one image: the later one is not an image of its own
        {
            const unsigned okb = __ballot_sync(UL_FULL, ok);
            bool dup = false;
#pragma unroll
            for (int q = 0; q < DEG - 1; ++q) {
                const double qx = __shfl_sync(UL_FULL, px, gbase + q), qy = __shfl_sync(UL_FULL, py, gbase + q);
                if (q < j && ((okb >> (gbase + q)) & 1u)) {
                    const double ddx = px - qx, ddy = py - qy;
                    if (ddx * ddx + ddy * ddy < 1e-10 * ul_max(1.0, px * px + py * py)) dup = true;
                }
            }
            ok = ok && !dup;
        }
        bool valid = run && ok, faint = false;
        double hr = 1e300, ht = 1e300, cr = 1e300, ct = 1e300;
        if (valid) {
            zr = px; zi = py;                            // polished image = better warm start
            local_extents(px, py, gx, gy, rho, hr, ht, cr, ct);
            // an image of magnification 1/|det J| < 1e-7 (the one sitting on top of a light lens) is
            // tracked but gets no box: at most N of them, i.e. < 3e-7 of A >= 1
            faint = fabs(detJ) > 1e7;
        }

        // ---- arc's first point: seeds from the images of the source CENTRE (step a2: found with an unrestricted
        // polish, duplicates removed, faint images seeded). Whatever a seed converges to is an image of this limb
        // point; if no slot holds it yet it takes a free one.
        if (__any_sync(UL_FULL, run && first)) {
            bool c_ok = false;
            double cx = 0.0, cy = 0.0, cdet = 0.0, cgx = 0.0, cgy = 0.0, cres;
            if (run && first && ((cmask >> j) & 1u)) {
                cx = czr[j]; cy = czi[j];
                c_ok = polish_image_ni<N>(L, wx, wy, cx, cy, 12, 1e-9, cdet, cres, cgx, cgy);
            }
            adopt_candidates<N, DEG>(run && first, j, gbase, gmask, rho, c_ok, cx, cy, cdet, cgx, cgy,
                                     valid, faint, px, py, zr, zi, hr, ht, cr, ct);
        }
        // ---- triple lens: wrong image parity at this limb point, or the source sits on the planetary caustic
        // of a light lens (a missing PAIR leaves the parity right): images next to a light lens hide in the root
        // cluster EA cannot resolve. Seed Eq. 1 from 8 points of that lens's Einstein ring |z - a| = sqrt(eps_a).
        if (N == 3) {
            const unsigned vb = __ballot_sync(UL_FULL, valid) & gmask;
            const int nv = __popc(vb);
            const bool bad_parity = (((nv - (N + 1)) & 1) != 0 || nv < N + 1);
            const bool want = run && (bad_parity || near_light != 0);
            if (__any_sync(UL_FULL, want)) {
#pragma unroll 1
                for (int a = 0; a < N; ++a) {
                    if (!(L.eps[a] < 1e-2)) continue;
                    const bool go = want && (bad_parity || ((near_light >> a) & 1u));
                    if (!__any_sync(UL_FULL, go)) continue;
                    bool c_ok = false;
                    double cx = 0.0, cy = 0.0, cdet = 0.0, cgx = 0.0, cgy = 0.0, cres;
                    if (go && j < 8) {
                        const double re = sqrt(L.eps[a]);
                        double s8, c8;
                        sincos(0.25 * UL_PI * j, &s8, &c8);
                        cx = L.ax[a] + re * c8; cy = L.ay[a] + re * s8;
                        c_ok = polish_image_ni<N>(L, wx, wy, cx, cy, 12, 1e-9, cdet, cres, cgx, cgy);
                    }
                    adopt_candidates<N, 8>(go, j, gbase, gmask, rho, c_ok, cx, cy, cdet, cgx, cgy,
                                           valid, faint, px, py, zr, zi, hr, ht, cr, ct);
                }
            }
        }

        // ---- adaptive step: halve and retry from the previous point when an image moved by more than ~4 % of its
        // distance from the origin (down to dphi / 4096) or when the set of images changed (down to dphi / 8)
        const unsigned validb = __ballot_sync(UL_FULL, valid) & gmask, vprevb = __ballot_sync(UL_FULL, vprev) & gmask;
        bool retry = false;
        {
            bool too_far = false;
            if (valid && vprev && !faint) {
                const double dx = px - pvx, dy = py - pvy;
                too_far = dx * dx + dy * dy > 0.0016 * ul_max(px * px + py * py, 0.04);
            }
            const bool any_far = (__ballot_sync(UL_FULL, too_far) & gmask) != 0;
            if (run && !first && ++guard < 4096) {
                const bool flipped = validb != vprevb;
                retry = (any_far && st_try > dphi * (1.0 / 4096.0)) || (flipped && st_try > dphi * 0.126);
            }
        }
        if (retry) { zr = ozr; zi = ozi; step = 0.5 * st_try; }
        const bool commit = run && !retry;

        // ---- own points: the box of the arc this slot is drawing
        if (commit) {
            if (noconv) status |= UL_ST_EA_NOCONV;
            if (valid && !faint) {
                const double rr = sqrt(px * px + py * py);
                // A box holds ONE arc. If this slot's image is nowhere near the last point of its box (the slot
                // swapped identity with another root, or lost its image and found a different one), the box is
                // finished and a new one starts.
                if (ab.open) {
                    const double dx = px - ab.lastx, dy = py - ab.lasty;
                    if (dx * dx + dy * dy > 0.0036 * ul_max(rr * rr, 0.04)) arcbox_flush<DUAL>(ab, E, n_box, box_cap, boxes, exts, status);
                }
                if (!ab.open) { arcbox_start(ab); if (DUAL) ext_reset(E); }
                box_add(ab.B, ab.t_cur, rr, atan2(py, px), hr, ht, cr, ct, true);
                ab.lastx = px; ab.lasty = py;
                // bulge of the boundary between samples: vertex of the parabola through the last three
                const double tt = ab.t_cur;
                if (ab.h_n >= 2) {
                    double yv;
                    if (parabola_vertex(ab.h_ph[0], ab.h_r[0], ab.h_ph[1], ab.h_r[1], ph_new, rr, yv)) {
                        ab.B.r_lo = ul_min(ab.B.r_lo, ul_max(yv, 0.0)); ab.B.r_hi = ul_max(ab.B.r_hi, yv);
                    }
                    if (parabola_vertex(ab.h_ph[0], ab.h_t[0], ab.h_ph[1], ab.h_t[1], ph_new, tt, yv)) {
                        ab.B.t_lo = ul_min(ab.B.t_lo, yv); ab.B.t_hi = ul_max(ab.B.t_hi, yv);
                    }
                }
                ab.h_ph[0] = ab.h_ph[1]; ab.h_r[0] = ab.h_r[1]; ab.h_t[0] = ab.h_t[1];
                ab.h_ph[1] = ph_new; ab.h_r[1] = rr; ab.h_t[1] = tt;
                if (ab.h_n < 2) ++ab.h_n;
                if (DUAL) {
                    if (rr < E.lo_r) { E.lo_r = rr; E.lo_x = px; E.lo_y = py; E.lo_ph = ph_new; }
                    if (rr > E.hi_r) { E.hi_r = rr; E.hi_x = px; E.hi_y = py; E.hi_ph = ph_new; }
                    if (tt < E.tlo_t) { E.tlo_t = tt; E.tlo_x = px; E.tlo_y = py; E.tlo_ph = ph_new; }
                    if (tt > E.thi_t) { E.thi_t = tt; E.thi_x = px; E.thi_y = py; E.thi_ph = ph_new; }
                }
            }
        }
        // ---- links: a slot that switched off (its last point) or on (its first point) between two limb points is one
        // half of an image pair destroyed / created on a critical curve somewhere between the two partners' end
        // points: each partner's box takes the other's end point, so that the pair's boxes overlap.
        // Partner = the nearest other switching slot, if closer than 0.5 (unrelated flips are not linked).
        {
            const bool sw = commit && !first && (vprev != valid) && !(faint || fprev);
            const unsigned swb = __ballot_sync(UL_FULL, sw);
            if (swb) {                                   // warp-uniform
                const unsigned mine = (swb & gmask) >> gbase;
                const double ex = (vprev && !valid) ? pvx : px, ey = (vprev && !valid) ? pvy : py;
                int nb = -1; double bd = 0.25;
#pragma unroll 1
                for (int q = 0; q < DEG; ++q) {
                    const double qx = __shfl_sync(UL_FULL, ex, gbase + q), qy = __shfl_sync(UL_FULL, ey, gbase + q);
                    if (sw && q != j && ((mine >> q) & 1u)) {
                        const double dx = ex - qx, dy = ey - qy, d = dx * dx + dy * dy;
                        if (d < bd) { bd = d; nb = q; }
                    }
                }
#pragma unroll 1
                for (int q = 0; q < DEG; ++q) {
                    const double qx = __shfl_sync(UL_FULL, ex, gbase + q), qy = __shfl_sync(UL_FULL, ey, gbase + q);
                    const int qnb = __shfl_sync(UL_FULL, nb, gbase + q);
                    if (ab.open && q != j && ((sw && nb == q) || (((mine >> q) & 1u) && qnb == j)))
                        box_add(ab.B, ab.t_cur, sqrt(qx * qx + qy * qy), atan2(qy, qx), 1e300, 1e300, 1e300, 1e300, false);
                }
            }
        }
        if (commit) {
            pvx = px; pvy = py; vprev = valid; fprev = faint;
            ozr = zr; ozi = zi;
            if (!first) { ph = ph_new; step = ul_min(2.0 * st_try, dphi); }
            first = false;
            if (!(ph < ph_end - 1e-9 * dphi)) arc_done = true;
        }
    }
    arcbox_flush<DUAL>(ab, E, n_box, box_cap, boxes, exts, status);
    n_solves_out = n_solves;
    return status;
}

}  // namespace ulens
