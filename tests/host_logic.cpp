// Host-compiled check of the device headers' per-thread logic (test infrastructure only: the product has no CPU
// path -- ulens_create fails without a CUDA device). The .cuh files compile as plain C++; this runs, for ONE source
// point, the code the kernels run per thread: centre_images (k_roots), sectors_from_boxes (k_sectors), every scan
// line of every sector (k_shoot) and the ordered sum (k_finalize), and prints machine-readable lines for
// tests/test_host_logic.py. The limb tracker itself (k_limb) is warp-cooperative device code; here a plain serial
// stand-in (limb_boxes_serial below: a cold solve at every limb point, boxes grown by proximity) feeds the sector
// builder with boxes made by the same helpers (box_add, local_extents).
//
// usage: host_logic N eps.. ax.. ay..  rho u1 wx wy n_limb n_r n_theta
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include "../paper_2510_02639_b200/csrc/ulens_core.cuh"
#include "../paper_2510_02639_b200/csrc/ulens_regions.cuh"
#include "../paper_2510_02639_b200/csrc/ulens_host.hpp"
using namespace ulens;

// test-side stand-in for k_limb: uniform limb sampling (Eq. 8), a cold Ehrlich-Aberth solve + Eq.-1 polish at every
// limb point (centre_images), each image joining the open box whose last point is nearest (else opening a new one)
template <int N>
static int limb_boxes_serial(const Lens& L, const LensPoly& T, double wx, double wy, double rho, int n_limb, SubBox* box,
                             int cap, int& n_solves)
{
    constexpr int DEG = N * N + 1;
    struct Open { double t_cur, lx, ly; bool open; } op[64];
    int nb = 0;
    for (int s = 0; s <= n_limb; ++s) {
        const double ph = 2.0 * UL_PI * s / n_limb;
        const double px = wx + rho * cos(ph), py = wy + rho * sin(ph);
        double zr[DEG], zi[DEG]; unsigned mask = 0;
        centre_images<N>(L, T, px, py, zr, zi, mask);
        ++n_solves;
        bool used[64] = {false};
        for (int k = 0; k < DEG; ++k) {
            if (!((mask >> k) & 1u)) continue;
            double fx, fy, gx, gy, dm2;
            lens_resid<N>(L, zr[k], zi[k], px, py, fx, fy, gx, gy, dm2);
            if (fabs(1.0 - (gx * gx + gy * gy)) > 1e7) continue;
            double hr, ht, cr, ct;
            local_extents(zr[k], zi[k], gx, gy, rho, hr, ht, cr, ct);
            int best = -1; double bd = 0.0036 * ul_max(zr[k] * zr[k] + zi[k] * zi[k], 0.04);
            for (int b = 0; b < nb; ++b) {
                if (!op[b].open || used[b]) continue;
                double dx = zr[k] - op[b].lx, dy = zi[k] - op[b].ly, d = dx * dx + dy * dy;
                if (d < bd) { bd = d; best = b; }
            }
            if (best < 0) {
                if (nb == cap || nb == 64) continue;
                best = nb++;
                box[best].r_lo = 1.0; box[best].r_hi = -1.0; box[best].t_lo = box[best].t_hi = 0.0;
                box[best].hr = box[best].ht = box[best].cr = box[best].ct = 1e300;
                op[best].t_cur = 0.0; op[best].open = true;
            }
            used[best] = true;
            box_add(box[best], op[best].t_cur, sqrt(zr[k] * zr[k] + zi[k] * zi[k]), atan2(zi[k], zr[k]), hr, ht, cr, ct, true);
            op[best].lx = zr[k]; op[best].ly = zi[k];
        }
        for (int b = 0; b < nb; ++b) if (op[b].open && !used[b]) op[b].open = false;
    }
    for (int b = 0; b < nb; ++b) {
        // the boundary bulges beyond its samples by ~ (step)^2 / 8 x curvature: a margin instead of k_limb's parabola vertex
        double mr = 0.01 * (box[b].r_hi - box[b].r_lo), mt = 0.01 * (box[b].t_hi - box[b].t_lo);
        box[b].r_lo = ul_max(box[b].r_lo - mr, 0.0); box[b].r_hi += mr; box[b].t_lo -= mt; box[b].t_hi += mt;
        double sh = 2.0 * UL_PI * floor((box[b].t_lo + UL_PI) / (2.0 * UL_PI));
        box[b].t_lo -= sh; box[b].t_hi -= sh;
        if (box[b].t_hi - box[b].t_lo > 2.0 * UL_PI) box[b].t_hi = box[b].t_lo + 2.0 * UL_PI;
    }
    return nb;
}

template <int N, bool LD>
static int run(const Lens& L, double rho, double u1, double wx, double wy, RegionParams rp)
{
    constexpr int DEG = N * N + 1;
    LensPoly T; lens_poly_basis(N, L.eps, L.ax, L.ay, &T);
    double br[DEG + 1], bi[DEG + 1];
    poly_coeffs<N>(L, T, wx, wy, br, bi);
    for (int l = 0; l <= DEG; ++l) printf("coef %d %.17g %.17g\n", l, br[l], bi[l]);
    double zr[DEG], zi[DEG]; unsigned mask = 0;
    unsigned st = centre_images<N>(L, T, wx, wy, zr, zi, mask);
    for (int k = 0; k < DEG; ++k) printf("root %d %.17g %.17g %d\n", k, zr[k], zi[k], (int)((mask >> k) & 1));
    int n_solves = 0;
    static SubBox box[64];
    static Patch patch[UL_MAXP];
    const int nbox = limb_boxes_serial<N>(L, T, wx, wy, rho, rp.n_limb, box, 64, n_solves);
    int np = sectors_from_boxes<N>(box, nullptr, nbox, rp, 0, L, wx, wy, rho, st, nullptr, patch, nullptr);
    double tot = 0.0, tot_odd = 0.0; long long rays = 0; int clipped = 0;
    for (int p = 0; p < np; ++p) {
        const Patch& P = patch[p];
        printf("patch %d %.17g %.17g %.17g %.17g %d %d %d\n", p, P.r0, P.r0 + P.dr * P.n_r, P.th0, P.th0 + P.dth * P.n_th,
               P.n_r, P.n_th, P.flags);
        const int nl = 32 * P.n_units;
        for (int line = 0; line < nl; ++line) {
            double U, S, f; bool edge;
            if (P.flags & UL_PATCH_SCAN_R) {
                double th, wt; line_node(P.flags, P.n_th, line, P.th0, P.dth, th, wt);
                shoot_col<N, LD>(L, wx, wy, rho * rho, th, P.r0, P.dr, P.n_r, U, S, edge);
                f = (1.0 - u1) * U; if (LD) f += (u1 / rho) * S;
                f *= wt;
                rays += P.n_r + 4;
            } else {
                double r, wr; line_node(P.flags, P.n_r, line, P.r0, P.dr, r, wr);
                shoot_ring<N, LD>(L, wx, wy, rho * rho, r, P.th0, P.dth, P.n_th, (P.flags & UL_PATCH_PERIODIC) != 0, U, S, edge);
                f = (1.0 - u1) * U; if (LD) f += (u1 / rho) * S;
                f *= r * P.dth * wr;
                rays += P.n_th + 4;
            }
            clipped |= (int)edge;
            tot += f; if (line & 1) tot_odd += 2.0 * f;
        }
    }
    const double F0 = UL_PI * rho * rho * (1.0 - u1 / 3.0);
    printf("result %.17g %.17g %u %d %lld %d %d\n", tot / F0, fabs(tot - tot_odd) / (1.8284271247461903 * fabs(tot)), st, np, rays,
           n_solves, clipped);
    return 0;
}

int main(int argc, char** argv)
{
    int k = 1;
    Lens L; memset(&L, 0, sizeof L);
    L.n = atoi(argv[k++]);
    if (L.n < 1 || L.n > 3 || argc < 1 + 1 + 3 * L.n + 7) { fprintf(stderr, "bad arguments\n"); return 2; }
    for (int i = 0; i < L.n; ++i) L.eps[i] = atof(argv[k++]);
    for (int i = 0; i < L.n; ++i) L.ax[i] = atof(argv[k++]);
    for (int i = 0; i < L.n; ++i) L.ay[i] = atof(argv[k++]);
    const double rho = atof(argv[k++]), u1 = atof(argv[k++]), wx = atof(argv[k++]), wy = atof(argv[k++]);
    RegionParams rp;
    rp.n_limb = atoi(argv[k++]); rp.n_r = atoi(argv[k++]); rp.n_theta = atoi(argv[k++]);
    rp.max_nr = 8192; rp.max_nth = 32768; rp.max_units_pt = 1024;
    const bool ld = u1 > 0.0;
    if (L.n == 1) return ld ? run<1, true>(L, rho, u1, wx, wy, rp) : run<1, false>(L, rho, u1, wx, wy, rp);
    if (L.n == 2) return ld ? run<2, true>(L, rho, u1, wx, wy, rp) : run<2, false>(L, rho, u1, wx, wy, rp);
    return ld ? run<3, true>(L, rho, u1, wx, wy, rp) : run<3, false>(L, rho, u1, wx, wy, rp);
}
