// Host-compiled check of the device headers' per-thread / per-warp logic (test infrastructure only: the
// product has no CPU path -- ulens_create fails without a CUDA device). The .cuh files compile as plain C++;
// this runs, for ONE source point, exactly the code the kernels run: centre_images (k_roots), the three
// phases of the region builder lane by lane (k_regions), every scan line of every sector (k_shoot) and the
// ordered sum (k_finalize), and prints machine-readable lines for tests/test_host_logic.py.
//
// usage: host_logic N eps.. ax.. ay..  rho u1 wx wy n_limb n_r n_theta
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include "../paper_2510_02639_b200/csrc/ulens_core.cuh"
#include "../paper_2510_02639_b200/csrc/ulens_regions.cuh"
#include "../paper_2510_02639_b200/csrc/ulens_host.hpp"
using namespace ulens;

template <int N, bool LD>
static int run(const Lens& L, double rho, double u1, double wx, double wy, RegionParams rp)
{
    constexpr int DEG = N * N + 1;
    LensPoly T; lens_poly_basis(N, L.eps, L.ax, L.ay, &T);
    static RegionWork<DEG> W; W.ext = nullptr;
    double br[DEG + 1], bi[DEG + 1];
    poly_coeffs<N>(L, T, wx, wy, br, bi);
    for (int l = 0; l <= DEG; ++l) printf("coef %d %.17g %.17g\n", l, br[l], bi[l]);
    double zr[DEG], zi[DEG]; unsigned mask = 0;
    unsigned st = centre_images<N>(L, T, wx, wy, zr, zi, mask);
    for (int k = 0; k < DEG; ++k) printf("root %d %.17g %.17g %d\n", k, zr[k], zi[k], (int)((mask >> k) & 1));
    int n_solves = 0;
    for (int lane = 0; lane < 32; ++lane) {
        unsigned s = 0;
        regions_phaseA<N>(lane, L, T, wx, wy, rho, rp, W, s, n_solves, zr, zi, mask);
        st |= s;
    }
    for (int lane = 0; lane < 32; ++lane) regions_phaseB_keys<DEG>(lane, W);
    for (int lane = 0; lane < 32; ++lane) regions_phaseB<DEG>(lane, W);
    int np = regions_phaseC<N>(W, rp, 0, L, wx, wy, rho, st);
    double tot = 0.0, tot_odd = 0.0; long long rays = 0; int clipped = 0;
    for (int p = 0; p < np; ++p) {
        const Patch& P = W.patch[p];
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
