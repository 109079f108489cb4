// ulens_f32.cuh -- mixed-precision ray shooting (BASELINE.json north_star: "for a mixed-precision
// variant, FP32"): the rays of steps a5 / a6 on the FP32 pipe, FP64 only for segment constants, edge events and
// accumulation. Device code only (inline PTX for the approximate reciprocal / square root).
//
// Why plain FP32 does not work: F = |w(z) - w_c|^2 - rho^2 decides inside / outside, and w = z - sum eps_i/conj(z - a_i)
// with |z| ~ 1 carries an absolute rounding error ~1e-7 in single precision -- 1e-4 of a source of radius 1e-3.
// Cancellation-free difference form: a scan line is cut into SEGMENTS of up to 64 nodes around a reference ray z0 whose
// map is evaluated in FP64 (c_i = z0 - a_i, w0 = w(z0) - w_c, F0 = |w0|^2 - rho^2). For a ray z = z0 + d,
//     1/conj(c + d) - 1/conj(c) = -conj( d / (c (c + d)) )
//     w(z) - w_c = w0 + D,   D = d + sum_i eps_i conj( d / (c_i (c_i + d)) )
//     F = F0 + 2 Re(conj(w0) D) + |D|^2
// in which every FP32 operation acts on a quantity that is O(|d|) or O(rho): the rounding error of F is ~1e-7 of F's own
// scale (rho^2) times |d| / rho, instead of ~1e-7 / rho. The displacement d itself is formed without cancellation: along
// a radial line d = t (cos th, sin th); along a ring d = z0 (e^{i x} - 1) with x the angle from the reference ray and
// sin x, cos x - 1 from their Taylor series (|x| <= 1/2 by the choice of the segment length).
// The loop only needs the SIGN of F at every node (inside / outside) and sqrt(-F) on inside rays; where the sign changes
// between two nodes it notes the node, and the edge event (cubic root, Hurwitz-zeta end correction: two per line) is
// resolved after the loop in FP64 from four recomputed FP64 rays, by the very code the FP64 kernel uses (ring_event /
// col_event, ulens_core.cuh). Counts are integers, sums of sqrt(-F) are FP32 within a segment and FP64 across segments.
#pragma once
#include "ulens_core.cuh"

namespace ulens {

__device__ __forceinline__ float rcp_approx(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float sqrt_approx(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

#define UL_F32_BIG 1e30f

// segment constants (FP64 work, once per segment), held in FP32
template <int N>
struct SegRef {
    float cx[N], cy[N], eps[N];      // c_i = z0 - a_i
    float w0x, w0y, F0;              // w(z0) - w_c, |w0|^2 - rho^2
};

template <int N>
__device__ __forceinline__ void seg_ref(const Lens& L, double x0, double y0, double wcx, double wcy, double rho2, SegRef<N>& R)
{
    double ex = x0 - wcx, ey = y0 - wcy;
#pragma unroll
    for (int i = 0; i < N; ++i) {
        const double dx = x0 - L.ax[i], dy = y0 - L.ay[i];
        const double inv = L.eps[i] / (dx * dx + dy * dy);
        ex -= dx * inv; ey -= dy * inv;
        R.cx[i] = (float)dx; R.cy[i] = (float)dy; R.eps[i] = (float)L.eps[i];
    }
    const double F0 = ex * ex + ey * ey - rho2;
    // a reference ray on a lens (inf / NaN): the whole segment counts as outside
    const bool okv = F0 == F0 && fabs(F0) < 1e30;
    R.w0x = okv ? (float)ex : 0.0f; R.w0y = okv ? (float)ey : 0.0f; R.F0 = okv ? (float)F0 : UL_F32_BIG;
}

// F at the ray z0 + (dx, dy)
template <int N>
__device__ __forceinline__ float ray_F_f32(const SegRef<N>& R, float dx, float dy)
{
    float Dx = dx, Dy = dy;
#pragma unroll
    for (int i = 0; i < N; ++i) {
        const float ux = R.cx[i] + dx, uy = R.cy[i] + dy;
        const float px = R.cx[i] * ux - R.cy[i] * uy, py = R.cx[i] * uy + R.cy[i] * ux;      // c (c + d)
        const float inv = R.eps[i] * rcp_approx(px * px + py * py);
        // eps conj(d / p) = eps conj(d conj(p)) / |p|^2
        Dx += (dx * px + dy * py) * inv;
        Dy -= (dy * px - dx * py) * inv;
    }
    const float F = R.F0 + 2.0f * (R.w0x * Dx + R.w0y * Dy) + (Dx * Dx + Dy * Dy);
    return fminf(F, UL_F32_BIG);                          // fminf returns the non-NaN operand
}

// shoot_ring of ulens_core.cuh on the FP32 pipe. Same nodes, same rule; U, S as there (in cells).
template <int N, bool LD>
__device__ __forceinline__ void shoot_ring_f32(const Lens& L, double wcx, double wcy, double rho2, double r, double th0,
                                               double dth, int n_th, bool periodic, double& U_out, double& S_out, bool& edge)
{
    // segment half-length: |x| = |j - jc| dth <= 1/2 so that the Taylor series below hold to 1e-8
    int half = (int)(0.5 / dth);
    half = half > 32 ? 32 : (half < 1 ? 1 : half);
    const float dthf = (float)dth;
    float f1 = UL_F32_BIG, f2 = UL_F32_BIG;
    double U = 0.0, S = 0.0;
    edge = false;
    const int j_first = periodic ? 2 : 1;
    const double cd = cos(dth), sd = sin(dth);
    int npend = 0, pj0 = 0, pj1 = 0;
    unsigned pen = 0;
    // reference ray of the first segment, then rotated from segment to segment in FP64
    double sn, cs, sstep, cstep;
    sincos(th0 + (-2 + half + 0.5) * dth, &sn, &cs);
    sincos(2.0 * half * dth, &sstep, &cstep);
    for (int j0 = -2; j0 <= n_th + 1; j0 += 2 * half) {
        SegRef<N> R;
        const double x0 = r * cs, y0 = r * sn;
        seg_ref<N>(L, x0, y0, wcx, wcy, rho2, R);
        const float zx = (float)x0, zy = (float)y0;
        int cnt = 0; float ssum = 0.0f;
        const int j1 = min(j0 + 2 * half - 1, n_th + 1);
#pragma unroll 2
        for (int j = j0; j <= j1; ++j) {
            const float x = (float)(j - j0 - half) * dthf, x2 = x * x;
            const float s = x * (1.0f + x2 * (-1.0f / 6.0f + x2 * (1.0f / 120.0f - x2 * (1.0f / 5040.0f))));
            const float cm1 = x2 * (-0.5f + x2 * (1.0f / 24.0f + x2 * (-1.0f / 720.0f + x2 * (1.0f / 40320.0f))));
            const float f3 = ray_F_f32<N>(R, zx * cm1 - zy * s, zx * s + zy * cm1);       // d = z0 (e^{ix} - 1)
            if (j >= 0 && j < n_th && f3 < 0.0f) {
                ++cnt;
                if (LD) ssum += sqrt_approx(-f3);
                if (!periodic && (j < 2 || j >= n_th - 2)) edge = true;
            }
            if (j >= j_first && ((f1 < 0.0f) != (f2 < 0.0f))) {
                if (npend == 2) {
                    ring_event<N, LD>(L, wcx, wcy, rho2, r, th0, dth, cd, sd, pj0, (pen & 1u) != 0, U, S);
                    pj0 = pj1; pen >>= 1; npend = 1;
                }
                if (npend == 0) pj0 = j; else pj1 = j;
                if (!(f1 < 0.0f)) pen |= 1u << npend;
                ++npend;
            }
            f1 = f2; f2 = f3;
        }
        U += (double)cnt; S += (double)ssum;
        const double cn = cs * cstep - sn * sstep;
        sn = sn * cstep + cs * sstep; cs = cn;
    }
    if (npend > 0) ring_event<N, LD>(L, wcx, wcy, rho2, r, th0, dth, cd, sd, pj0, (pen & 1u) != 0, U, S);
    if (npend > 1) ring_event<N, LD>(L, wcx, wcy, rho2, r, th0, dth, cd, sd, pj1, (pen & 2u) != 0, U, S);
    U_out = U; S_out = S;
}

// shoot_col of ulens_core.cuh on the FP32 pipe: radial line at angle th, nodes r0 + (i + 1/2) dr.
template <int N, bool LD>
__device__ __forceinline__ void shoot_col_f32(const Lens& L, double wcx, double wcy, double rho2, double th, double r0,
                                              double dr, int n_r, double& U_out, double& S_out, bool& edge)
{
    double sn, cs;
    sincos(th, &sn, &cs);
    const float cf = (float)cs, sf = (float)sn, drf = (float)dr;
    constexpr int half = 32;
    float f1 = UL_F32_BIG, f2 = UL_F32_BIG;
    double U = 0.0, S = 0.0, U2 = 0.0;
    edge = false;
    int npend = 0, pi0 = 0, pi1 = 0;
    unsigned pen = 0;
    for (int i0 = -2; i0 <= n_r + 1; i0 += 2 * half) {
        const double rc = r0 + (i0 + half + 0.5) * dr;     // reference node i0 + half
        SegRef<N> R;
        seg_ref<N>(L, rc * cs, rc * sn, wcx, wcy, rho2, R);
        int cnt = 0; float tsum = 0.0f, ssum = 0.0f, tssum = 0.0f;
        const int i1 = min(i0 + 2 * half - 1, n_r + 1);
#pragma unroll 2
        for (int i = i0; i <= i1; ++i) {
            const float t = (float)(i - i0 - half) * drf;
            const float f3 = ray_F_f32<N>(R, t * cf, t * sf);
            if (i >= 0 && i < n_r && f3 < 0.0f) {
                ++cnt; tsum += t;
                if (LD) { const float sq = sqrt_approx(-f3); ssum += sq; tssum += t * sq; }
                if ((i < 2 && r0 > 0.0) || i >= n_r - 2) edge = true;
            }
            // pair (i-2, i-1) = (f1, f2); the cell face between the pair must lie at r > 0
            if (i >= 1 && ((f1 < 0.0f) != (f2 < 0.0f)) && (r0 + (i - 1.0) * dr > 0.0)) {
                if (npend == 2) {
                    col_event<N, LD>(L, wcx, wcy, rho2, cs, sn, r0, dr, pi0, (pen & 1u) != 0, U2, S);
                    pi0 = pi1; pen >>= 1; npend = 1;
                }
                if (npend == 0) pi0 = i; else pi1 = i;
                if (!(f1 < 0.0f)) pen |= 1u << npend;
                ++npend;
            }
            f1 = f2; f2 = f3;
        }
        // sum over the inside nodes of r = rc + t, and of r sqrt(-F)
        U += (double)cnt * rc + (double)tsum;
        S += rc * (double)ssum + (double)tssum;
    }
    if (npend > 0) col_event<N, LD>(L, wcx, wcy, rho2, cs, sn, r0, dr, pi0, (pen & 1u) != 0, U2, S);
    if (npend > 1) col_event<N, LD>(L, wcx, wcy, rho2, cs, sn, r0, dr, pi1, (pen & 2u) != 0, U2, S);
    U_out = U * dr + U2; S_out = S * dr;
}

}  // namespace ulens
