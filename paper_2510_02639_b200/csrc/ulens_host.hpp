// ulens_host.hpp -- host-side set-up arithmetic of the C ABI (once per lens, not per point).
#pragma once
#include <string.h>
#include "ulens_core.cuh"

// T_k = Q^k G^(N-k) in long double (host, once per lens)
namespace {
struct LPoly { int deg; long double re[12], im[12]; };
inline LPoly lp_const(long double v) { LPoly p; memset(&p, 0, sizeof p); p.deg = 0; p.re[0] = v; return p; }
inline LPoly lp_mul(const LPoly& a, const LPoly& b)
{
    LPoly p; memset(&p, 0, sizeof p); p.deg = a.deg + b.deg;
    for (int i = 0; i <= a.deg; ++i)
        for (int j = 0; j <= b.deg; ++j) {
            p.re[i + j] += a.re[i] * b.re[j] - a.im[i] * b.im[j];
            p.im[i + j] += a.re[i] * b.im[j] + a.im[i] * b.re[j];
        }
    return p;
}
inline LPoly lp_add(const LPoly& a, const LPoly& b)
{
    LPoly p; memset(&p, 0, sizeof p); p.deg = a.deg > b.deg ? a.deg : b.deg;
    for (int i = 0; i <= a.deg; ++i) { p.re[i] += a.re[i]; p.im[i] += a.im[i]; }
    for (int i = 0; i <= b.deg; ++i) { p.re[i] += b.re[i]; p.im[i] += b.im[i]; }
    return p;
}
inline void lens_poly_basis(int N, const double* eps, const double* ax, const double* ay, ulens::LensPoly* out)
{
    memset(out, 0, sizeof *out);
    LPoly lin[3];
    for (int i = 0; i < N; ++i) { memset(&lin[i], 0, sizeof(LPoly)); lin[i].deg = 1; lin[i].re[0] = -(long double)ax[i]; lin[i].im[0] = -(long double)ay[i]; lin[i].re[1] = 1; }
    LPoly Q = lp_const(1), G = lp_const(0);
    for (int i = 0; i < N; ++i) Q = lp_mul(Q, lin[i]);
    for (int i = 0; i < N; ++i) {
        LPoly t = lp_const((long double)eps[i]);
        for (int m = 0; m < N; ++m) if (m != i) t = lp_mul(t, lin[m]);
        G = lp_add(G, t);
    }
    for (int k = 0; k <= N; ++k) {
        LPoly t = lp_const(1);
        for (int a = 0; a < k; ++a) t = lp_mul(t, Q);
        for (int a = 0; a < N - k; ++a) t = lp_mul(t, G);
        for (int l = 0; l <= t.deg && l < 10; ++l) { out->tr[k][l] = (double)t.re[l]; out->ti[k][l] = (double)t.im[l]; }
    }
}
}  // namespace
