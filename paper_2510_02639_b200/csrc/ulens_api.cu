// ulens_api.cu -- kernels and C ABI (include/ulens.h) of the B200-native ICRS hot path.
//
// Pipeline per chunk of source points (all on the caller's stream, no host round trip in between):
//   k_traj      (lightcurve entry only)  trajectory -> source centres
//   k_roots     thread per point: lens polynomial, Ehrlich-Aberth, validate + polish         Eq. 4, 7
//   k_limb      CTA per point, lane per root: limb images -> boxes of the image arcs          Sec. 3.2, Eq. 8
//   k_sectors   thread per point: boxes -> polar sectors -> 32-line work units                 Sec. 3.2
//   k_shoot     warp per work unit, lane per ring: rays along theta, edge events, ring sums  Sec. 3.3, App. A
//   k_finalize  thread per point: ordered sum of its units, normalise                        Eq. A5
//
// There is no CPU implementation behind this ABI: without a CUDA device every entry point fails.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>
#include <new>
#include <vector>

#include "../../include/ulens.h"
#include "ulens_core.cuh"
#include "ulens_dual.cuh"
#include "ulens_regions.cuh"
#include "ulens_limb.cuh"
#include "ulens_f32.cuh"
#include "ulens_host.hpp"

using namespace ulens;

// ------------------------------------------------------------------------------------------------ context

struct DevCounters {
    unsigned long long n_rays, n_patches, n_units, n_limb_solves, n_flagged, n_points;
};

struct ChunkCounters {          // reset per chunk
    unsigned int n_units;       // units allocated by k_regions
    unsigned int next_unit;     // dynamic scheduler of k_shoot
    unsigned int n_quiet;       // k_quiet: quiet points (listed from the front of limb_list) ...
    unsigned int n_full;        // ... and the others (listed from its back)
};

#define UL_N_STAGE 8
#define UL_MAX_POINTS (0x7fffffffLL - 4096)    // grid arithmetic (n + 1023) stays inside int
struct ulens_ctx {
    int device;
    ulens_options opt;
    RegionParams rp;
    int chunk;
    size_t cap_units;
    // workspace (device)
    Patch* patches;             // [chunk][UL_MAXP]
    int* n_patch;               // [chunk]
    unsigned* status_ws;        // [chunk]
    double* c_zr; double* c_zi; // [chunk][10] roots of the source centre (k_roots -> k_regions)
    unsigned* c_mask;           // [chunk]     which of them are images
    SubBox* boxes; int boxes_cap;       // [chunk][BoxCap] box lists of the points (k_limb -> k_sectors); boxes_cap = BoxCap allocated
    BoxExt* exts; int exts_cap;         // forward-mode runs: the boxes' extreme own points
    int* n_boxes;               // [chunk]
    unsigned char* quiet;       // [chunk] 1 = quiet source point (k_quiet): coarse limb sampling
    int* limb_list;             // [chunk] k_quiet -> k_limb: quiet points from the front, the others from the back
    double* quiet_drho;         // [chunk] quiet points: dA/drho from the probe (forward-mode runs)
    // forward-mode variant (allocated on first use)
    PatchTan* ptans;            // [chunk][UL_MAXP] tangents of the sectors' radial bounds
    double* unit_tan; int unit_tan_nt;  // [cap_units][NT] tangent sums of the units
    double* grad5;              // [chunk][UL_NT] intrinsic gradient dA/d(w_cx, w_cy, s, q, rho)
    TangentTable* tan_dev; size_t tan_cap;
    unsigned* unit_desc;        // [cap_units]  (patch slot << 11) | line block (< 2048)
    double* unit_sum;           // [cap_units]  all rings
    double* unit_odd;           // [cap_units]  odd rings only (half-resolution self-check)
    ChunkCounters* cc;
    DevCounters* counters;
    PointCfg* cfg_dev; LensPoly* poly_dev; size_t cfg_cap;
    double* traj_w; size_t traj_cap;    // lightcurve entry: source centres [2][n]
    double* io_buf; size_t io_cap;      // *_host entry: staging
    // point-source / finite-source switch (ulens_lightcurve_binary_ext): flags, block offsets, gather map
    unsigned char* ext_flag; int* ext_map; unsigned* ext_blk; size_t ext_cap;
    unsigned* st_all; size_t st_all_cap;    // status of every point when the caller passes none (the retry pass reads it)
    int last_launches;
    // host -> device uploads of the per-configuration tables go through context-owned PINNED staging buffers
    // (a pageable cudaMemcpyAsync would synchronise the stream first); a slot is reused only after the copy
    // that read it has completed (its event), so no entry point has to wait for the stream
    struct Stage { void* host; size_t cap; cudaEvent_t ev; bool used; };
    Stage stage[UL_N_STAGE]; int stage_next;
    // the tables of the last call: an identical (lenses, rho, u1) array is neither rebuilt nor uploaded again
    std::vector<ulens_lens>* last_lenses; std::vector<double>* last_rho; std::vector<double>* last_u1;
    int last_N; bool last_ld; bool last_tan_valid;
    // optional per-kernel device timing (ulens_set_timing): event pairs recorded on the caller's stream
    int timing_on;
    struct TimedLaunch { cudaEvent_t a, b; int which; };
    std::vector<TimedLaunch>* timed;
    double k_ms[ULENS_K_COUNT]; int k_launches[ULENS_K_COUNT];
    char cuda_err[256];
};

// RAII-free helper: record an event pair around one launch when timing is on
struct KTimer {
    ulens_ctx* c; cudaStream_t st; cudaEvent_t a, b; int which; bool on;
    KTimer(ulens_ctx* ctx, int w, cudaStream_t s) : c(ctx), st(s), a(nullptr), b(nullptr), which(w), on(ctx->timing_on != 0)
    {
        if (on) { cudaEventCreate(&a); cudaEventCreate(&b); cudaEventRecord(a, st); }
    }
    ~KTimer()
    {
        if (on) { cudaEventRecord(b, st); c->timed->push_back({a, b, which}); }
    }
};

static int fail_cuda(ulens_ctx* c, cudaError_t e, const char* where)
{
    if (c) snprintf(c->cuda_err, sizeof c->cuda_err, "%s: %s", where, cudaGetErrorString(e));
    return ULENS_ECUDA;
}
#define CK(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return fail_cuda(ctx, e_, #call); } while (0)

// ------------------------------------------------------------------------------------------------ host geometry

static bool finite_pos(double x) { return isfinite(x) && x > 0.0; }

extern "C" int ulens_lens_binary(ulens_lens* out, double s, double q)
{
    if (!out || !finite_pos(s) || !finite_pos(q)) return ULENS_EINVAL;
    memset(out, 0, sizeof *out);
    out->n_lens = 2;
    out->eps[0] = 1.0 / (1.0 + q);
    out->eps[1] = q / (1.0 + q);
    out->ax[0] = -s * q / (1.0 + q);          // G4: primary at negative x, barycentre of M1, M2 at the origin
    out->ax[1] = s / (1.0 + q);
    return ULENS_OK;
}

extern "C" int ulens_lens_triple(ulens_lens* out, double s, double q, double q3, double r3, double psi)
{
    if (!out || !finite_pos(s) || !finite_pos(q) || !(q3 >= 0.0) || !isfinite(q3) || !finite_pos(r3) || !isfinite(psi))
        return ULENS_EINVAL;
    memset(out, 0, sizeof *out);
    double tot = 1.0 + q + q3;
    out->n_lens = 3;
    out->eps[0] = 1.0 / tot; out->eps[1] = q / tot; out->eps[2] = q3 / tot;
    out->ax[0] = -s * q / (1.0 + q);
    out->ax[1] = s / (1.0 + q);
    double mid = 0.5 * (out->ax[0] + out->ax[1]);      // G5: M3 at polar (r3, psi) from the midpoint of M1-M2
    out->ax[2] = mid + r3 * cos(psi);
    out->ay[2] = r3 * sin(psi);
    return ULENS_OK;
}


// ------------------------------------------------------------------------------------------------ kernels

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// trajectory (G3): tau = (t - t0)/tE,  w = (tau cos a - u0 sin a) + i (tau sin a + u0 cos a)
__global__ void k_traj(int n_cfg, int n_ep, const double* __restrict__ theta, const double* __restrict__ t,
                       double* __restrict__ w_re, double* __restrict__ w_im)
{
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)n_cfg * n_ep) return;
    int c = (int)(i / n_ep), e = (int)(i % n_ep);
    const double* th = theta + 7 * c;
    double tau = (t[e] - th[0]) / th[2];
    double ca = cos(th[6]), sa = sin(th[6]);
    w_re[i] = tau * ca - th[1] * sa;
    w_im[i] = tau * sa + th[1] * ca;
}

// One thread per source point: all roots, image flags, images polished on Eq. 1.
// out_* may be NULL (then only the status word is produced).
template <int N>
__global__ void k_roots(int n, int pt_base, int n_pts_per_cfg, const PointCfg* __restrict__ cfg,
                        const LensPoly* __restrict__ poly, const double* __restrict__ w_re,
                        const double* __restrict__ w_im, double* __restrict__ out_re, double* __restrict__ out_im,
                        uint8_t* __restrict__ out_img, unsigned* __restrict__ status,
                        double* __restrict__ c_zr, double* __restrict__ c_zi, unsigned* __restrict__ c_mask,
                        double* __restrict__ A_ps = nullptr, unsigned* __restrict__ status_global = nullptr,
                        const int* __restrict__ pmap = nullptr, const unsigned* __restrict__ n_dev = nullptr)
{
    constexpr int DEG = N * N + 1;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (n_dev) n = min(n, (int)*n_dev - pt_base);    // retry pass: the point count lives on the device
    if (i >= n) return;
    long long gp = pmap ? (long long)pmap[pt_base + i] : (long long)pt_base + i;
    int c = (int)(gp / n_pts_per_cfg);
    Lens L = cfg[c].lens;
    double wx = w_re[gp], wy = w_im[gp];
    double zr[DEG], zi[DEG];
    unsigned mask = 0;
    unsigned st = centre_images<N>(L, poly[c], wx, wy, zr, zi, mask);
    if (status) status[i] = st;
    if (A_ps) {
        // point-source magnification (Eq. 2-3): A = sum over the images of 1 / |det J|, det J = 1 - |g|^2
        double a = 0.0;
#pragma unroll
        for (int k = 0; k < DEG; ++k) {
            if (!((mask >> k) & 1u)) continue;
            double fx, fy, gx, gy, dm2;
            lens_resid<N>(L, zr[k], zi[k], wx, wy, fx, fy, gx, gy, dm2);
            a += 1.0 / fabs(1.0 - (gx * gx + gy * gy));
        }
        A_ps[gp] = a;
        if (status_global) status_global[gp] = st;
    }
    if (c_zr) {
#pragma unroll
        for (int k = 0; k < DEG; ++k) { c_zr[(long long)i * 10 + k] = zr[k]; c_zi[(long long)i * 10 + k] = zi[k]; }
        c_mask[i] = mask;
    }
    if (out_re) {
#pragma unroll
        for (int k = 0; k < DEG; ++k) {
            out_re[(long long)i * DEG + k] = zr[k];
            out_im[(long long)i * DEG + k] = zi[k];
            out_img[(long long)i * DEG + k] = (mask >> k) & 1u;
        }
    }
}


// ------------------------------------------------------------------------------------------------
// Point-source / finite-source switch ("(iii) ... only a preselected set of N_ext epochs
// (e.g., near caustics) are modeled" with the extended source; the other epochs take Eq. 2-3).
// ------------------------------------------------------------------------------------------------

// Point-source magnification of one source position, A = sum_j 1/|D_j|, D = det J = 1 - |g|^2 (Eq. 2-3), from the
// images already found (zr, zi, mask) and, if tt != nullptr, its tangents in the UL_NT intrinsic directions by
// implicit differentiation of Eq. 1 at every image (P:163-175 does this through the polynomial; the lens
// equation itself is better conditioned). With d_i = z - a_i, g_i = eps_i/conj(d_i)^2, g = sum_i g_i:
//   delta w = dz + g conj(dz) - sum_i g_i conj(da_i) - sum_i deps_i/conj(d_i)
//   =>  dz = (R - g conj(R))/D,   R = dw + sum_i g_i conj(da_i) + sum_i deps_i/conj(d_i)
//   dg = sum_i deps_i/conj(d_i)^2 - 2 sum_i eps_i conj(dz - da_i)/conj(d_i)^3
//   dA_j = sign(D) d|g|^2/D^2,   d|g|^2 = 2 Re(conj(g) dg)
template <int N>
__device__ double point_mag(const Lens& L, const TangentTable* tt, const double* zr, const double* zi, unsigned mask,
                            double* g5)
{
    constexpr int DEG = N * N + 1;
    double A = 0.0;
    if (g5) for (int k = 0; k < UL_NT; ++k) g5[k] = 0.0;
#pragma unroll 1
    for (int j = 0; j < DEG; ++j) {
        if (!((mask >> j) & 1u)) continue;
        double qx[N], qy[N];        // 1/conj(d_i) = d_i/|d_i|^2
        double gx = 0.0, gy = 0.0;
#pragma unroll
        for (int i = 0; i < N; ++i) {
            double dx = zr[j] - L.ax[i], dy = zi[j] - L.ay[i];
            double inv = 1.0 / (dx * dx + dy * dy);
            qx[i] = dx * inv; qy[i] = dy * inv;
            gx += L.eps[i] * (qx[i] * qx[i] - qy[i] * qy[i]);
            gy += L.eps[i] * (2.0 * qx[i] * qy[i]);
        }
        const double D = 1.0 - (gx * gx + gy * gy);
        A += 1.0 / fabs(D);
        if (!g5) continue;
        const double sD = (D >= 0.0 ? 1.0 : -1.0) / (D * D);
#pragma unroll 1
        for (int k = 0; k < UL_NT; ++k) {
            double Rx = tt->dwx[k], Ry = tt->dwy[k];
#pragma unroll
            for (int i = 0; i < N; ++i) {
                double q2x = qx[i] * qx[i] - qy[i] * qy[i], q2y = 2.0 * qx[i] * qy[i];      // 1/conj(d)^2
                double gix = L.eps[i] * q2x, giy = L.eps[i] * q2y;
                double ax = tt->dax[k][i], ay = -tt->day[k][i];                             // conj(da_i)
                Rx += gix * ax - giy * ay + tt->deps[k][i] * qx[i];
                Ry += gix * ay + giy * ax + tt->deps[k][i] * qy[i];
            }
            // dz = (R - g conj(R))/D
            double dzx = (Rx - (gx * Rx + gy * Ry)) / D;
            double dzy = (Ry - (gy * Rx - gx * Ry)) / D;
            double dgx = 0.0, dgy = 0.0;
#pragma unroll
            for (int i = 0; i < N; ++i) {
                double q2x = qx[i] * qx[i] - qy[i] * qy[i], q2y = 2.0 * qx[i] * qy[i];
                double q3x = q2x * qx[i] - q2y * qy[i], q3y = q2x * qy[i] + q2y * qx[i];    // 1/conj(d)^3
                double cx = dzx - tt->dax[k][i], cy = -(dzy - tt->day[k][i]);               // conj(dz - da_i)
                dgx += tt->deps[k][i] * q2x - 2.0 * L.eps[i] * (cx * q3x - cy * q3y);
                dgy += tt->deps[k][i] * q2y - 2.0 * L.eps[i] * (cx * q3y + cy * q3x);
            }
            g5[k] += sD * 2.0 * (gx * dgx + gy * dgy);
        }
    }
    return A;
}

// One thread per epoch: point-source A (and tangents) of the source centre, and the decision which path the epoch takes.
//   mask_in != nullptr: the caller preselected the finite-source epochs (the paper's reading).
//   mask_in == nullptr: [proposal] multipole probe. A_ps is evaluated at 8 points of the limb (4 on the axes,
//     4 on the diagonals). For a source that no caustic touches, the disk average of A_ps differs from A_ps(centre)
//     by rho^2/8 lap A + O(rho^4) (uniform; less when limb-darkened) and the mean over the 8 limb points by
//     rho^2/4 lap A + O(rho^4), so  Q = |mean_8 - A_c|/2  estimates the finite-source correction and
//     H = |mean_axes - mean_diagonals| the size of the fourth-order term. The epoch keeps the point-source value
//     when every probe has as many images as the centre (no caustic between them) and Q + H <= sel_tol * A_c.
template <int N>
__global__ void k_point_ext(int n, int n_pts_per_cfg, const PointCfg* __restrict__ cfg, const LensPoly* __restrict__ poly,
                            const TangentTable* __restrict__ tans, const double* __restrict__ w_re,
                            const double* __restrict__ w_im, const unsigned char* __restrict__ mask_in, double sel_tol,
                            double* __restrict__ A_out, double* __restrict__ err_out, unsigned* __restrict__ status_out,
                            double* __restrict__ grad5, unsigned char* __restrict__ flag_out)
{
    constexpr int DEG = N * N + 1;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int c = i / n_pts_per_cfg;
    Lens L = cfg[c].lens;
    const double rho = cfg[c].rho;
    const double wx = w_re[i], wy = w_im[i];
    double zr[DEG], zi[DEG], g5[UL_NT];
    double A_c = 0.0, s_axes = 0.0, s_diag = 0.0;
    unsigned st_c = 0;
    bool ext = mask_in ? (mask_in[i] != 0) : false;
    const int n_probe = mask_in ? 1 : 9;
#pragma unroll 1
    for (int p = 0; p < n_probe; ++p) {
        double px = wx, py = wy;
        if (p > 0) {
            const double r = (p > 4) ? rho * 0.70710678118654752 : rho;
            const int k = (p - 1) & 3;
            const double ex = (k == 0) ? 1.0 : (k == 2) ? -1.0 : 0.0, ey = (k == 1) ? 1.0 : (k == 3) ? -1.0 : 0.0;
            if (p > 4) { px += r * (ex - ey); py += r * (ex + ey); }     // diagonals: e rotated by pi/4, |.| = rho
            else { px += r * ex; py += r * ey; }
        }
        unsigned mask = 0;
        // (the limb probes start the simultaneous iteration from the previous probe's roots, as in k_quiet)
        unsigned st = centre_images<N>(L, poly[c], px, py, zr, zi, mask, p > 0);
        if (p == 0) {
            st_c = st;
            A_c = point_mag<N>(L, grad5 ? &tans[c] : nullptr, zr, zi, mask, grad5 ? g5 : nullptr);
            if (st & (UL_ST_EA_NOCONV | UL_ST_IMG_PARITY)) ext = ext || !mask_in;     // doubtful centre: integrate
        } else {
            double a = point_mag<N>(L, nullptr, zr, zi, mask, nullptr);
            if (((st ^ st_c) >> 8) & 0xfu) ext = true;                              // image count changed
            if (st & (UL_ST_EA_NOCONV | UL_ST_IMG_PARITY)) ext = true;
            if (p > 4) s_diag += a; else s_axes += a;
        }
    }
    if (!mask_in && !ext) {
        const double Q = 0.5 * fabs(0.125 * (s_axes + s_diag) - A_c);
        const double H = 0.25 * fabs(s_axes - s_diag);
        if (!(Q + H <= sel_tol * A_c)) ext = true;
    }
    flag_out[i] = ext ? 1 : 0;
    A_out[i] = A_c;
    if (err_out) err_out[i] = 0.0;
    if (status_out) status_out[i] = st_c | UL_ST_POINT_SRC;
    if (grad5) for (int k = 0; k < UL_NT; ++k) grad5[(long long)i * UL_NT + k] = g5[k];
}

// which points the retry pass takes: a doubtful finite-source result (not the centre's image parity, which is
// informational, nor a resolution cap, which more limb points cannot lift); never a point-source epoch
#define UL_ST_RETRY_MASK (UL_ST_EA_NOCONV | UL_ST_PATCH_CAP | UL_ST_CLIPPED | UL_ST_ERR_HIGH | UL_ST_NO_IMAGE)
__global__ void k_retry_flag(int n, const unsigned* __restrict__ status, unsigned char* __restrict__ flag)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    unsigned st = status[i];
    flag[i] = ((st & UL_ST_RETRY_MASK) && !(st & UL_ST_POINT_SRC)) ? 1 : 0;
}

// ordered stream compaction of the flagged epochs into the gather map (three small kernels, 1024 epochs per block)
__global__ void k_ext_count(int n, const unsigned char* __restrict__ flag, unsigned* __restrict__ blk)
{
    __shared__ unsigned wsum[32];
    int i = blockIdx.x * 1024 + threadIdx.x;
    unsigned b = __ballot_sync(0xffffffffu, i < n && flag[i]);
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = __popc(b);
    __syncthreads();
    if (threadIdx.x < 32) {
        unsigned v = wsum[threadIdx.x];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (threadIdx.x == 0) blk[blockIdx.x] = v;
    }
}
// exclusive scan of the block counts by one block (n_blk <= a few thousand); blk[n_blk] = total
__global__ void k_ext_scan(int n_blk, unsigned* __restrict__ blk)
{
    __shared__ unsigned part[1024];
    const int per = (n_blk + 1023) / 1024;
    const int lo = threadIdx.x * per, hi = min(lo + per, n_blk);
    unsigned s = 0;
    for (int j = lo; j < hi; ++j) s += blk[j];
    part[threadIdx.x] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned run = 0;
        for (int j = 0; j < 1024; ++j) { unsigned v = part[j]; part[j] = run; run += v; }
        blk[n_blk] = run;
    }
    __syncthreads();
    unsigned run = part[threadIdx.x];
    for (int j = lo; j < hi; ++j) { unsigned v = blk[j]; blk[j] = run; run += v; }
}
__global__ void k_ext_scatter(int n, const unsigned char* __restrict__ flag, const unsigned* __restrict__ blk,
                              int* __restrict__ map)
{
    __shared__ unsigned wsum[32];
    int i = blockIdx.x * 1024 + threadIdx.x;
    const bool f = i < n && flag[i];
    unsigned b = __ballot_sync(0xffffffffu, f);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) wsum[w] = __popc(b);
    __syncthreads();
    if (threadIdx.x < 32) {
        unsigned v = wsum[threadIdx.x], inc = v;
        for (int o = 1; o < 32; o <<= 1) { unsigned t = __shfl_up_sync(0xffffffffu, inc, o); if (threadIdx.x >= o) inc += t; }
        wsum[threadIdx.x] = inc - v;
    }
    __syncthreads();
    if (f) map[blk[blockIdx.x] + wsum[w] + __popc(b & ((1u << l) - 1u))] = i;
}

// Quiet source points [proposal]. Far from every caustic the images are smooth near-ellipses and an eighth of the limb
// samples bounds them as well as all of them; the limb tracker is the second most expensive step, so such points are
// worth recognising. Same multipole probe as the point-source switch (k_point_ext): the point-source magnification at
// the centre and at 8 limb points; the point is quiet when every probe has as many images as the centre (no caustic
// between them), every solve is clean, and Q + H <= tol A_c, i.e. the finite-source effect itself is below tol.
// Only the sampling density changes: the images are still found by tracking, the rays still decide what is inside.
#ifndef UL_QUIET_TOL
#define UL_QUIET_TOL 1e-4
#endif
// Ray grid of the quiet points relative to ulens_options.n_r (scan lines per half-extent) and n_theta (nodes per half-chord
// along a line). Measured over every point of C1-C3 against the full grid: half the lines cost a broad
// ~2e-5 (largest 4e-5), half the nodes a heavy tail (1.3e-4 on 3 points: refused); (0.5, 0.75) keeps the largest
// difference at 4.3e-5 and the largest error on the stored oracle samples at 5.0e-5, for 56 % fewer rays on those points.
// Ray grid of a quiet point's sectors that end at the true extremes of their image (ulens_regions.cuh quiet_image_extremes),
// relative to ulens_options.n_r (scan lines per half-extent) and n_theta (nodes per half-chord along a line). Measured over
// every point of C1-C3 and 1.4 M random-lens points against the full treatment, and on the stored oracle samples
// (DESIGN.md 5.3): with exact ends (3/8, 3/4) stays within 3.3e-5 of the full grid; 5/8 of the nodes puts single points at
// 6.7e-5 (refused); a quarter of the lines costs a broad 2e-5 ... 5e-5 (refused).
#ifndef UL_QUIET_LIMB_DIV
#define UL_QUIET_LIMB_DIV 8       // quiet points: n_limb / this many limb samples (16: 2 points each of C1 and C3 wrong by 1e-2 ... 3.5e-2: refused)
#endif
#ifndef UL_QUIET_RES_LINES
#define UL_QUIET_RES_LINES 0.375
#endif
#ifndef UL_QUIET_RES_NODES
#define UL_QUIET_RES_NODES 0.75
#endif
template <int N>
__global__ void k_quiet(int n, int pt_base, int n_pts_per_cfg, const PointCfg* __restrict__ cfg, const LensPoly* __restrict__ poly,
                        const double* __restrict__ w_re, const double* __restrict__ w_im, double tol,
                        unsigned char* __restrict__ quiet, double* __restrict__ quiet_drho, int* __restrict__ limb_list,
                        ChunkCounters* cc, const int* __restrict__ pmap = nullptr, const unsigned* __restrict__ n_dev = nullptr)
{
    constexpr int DEG = N * N + 1;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (n_dev) n = min(n, (int)*n_dev - pt_base);
    const bool live = i < n;                             // (no early return: the warp lists its points together)
    const long long gp = !live ? 0 : (pmap ? (long long)pmap[pt_base + i] : (long long)pt_base + i);
    const int c = (int)(gp / n_pts_per_cfg);
    const Lens L = cfg[c].lens;
    const double rho = cfg[c].rho, wx = w_re[gp], wy = w_im[gp];
    double zr[DEG], zi[DEG];
    double A_c = 0.0, s_axes = 0.0, s_diag = 0.0;
    unsigned st_c = 0;
    bool ok = live;
    // never next to a light lens: within 8 sqrt(eps_a) + 2 rho of its planetary caustic (centred on
    // w_a = a_a - sum_{b != a} eps_b / conj(a_a - a_b)) images hide in a root cluster that the polynomial solve -- and
    // with it this probe -- can miss altogether (measured on C3: a pair of 4.5e-4 A each, found only by the limb
    // tracker's seeds on that lens's Einstein ring, which need the dense sampling)
    if (N > 1) {
#pragma unroll
        for (int a = 0; a < N; ++a) {
            if (!(L.eps[a] < 1e-2)) continue;
            double tx = L.ax[a] - wx, ty = L.ay[a] - wy;
#pragma unroll
            for (int b = 0; b < N; ++b) {
                if (b == a) continue;
                const double dx = L.ax[a] - L.ax[b], dy = L.ay[a] - L.ay[b];
                const double i2 = L.eps[b] / (dx * dx + dy * dy);
                tx -= dx * i2; ty -= dy * i2;
            }
            const double R = 8.0 * sqrt(L.eps[a]) + 2.0 * rho;
            if (tx * tx + ty * ty < R * R) ok = false;
        }
    }
#pragma unroll 1
    for (int p = 0; p < 9 && ok; ++p) {
        double px = wx, py = wy;
        if (p > 0) {
            const int k = (p - 1) & 3;
            const double ex = (k == 0) ? 1.0 : (k == 2) ? -1.0 : 0.0, ey = (k == 1) ? 1.0 : (k == 3) ? -1.0 : 0.0;
            if (p > 4) { const double r = rho * 0.70710678118654752; px += r * (ex - ey); py += r * (ex + ey); }
            else { px += rho * ex; py += rho * ey; }
        }
        unsigned mask = 0;
        // (the limb probes start the simultaneous iteration from the previous probe's roots, one source radius away)
        const unsigned st = centre_images<N>(L, poly[c], px, py, zr, zi, mask, p > 0);
        if (st & (UL_ST_EA_NOCONV | UL_ST_IMG_PARITY)) ok = false;
        const double a = point_mag<N>(L, nullptr, zr, zi, mask, nullptr);
        if (p == 0) { st_c = st; A_c = a; }
        else {
            if (((st ^ st_c) >> 8) & 0xfu) ok = false;   // image count changed
            if (p > 4) s_diag += a; else s_axes += a;
        }
    }
    if (ok) {
        const double Q = 0.5 * fabs(0.125 * (s_axes + s_diag) - A_c);
        const double H = 0.25 * fabs(s_axes - s_diag);
        ok = (Q + H <= tol * A_c);
    }
    if (live) {
        quiet[i] = ok ? 1 : 0;
        // dA/drho of a quiet point from the same probe. Angular mean of A_ps on the limb = A_c + rho^2/4 lap A + O(rho^4), so
        // for the limb-darkened disk (I = 1 - u1 (1 - sqrt(1 - r^2)), <r^2>_I = (1 - 7 u1/15) / (2 (1 - u1/3))):
        //   A_fs = A_c + (mean_8 - A_c)/2 * LD + O(rho^4),  LD = (1 - 7 u1/15)/(1 - u1/3)   =>   dA_fs/drho = (mean_8 - A_c) LD / rho
        // (the quadrupole term of Gould 2008 / Pejcha & Heyrovsky 2009; what "quiet" certifies is that the series converges).
        // Forward mode uses it in place of the rule's own dA/drho, which far from caustics is the small difference of two
        // terms ~ 2A/rho and carries the derivative of the along-line quadrature error.
        const double u1 = cfg[c].u1;
        quiet_drho[i] = ok ? (0.125 * (s_axes + s_diag) - A_c) * ((1.0 - 7.0 * u1 / 15.0) / (1.0 - u1 / 3.0)) / rho : 0.0;
    }
    // work lists of k_limb (one atomicAdd per warp and list): a quiet point is ONE work item, the others WARPS each; listing
    // them apart keeps the working warps of k_limb packed (left in place, a quiet point's other WARPS - 1 work items would
    // return at once and leave their CTA with a single resident warp). The order inside a list is whatever the atomics give:
    // a point's result does not depend on which warp takes it.
    const int lane = threadIdx.x & 31;
    const unsigned bq = __ballot_sync(0xffffffffu, ok), bf = __ballot_sync(0xffffffffu, live && !ok);
    unsigned base_q = 0, base_f = 0;
    if (lane == 0) {
        if (bq) base_q = atomicAdd(&cc->n_quiet, (unsigned)__popc(bq));
        if (bf) base_f = atomicAdd(&cc->n_full, (unsigned)__popc(bf));
    }
    base_q = __shfl_sync(0xffffffffu, base_q, 0); base_f = __shfl_sync(0xffffffffu, base_f, 0);
    const unsigned below = (1u << lane) - 1u;
    if (ok) limb_list[base_q + __popc(bq & below)] = i;
    else if (live) limb_list[n - 1 - (int)(base_f + __popc(bf & below))] = i;
}

// Image-region builder, first half (ulens_limb.cuh): a group of N^2+1 lanes per limb arc, one lane per root; a warp holds
// GPW arcs, and the WARPS warps that share a source point are independent work items (4 per CTA, any mix of points).
// Appends to the point's box list (n_boxes zeroed before the launch).
#ifndef UL_LIMB_MINB
#define UL_LIMB_MINB(N) ((N) == 3 ? 4 : 4)
#endif
template <int N, bool DUAL>
__global__ void __launch_bounds__(128, UL_LIMB_MINB(N))
k_limb(int n, int pt_base, int n_pts_per_cfg, const PointCfg* __restrict__ cfg, const LensPoly* __restrict__ poly,
       const double* __restrict__ w_re, const double* __restrict__ w_im, RegionParams rp,
       SubBox* __restrict__ boxes, BoxExt* __restrict__ exts, int* __restrict__ n_boxes, unsigned* __restrict__ status,
       DevCounters* ctr, const double* __restrict__ c_zr, const double* __restrict__ c_zi,
       const unsigned* __restrict__ c_mask, const int* __restrict__ pmap = nullptr, const unsigned* __restrict__ n_dev = nullptr,
       const unsigned char* __restrict__ quiet = nullptr, const int* __restrict__ limb_list = nullptr,
       const ChunkCounters* __restrict__ cc = nullptr)
{
    typedef LimbGeom<N> G;
    __shared__ LimbShared<N> sh[4];
    const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (n_dev) n = min(n, (int)*n_dev - pt_base);
    const long long item = (long long)blockIdx.x * 4 + wib;          // (point, warp of the point)
    int i, w;
    bool q = false;
    if (limb_list) {
        // work lists of k_quiet: the quiet points first (one work item each: warp 0 follows the whole limb, GPW arcs, an
        // eighth of the samples), then WARPS items for each of the others; the grid is sized for the worst case and the
        // items past the end leave at once, whole CTAs at a time
        const long long nq = cc->n_quiet, nf = cc->n_full;
        if (item < nq) { i = limb_list[item]; w = 0; q = true; }
        else {
            const long long it = item - nq;
            if (it >= nf * G::WARPS) return;
            i = limb_list[n - 1 - (int)(it / G::WARPS)]; w = (int)(it % G::WARPS);
        }
    } else {
        i = (int)(item / G::WARPS); w = (int)(item % G::WARPS);
        if (i >= n) return;                              // whole warp leaves together
    }
    const long long gp = pmap ? (long long)pmap[pt_base + i] : (long long)pt_base + i;
    const int c = (int)(gp / n_pts_per_cfg);
    const Lens L = cfg[c].lens;
    constexpr int CAP = BoxCap<N>::value;
    int n_solves = 0;
    const int n_arcs = q ? G::GPW : G::NARC;
    const int per_arc = q ? max(2, (rp.n_limb / UL_QUIET_LIMB_DIV + G::GPW - 1) / G::GPW) : 0;
    unsigned st = limb_track<N, DUAL>(sh[wib], w, L, poly[c], w_re[gp], w_im[gp], cfg[c].rho, rp, c_zr + (long long)i * 10,
                                      c_zi + (long long)i * 10, c_mask[i], boxes + (size_t)i * CAP,
                                      DUAL ? exts + (size_t)i * CAP : nullptr, n_boxes + i, CAP, n_solves, n_arcs, per_arc);
    st = __reduce_or_sync(0xffffffffu, st);
    n_solves = __reduce_add_sync(0xffffffffu, n_solves);
    if (lane == 0) {
        if (st) atomicOr(&status[i], st);                // k_roots wrote the word first
        atomicAdd(&ctr->n_limb_solves, (unsigned long long)n_solves);
    }
}

// Image-region builder, second half (ulens_regions.cuh sectors_from_boxes): one thread per source point turns the
// box list into sectors, sizes their ray grids and claims their 32-line work units in the chunk's queue.
template <int N>
__global__ void __launch_bounds__(128)
k_sectors(int n, int pt_base, int n_pts_per_cfg, const PointCfg* __restrict__ cfg, const double* __restrict__ w_re,
          const double* __restrict__ w_im, RegionParams rp, const SubBox* __restrict__ boxes, const BoxExt* __restrict__ exts,
          const int* __restrict__ n_boxes, Patch* __restrict__ patches, int* __restrict__ n_patch, unsigned* __restrict__ status,
          unsigned* __restrict__ unit_desc, unsigned cap_units, ChunkCounters* cc, DevCounters* ctr,
          const TangentTable* __restrict__ tans, PatchTan* __restrict__ ptans, const int* __restrict__ pmap = nullptr,
          const unsigned* __restrict__ n_dev = nullptr, const unsigned char* __restrict__ quiet = nullptr,
          const double* __restrict__ c_zr = nullptr, const double* __restrict__ c_zi = nullptr,
          const unsigned* __restrict__ c_mask = nullptr)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    if (n_dev) n = min(n, (int)*n_dev - pt_base);
    const bool live = i < n;                             // (no early return: the warp claims its units together)
    constexpr int CAP = BoxCap<N>::value;
    Patch* pp = patches + (long long)i * UL_MAXP;
    unsigned st = 0;
    int np = 0, total_units = 0;
    if (live) {
        const long long gp = pmap ? (long long)pmap[pt_base + i] : (long long)pt_base + i;
        const int c = (int)(gp / n_pts_per_cfg);
        const Lens L = cfg[c].lens;
        PatchTan* pt = tans ? ptans + (long long)i * UL_MAXP : nullptr;
        // spacing of the limb samples k_limb took for this point (quiet points: GPW arcs of max(2, ...) points)
        typedef LimbGeom<N> G;
        const bool q = quiet && quiet[i];
        const int n_samp = q ? G::GPW * max(2, (rp.n_limb / UL_QUIET_LIMB_DIV + G::GPW - 1) / G::GPW) : G::NARC * max(1, (rp.n_limb + G::NARC / 2) / G::NARC);
        // quiet points: a sector that ends at the true extremes of a smooth near-elliptical image (quiet_image_extremes) is
        // shot with fewer lines and fewer nodes per line: with exact ends the sin-spaced rule across the lines is all but exact
        RegionParams rpq = rp;
        rpq.n_r = max(16, (int)(rp.n_r * UL_QUIET_RES_LINES + 0.5)); rpq.n_theta = max(8, (int)(rp.n_theta * UL_QUIET_RES_NODES + 0.5));
        np = sectors_from_boxes<N>(boxes + (size_t)i * CAP, tans ? exts + (size_t)i * CAP : nullptr, min(n_boxes[i], CAP), rp, i, L,
                                   w_re[gp], w_im[gp], cfg[c].rho, st, tans ? &tans[c] : nullptr, pp, pt, 2.0 * UL_PI / n_samp,
                                   q ? &rpq : nullptr, c_zr + (long long)i * 10, c_zi + (long long)i * 10, c_mask[i]);
        for (int p = 0; p < np; ++p) total_units += pp[p].n_units;
    }
    // one atomicAdd per warp: exclusive prefix sum of the lanes' unit counts, lane 31 holds the warp's total
    unsigned incl = (unsigned)total_units;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const unsigned t = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += t; }
    unsigned wbase = 0;
    if (lane == 31 && incl) wbase = atomicAdd(&cc->n_units, incl);
    wbase = __shfl_sync(0xffffffffu, wbase, 31);
    unsigned base = wbase + incl - (unsigned)total_units;
    if (!live) return;
    // The queue holds chunk x max_units_pt units, so this cannot fail with the built-in per-point cap. If it does
    // (hand-made options), the point is refused and the part of the queue it claimed is filled with void descriptors,
    // which k_shoot skips: the queue never holds an unwritten descriptor.
    if ((unsigned long long)base + (unsigned)total_units > cap_units) {
        for (unsigned u = base; u < cap_units && u < base + (unsigned)total_units; ++u) unit_desc[u] = 0xffffffffu;
        st |= UL_ST_UNIT_OVF; np = 0; total_units = 0;
    }
    unsigned u = base;
    for (int p = 0; p < np; ++p) {
        const int nu = pp[p].n_units;
        pp[p].unit0 = (int)u;
        for (int b = 0; b < nu; ++b) unit_desc[u + b] = ((unsigned)(i * UL_MAXP + p) << 11) | (unsigned)b;
        u += nu;
    }
    n_patch[i] = np;
    if (st) status[i] |= st;
    if (np) atomicAdd(&ctr->n_patches, (unsigned long long)np);
}

// One warp per 32-ring work unit, one lane per ring (Sec. 3.3; App. A). Units are pulled from a device counter.
#ifndef UL_SHOOT_MINB
#define UL_SHOOT_MINB 5
#endif
template <int N, bool LD>
__global__ void __launch_bounds__(128, UL_SHOOT_MINB)
k_shoot(int pt_base, int n_pts_per_cfg, const PointCfg* __restrict__ cfg, const double* __restrict__ w_re,
        const double* __restrict__ w_im, const Patch* __restrict__ patches, const unsigned* __restrict__ unit_desc,
        double* __restrict__ unit_sum, double* __restrict__ unit_odd, unsigned* __restrict__ status,
        ChunkCounters* cc, DevCounters* ctr, unsigned cap_units, const int* __restrict__ pmap = nullptr)
{
    const int lane = threadIdx.x & 31;
    const unsigned n_units = min(cc->n_units, cap_units);       // an overflowing point allocated nothing (UL_ST_UNIT_OVF)
    unsigned long long rays = 0;
    for (;;) {
        unsigned u = 0;
        if (lane == 0) u = atomicAdd(&cc->next_unit, 1u);
        u = __shfl_sync(0xffffffffu, u, 0);
        if (u >= n_units) break;
        unsigned d = unit_desc[u];
        if (d == 0xffffffffu) continue;                  // void descriptor (refused point, k_sectors)
        const Patch P = patches[d >> 11];
        int blk = (int)(d & 0x7ffu);
        long long gp = pmap ? (long long)pmap[pt_base + P.point] : (long long)pt_base + P.point;
        int c = (int)(gp / n_pts_per_cfg);
        Lens L = cfg[c].lens;
        double rho = cfg[c].rho, u1 = cfg[c].u1;
        double wcx = w_re[gp], wcy = w_im[gp];
        int line = blk * 32 + lane;
        double U, S, f; bool edge, clipped;
        // line flux: (1-u1) Int chi dA + (u1/rho) Int chi sqrt(-F) dA      (Eq. A6 split, G12)
        if (P.flags & UL_PATCH_SCAN_R) {
            double th, wt; line_node(P.flags, P.n_th, line, P.th0, P.dth, th, wt);
            shoot_col<N, LD>(L, wcx, wcy, rho * rho, th, P.r0, P.dr, P.n_r, U, S, edge);
            f = ((1.0 - u1) * U + (LD ? (u1 / rho) * S : 0.0)) * wt;
            clipped = edge || (!(P.flags & UL_PATCH_PERIODIC) && (line < 1 || line >= P.n_th - 1) && U > 0.0);
        } else {
            double r, wr; line_node(P.flags, P.n_r, line, P.r0, P.dr, r, wr);
            bool periodic = (P.flags & UL_PATCH_PERIODIC) != 0;
            shoot_ring<N, LD>(L, wcx, wcy, rho * rho, r, P.th0, P.dth, P.n_th, periodic, U, S, edge);
            f = r * ((1.0 - u1) * U + (LD ? (u1 / rho) * S : 0.0)) * P.dth * wr;
            clipped = edge || ((line < 1 || line >= P.n_r - 1) && U > 0.0 && P.r0 > 0.0);
        }
        double tot = warp_sum(f);
        double odd = warp_sum((lane & 1) ? f : 0.0);
        unsigned any_clip = __ballot_sync(0xffffffffu, clipped);
        if (lane == 0) {
            unit_sum[u] = tot;
            unit_odd[u] = 2.0 * odd;
            if (any_clip) atomicOr(&status[P.point], UL_ST_CLIPPED);
            rays += 32ull * (unsigned long long)(((P.flags & UL_PATCH_SCAN_R) ? P.n_r : P.n_th) + 4);
        }
    }
    if (lane == 0 && rays) atomicAdd(&ctr->n_rays, rays);
}

// k_shoot on the FP32 pipe (ulens_f32.cuh; ULENS_OPT_F32_SHOOT): same queue, same lines, same rule; rays in
// segment-local single precision, segment constants / edge events / accumulation in FP64.
template <int N, bool LD>
__global__ void __launch_bounds__(128, UL_SHOOT_MINB)
k_shoot_f32(int pt_base, int n_pts_per_cfg, const PointCfg* __restrict__ cfg, const double* __restrict__ w_re,
            const double* __restrict__ w_im, const Patch* __restrict__ patches, const unsigned* __restrict__ unit_desc,
            double* __restrict__ unit_sum, double* __restrict__ unit_odd, unsigned* __restrict__ status,
            ChunkCounters* cc, DevCounters* ctr, unsigned cap_units, const int* __restrict__ pmap = nullptr)
{
    const int lane = threadIdx.x & 31;
    const unsigned n_units = min(cc->n_units, cap_units);
    unsigned long long rays = 0;
    for (;;) {
        unsigned u = 0;
        if (lane == 0) u = atomicAdd(&cc->next_unit, 1u);
        u = __shfl_sync(0xffffffffu, u, 0);
        if (u >= n_units) break;
        unsigned d = unit_desc[u];
        if (d == 0xffffffffu) continue;
        const Patch P = patches[d >> 11];
        int blk = (int)(d & 0x7ffu);
        long long gp = pmap ? (long long)pmap[pt_base + P.point] : (long long)pt_base + P.point;
        int c = (int)(gp / n_pts_per_cfg);
        Lens L = cfg[c].lens;
        double rho = cfg[c].rho, u1 = cfg[c].u1;
        double wcx = w_re[gp], wcy = w_im[gp];
        int line = blk * 32 + lane;
        double U, S, f; bool edge, clipped;
        if (P.flags & UL_PATCH_SCAN_R) {
            double th, wt; line_node(P.flags, P.n_th, line, P.th0, P.dth, th, wt);
            shoot_col_f32<N, LD>(L, wcx, wcy, rho * rho, th, P.r0, P.dr, P.n_r, U, S, edge);
            f = ((1.0 - u1) * U + (LD ? (u1 / rho) * S : 0.0)) * wt;
            clipped = edge || (!(P.flags & UL_PATCH_PERIODIC) && (line < 1 || line >= P.n_th - 1) && U > 0.0);
        } else {
            double r, wr; line_node(P.flags, P.n_r, line, P.r0, P.dr, r, wr);
            bool periodic = (P.flags & UL_PATCH_PERIODIC) != 0;
            shoot_ring_f32<N, LD>(L, wcx, wcy, rho * rho, r, P.th0, P.dth, P.n_th, periodic, U, S, edge);
            f = r * ((1.0 - u1) * U + (LD ? (u1 / rho) * S : 0.0)) * P.dth * wr;
            clipped = edge || ((line < 1 || line >= P.n_r - 1) && U > 0.0 && P.r0 > 0.0);
        }
        double tot = warp_sum(f);
        double odd = warp_sum((lane & 1) ? f : 0.0);
        unsigned any_clip = __ballot_sync(0xffffffffu, clipped);
        if (lane == 0) {
            unit_sum[u] = tot;
            unit_odd[u] = 2.0 * odd;
            if (any_clip) atomicOr(&status[P.point], UL_ST_CLIPPED);
            rays += 32ull * (unsigned long long)(((P.flags & UL_PATCH_SCAN_R) ? P.n_r : P.n_th) + 4);
        }
    }
    if (lane == 0 && rays) atomicAdd(&ctr->n_rays, rays);
}

// One thread per point: ordered (deterministic) sum over its sectors' units, normalisation (Eq. A5; F0 of P:99).
__global__ void k_finalize(int n, int pt_base, int n_pts_per_cfg, const PointCfg* __restrict__ cfg,
                           const Patch* __restrict__ patches, const int* __restrict__ n_patch,
                           const double* __restrict__ unit_sum, const double* __restrict__ unit_odd,
                           const unsigned* __restrict__ status_ws, double rel_tol,
                           double* __restrict__ A_out, double* __restrict__ err_out, unsigned* __restrict__ status_out,
                           DevCounters* ctr, const int* __restrict__ pmap = nullptr,
                           const unsigned* __restrict__ n_dev = nullptr, unsigned st_or = 0)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (n_dev) n = min(n, (int)*n_dev - pt_base);
    if (i >= n) return;
    long long gp = pmap ? (long long)pmap[pt_base + i] : (long long)pt_base + i;
    int c = (int)(gp / n_pts_per_cfg);
    double rho = cfg[c].rho, u1 = cfg[c].u1;
    double F0 = UL_PI * rho * rho * (1.0 - u1 / 3.0);
    int np = n_patch[i];
    double s = 0.0, so = 0.0;
    unsigned long long nu_tot = 0;
    for (int p = 0; p < np; ++p) {
        const Patch& P = patches[(long long)i * UL_MAXP + p];
        int nu = P.n_units;
        nu_tot += nu;
        for (int b = 0; b < nu; ++b) { s += unit_sum[P.unit0 + b]; so += unit_odd[P.unit0 + b]; }
    }
    unsigned st = status_ws[i] | st_or;
    double A = s / F0, Ao = so / F0;
    if (np == 0) { A = nan(""); Ao = A; }
    // half-resolution self check: the radial rule errs like dr^1.5 (square-root ring ends), so the error
    // of the full sum is about |A - A_half| / (2^1.5 - 1)
    double err = fabs(A - Ao) / (1.8284271247461903 * fabs(A));
    if (!(err <= rel_tol)) st |= UL_ST_ERR_HIGH;
    atomicAdd(&ctr->n_units, nu_tot);
    if (st_or) {
        // retry pass: the new result replaces the first one only if it is finite and no worse (fewer doubtful
        // bits, or as many and a smaller self-error); a point that keeps its first result keeps its first status
        const unsigned st0 = status_out[gp];
        const int b0 = __popc(st0 & UL_ST_RETRY_MASK), b1 = __popc(st & UL_ST_RETRY_MASK);
        const double err0 = err_out ? err_out[gp] : 1e300;
        const bool better = (A == A) && (b1 < b0 || (b1 == b0 && !(err > err0)));
        if (!better) return;
    }
    A_out[gp] = A;
    if (err_out) err_out[gp] = err;
    if (status_out) status_out[gp] = st;
    if (st_or) {                                         // the point was counted (and counted as flagged) before
        if (!(st & 0xffu)) atomicAdd(&ctr->n_flagged, ~0ull);
    } else {
        if (i == 0) atomicAdd(&ctr->n_points, (unsigned long long)n);
        if (st & 0xffu) atomicAdd(&ctr->n_flagged, 1ull);
    }
}

// ------------------------------------------------------------------------------------------------ forward-mode variant (a8)

// k_shoot with tangents: same unit queue, same lines. The scan accumulates, per line, the line sums U, S and two
// tangent-statistic sets (ulens_dual.cuh); the NT directions (5 binary: w_cx, w_cy, s, q, rho; 8 triple: w_cx, w_cy,
// s, q, q3, r3, psi, rho) only enter per LINE, when the sets are contracted with the configuration's tangent table.
// The sector's grid moves with the image ACROSS the lines: x0' = lo' - kap_lo (hi' - lo'), dx' = (hi' - lo')(1 + kap_lo + kap_hi) / n.
#ifndef UL_SHOOT_DUAL_MINB
#define UL_SHOOT_DUAL_MINB 4
#endif
template <int N, bool LD>
__global__ void __launch_bounds__(128, UL_SHOOT_DUAL_MINB)
k_shoot_dual(int pt_base, int n_pts_per_cfg, const PointCfg* __restrict__ cfg, const TangentTable* __restrict__ tans,
             const double* __restrict__ w_re, const double* __restrict__ w_im, const Patch* __restrict__ patches,
             const PatchTan* __restrict__ ptans, const unsigned* __restrict__ unit_desc, double* __restrict__ unit_sum,
             double* __restrict__ unit_odd, double* __restrict__ unit_tan, unsigned* __restrict__ status,
             ChunkCounters* cc, DevCounters* ctr, unsigned cap_units, const int* __restrict__ pmap = nullptr)
{
    constexpr int NT = TanDirs<N>::NT;
    typedef Dual<NT> DN;
    const int lane = threadIdx.x & 31;
    const unsigned n_units = min(cc->n_units, cap_units);
    unsigned long long rays = 0;
    for (;;) {
        unsigned u = 0;
        if (lane == 0) u = atomicAdd(&cc->next_unit, 1u);
        u = __shfl_sync(0xffffffffu, u, 0);
        if (u >= n_units) break;
        unsigned d = unit_desc[u];
        if (d == 0xffffffffu) continue;                  // void descriptor (refused point, k_sectors)
        const Patch P = patches[d >> 11];
        const PatchTan& PT = ptans[d >> 11];
        int blk = (int)(d & 0x7ffu);
        long long gp = pmap ? (long long)pmap[pt_base + P.point] : (long long)pt_base + P.point;
        int c = (int)(gp / n_pts_per_cfg);
        Lens L = cfg[c].lens;
        const TangentTable& T = tans[c];
        double rho = cfg[c].rho, u1 = cfg[c].u1;
        double wcx = w_re[gp], wcy = w_im[gp];
        int line = blk * 32 + lane;
        // co-moving grid ACROSS the scan lines: the span's two ends follow the image's extreme
        // limb points; ALONG the lines the nodes are frozen (the margins there are generous)
        const bool scan_r = (P.flags & UL_PATCH_SCAN_R) != 0, periodic = (P.flags & UL_PATCH_PERIODIC) != 0;
        DN x0 = dual_const<NT>(scan_r ? P.th0 : P.r0), dx = dual_const<NT>(scan_r ? P.dth : P.dr);
        const int n_lines = scan_r ? P.n_th : P.n_r;
        if (!(scan_r && periodic)) {
#pragma unroll
            for (int k = 0; k < NT; ++k) {
                double lo = scan_r ? PT.tlo_dot[k] : PT.rlo_dot[k], hi = scan_r ? PT.thi_dot[k] : PT.rhi_dot[k];
                x0.d[k] = lo - P.kap_lo * (hi - lo); dx.d[k] = (hi - lo) * (1.0 + P.kap_lo + P.kap_hi) / n_lines;
            }
        }
        DN xl, wl;
        line_node_d<NT>(P.flags, n_lines, line, x0, dx, xl, wl);
        DN U, S, f; bool edge, clipped;
        {
            TanStat<N> SU, SS;
            if (scan_r) {
                shoot_col_t<N, LD>(L, wcx, wcy, rho * rho, cos(xl.v), sin(xl.v), P.r0, P.dr, P.n_r, U.v, S.v, SU, SS, edge);
                stat_contract<N, NT>(L, T, rho, SU, xl.d, 1.0, U.d);
                if (LD) stat_contract<N, NT>(L, T, rho, SS, xl.d, P.dr, S.d);
            } else {
                shoot_ring_t<N, LD>(L, wcx, wcy, rho * rho, xl.v, P.th0, P.dth, P.n_th, periodic, U.v, S.v, SU, SS, edge);
                stat_contract<N, NT>(L, T, rho, SU, xl.d, 1.0, U.d);
                if (LD) stat_contract<N, NT>(L, T, rho, SS, xl.d, 1.0, S.d);
            }
            if (!LD) { S.v = 0.0; for (int k = 0; k < NT; ++k) S.d[k] = 0.0; }
        }
        DN rho_d = dual_const<NT>(rho);
#pragma unroll
        for (int k = 0; k < NT; ++k) rho_d.d[k] = T.drho[k];
        if (P.flags & UL_PATCH_SINR) {
            // Tip caps. The sin-spaced lines crowd towards the two tips of the image, where a line
            // cuts a chord shorter than a few node spacings: harmless for the value (those lines weigh ~phi^2),
            // but the edge terms of a chord the nodes do not resolve are (small)/(small) and can be arbitrarily
            // wrong. Near a tip the boundary is a parabola in co-moving coordinates, so the line integrals of the
            // cap lines all scale with the parameters by ONE common factor (U ~ sqrt(h/kappa), S ~ h b/sqrt(a),
            // times a function of the line index only): a line whose chord spans < 3 node spacings takes its
            // relative tangents from the nearest resolved line on the side away from the tip (same warp);
            // if there is none in this unit its tangents are dropped (bounded: such lines carry < 1e-3 of the flux).
            const double cells = scan_r ? U.v / ((P.r0 + 0.5 * P.n_r * P.dr) * P.dr) : U.v;
            const unsigned m_ne = __ballot_sync(0xffffffffu, cells > 0.0);
            const unsigned m_res = __ballot_sync(0xffffffffu, cells >= 3.0);
            const unsigned below = (1u << lane) - 1u, above = ~((2u << lane) - 1u);   // (2u << 31) == 0: no lanes above
            int src = lane;
            const bool unresolved = cells > 0.0 && cells < 3.0;
            if (unresolved) {
                const unsigned res_dn = m_res & below, emp_dn = ~m_ne & below;
                const unsigned res_up = m_res & above, emp_up = ~m_ne & above;
                const int s_dn = res_dn ? 31 - __clz(res_dn) : -1, e_dn = emp_dn ? 31 - __clz(emp_dn) : -1;
                const int s_up = res_up ? __ffs(res_up) - 1 : 32, e_up = emp_up ? __ffs(emp_up) - 1 : 32;
                // unit edges: line -1 and line n_lines count as empty (the sector ends there)
                const bool tip_below = (e_dn > s_dn) || (s_dn < 0 && blk == 0);
                const bool tip_above = (e_up < s_up) || (s_up > 31 && blk == P.n_units - 1);
                if (tip_below && !tip_above && s_up <= 31) src = s_up;
                else if (tip_above && !tip_below && s_dn >= 0) src = s_dn;
                else src = -1;
            }
            const int from = src < 0 ? lane : src;
            const double Ucv = __shfl_sync(0xffffffffu, U.v, from), Scv = __shfl_sync(0xffffffffu, S.v, from);
            const double ku = (unresolved && src >= 0 && Ucv > 0.0) ? U.v / Ucv : 0.0;
            const double ks = (unresolved && src >= 0 && Scv > 0.0) ? S.v / Scv : 0.0;
#pragma unroll
            for (int k = 0; k < NT; ++k) {
                const double ud = __shfl_sync(0xffffffffu, U.d[k], from), sd = __shfl_sync(0xffffffffu, S.d[k], from);
                if (unresolved) { U.d[k] = ku * ud; S.d[k] = ks * sd; }
            }
        }
        f = U * (1.0 - u1);
        if (LD) f = f + (S / rho_d) * u1;
        if (scan_r) {
            f = f * wl;
            clipped = edge || (!periodic && (line < 1 || line >= P.n_th - 1) && U.v > 0.0);
        } else {
            f = xl * f * wl * P.dth;
            clipped = edge || ((line < 1 || line >= P.n_r - 1) && U.v > 0.0 && P.r0 > 0.0);
        }
        double tot = warp_sum(f.v);
        double odd = warp_sum((lane & 1) ? f.v : 0.0);
        double tk[NT];
#pragma unroll
        for (int k = 0; k < NT; ++k) tk[k] = warp_sum(f.d[k]);
        unsigned any_clip = __ballot_sync(0xffffffffu, clipped);
        if (lane == 0) {
            unit_sum[u] = tot;
            unit_odd[u] = 2.0 * odd;
#pragma unroll
            for (int k = 0; k < NT; ++k) unit_tan[(size_t)u * NT + k] = tk[k];
            if (any_clip) atomicOr(&status[P.point], UL_ST_CLIPPED);
            rays += 32ull * (unsigned long long)(((P.flags & UL_PATCH_SCAN_R) ? P.n_r : P.n_th) + 4);
        }
    }
    if (lane == 0 && rays) atomicAdd(&ctr->n_rays, rays);
}

// per point: ordered sum of the units' tangents, normalisation A = flux / F0(rho) differentiated:
//   dA/dp_k = (dflux_k - A dF0_k) / F0,  F0 = pi rho^2 (1 - u1/3)
template <int NT>
__global__ void k_finalize_dual(int n, int pt_base, int n_pts_per_cfg, const PointCfg* __restrict__ cfg,
                                const TangentTable* __restrict__ tans, const Patch* __restrict__ patches,
                                const int* __restrict__ n_patch, const double* __restrict__ unit_sum,
                                const double* __restrict__ unit_tan, double* __restrict__ grad, const int* __restrict__ pmap = nullptr,
                                const unsigned* __restrict__ n_dev = nullptr, const unsigned* __restrict__ status_retry = nullptr,
                                const unsigned char* __restrict__ quiet = nullptr, const double* __restrict__ quiet_drho = nullptr)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (n_dev) n = min(n, (int)*n_dev - pt_base);
    if (i >= n) return;
    long long gp = pmap ? (long long)pmap[pt_base + i] : (long long)pt_base + i;
    if (status_retry && !(status_retry[gp] & UL_ST_RETRIED)) return;     // retry pass: k_finalize kept the first result
    int c = (int)(gp / n_pts_per_cfg);
    double rho = cfg[c].rho, u1 = cfg[c].u1;
    double F0 = UL_PI * rho * rho * (1.0 - u1 / 3.0);
    int np = n_patch[i];
    double s = 0.0, tk[NT];
    for (int k = 0; k < NT; ++k) tk[k] = 0.0;
    for (int p = 0; p < np; ++p) {
        const Patch& P = patches[(long long)i * UL_MAXP + p];
        for (int b = 0; b < P.n_units; ++b) {
            s += unit_sum[P.unit0 + b];
            for (int k = 0; k < NT; ++k) tk[k] += unit_tan[(size_t)(P.unit0 + b) * NT + k];
        }
    }
    double A = s / F0;
    for (int k = 0; k < NT; ++k) {
        double dF0 = 2.0 * UL_PI * rho * (1.0 - u1 / 3.0) * tans[c].drho[k];
        grad[gp * NT + k] = np ? (tk[k] - A * dF0) / F0 : nan("");
    }
    // quiet point: dA/drho from the multipole probe (k_quiet); direction NT-1 is rho in every tangent table
    if (quiet && quiet[i] && np) grad[gp * NT + NT - 1] = quiet_drho[i];
}

// chain rule through the trajectory (reading G3): (w_cx, w_cy, s, q, rho) -> (t0, u0, tE, s, q, rho, alpha)
__global__ void k_chain7(int n_cfg, int n_ep, const double* __restrict__ theta, const double* __restrict__ t,
                         const double* __restrict__ w_re, const double* __restrict__ w_im,
                         const double* __restrict__ grad5, double* __restrict__ dA)
{
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)n_cfg * n_ep) return;
    int c = (int)(i / n_ep), e = (int)(i % n_ep);
    const double* th = theta + 7 * c;
    double tE = th[2], tau = (t[e] - th[0]) / tE;
    double ca = cos(th[6]), sa = sin(th[6]);
    const double* g = grad5 + i * UL_NT;
    double along = g[0] * ca + g[1] * sa;
    double* o = dA + i * 7;
    o[0] = -along / tE;
    o[1] = -g[0] * sa + g[1] * ca;
    o[2] = -tau * along / tE;
    o[3] = g[2];
    o[4] = g[3];
    o[5] = g[4];
    o[6] = -g[0] * w_im[i] + g[1] * w_re[i];
}


// the same for the triple lens: (w_cx, w_cy, s, q, q3, r3, psi, rho) -> (t0, u0, tE, s, q, rho, alpha, q3, r3, psi)
__global__ void k_chain10(int n_cfg, int n_ep, const double* __restrict__ theta, const double* __restrict__ t,
                          const double* __restrict__ w_re, const double* __restrict__ w_im,
                          const double* __restrict__ grad8, double* __restrict__ dA)
{
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)n_cfg * n_ep) return;
    int c = (int)(i / n_ep), e = (int)(i % n_ep);
    const double* th = theta + 10 * c;
    double tE = th[2], tau = (t[e] - th[0]) / tE;
    double ca = cos(th[6]), sa = sin(th[6]);
    const double* g = grad8 + i * 8;
    double along = g[0] * ca + g[1] * sa;
    double* o = dA + i * 10;
    o[0] = -along / tE;
    o[1] = -g[0] * sa + g[1] * ca;
    o[2] = -tau * along / tE;
    o[3] = g[2];
    o[4] = g[3];
    o[5] = g[7];
    o[6] = -g[0] * w_im[i] + g[1] * w_re[i];
    o[7] = g[4];
    o[8] = g[5];
    o[9] = g[6];
}

// trajectory for the 10-parameter triple-lens vector (t0, u0, tE, s, q, rho, alpha, q3, r3, psi)
__global__ void k_traj10(int n_cfg, int n_ep, const double* __restrict__ theta, const double* __restrict__ t,
                         double* __restrict__ w_re, double* __restrict__ w_im)
{
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)n_cfg * n_ep) return;
    int c = (int)(i / n_ep), e = (int)(i % n_ep);
    const double* th = theta + 10 * c;
    double tau = (t[e] - th[0]) / th[2];
    double ca = cos(th[6]), sa = sin(th[6]);
    w_re[i] = tau * ca - th[1] * sa;
    w_im[i] = tau * sa + th[1] * ca;
}


// ------------------------------------------------------------------------------------------------
// Marginalised-flux negative log-likelihood and its gradient (App. B.2, Eqs. B17-B23).
// One CTA per light curve. With m_i = A_i - 1, M_i = (m_i, 1), r = F - M mu, C = diag(sigma_i^2), Lambda = diag(l1, l2):
//   S = Lambda^-1 + M^T C^-1 M (2x2),  v = M^T C^-1 r,
//   NLL = 1/2 [ sum r_i^2/sigma_i^2 - v^T S^-1 v ] + 1/2 [ sum ln sigma_i^2 + ln l1 + ln l2 + ln det S ]      (B17-B19)
// and, with alpha = B^-1 r, bm = B^-1 m (B = C + M Lambda M^T, both through B18),
//   dNLL/dA_i = -(mu_1 + l1 m.alpha) alpha_i + l1 bm_i,     grad_k = sum_i dNLL/dA_i dA_i/dtheta_k.
// ------------------------------------------------------------------------------------------------
template <int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double* sh)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
#pragma unroll
    for (int k = 0; k < NV; ++k) v[k] = warp_sum(v[k]);
    __syncthreads();
    if (lane == 0) for (int k = 0; k < NV; ++k) sh[w * NV + k] = v[k];
    __syncthreads();
    // every thread adds the warp partials in the same order: deterministic, and all threads hold the totals
#pragma unroll
    for (int k = 0; k < NV; ++k) { double t = 0.0; for (int j = 0; j < nw; ++j) t += sh[j * NV + k]; v[k] = t; }
}

__global__ void __launch_bounds__(256)
k_nll(int n_ep, const double* __restrict__ A, const double* __restrict__ dA, const double* __restrict__ flux,
      const double* __restrict__ sigma, double mu1, double mu2, double l1, double l2,
      double* __restrict__ nll_out, double* __restrict__ grad_out)
{
    __shared__ double sh[8 * 15];
    const int c = blockIdx.x;
    const double* Ac = A + (size_t)c * n_ep;
    double a[7] = {0, 0, 0, 0, 0, 0, 0};       // S11', S12, S22', v1, v2, sum r^2/s^2, sum ln s^2
    for (int i = threadIdx.x; i < n_ep; i += blockDim.x) {
        const double m = Ac[i] - 1.0, s2 = sigma[i] * sigma[i], iw = 1.0 / s2;
        const double r = flux[i] - m * mu1 - mu2;
        a[0] += m * m * iw; a[1] += m * iw; a[2] += iw; a[3] += m * r * iw; a[4] += r * iw; a[5] += r * r * iw; a[6] += log(s2);
    }
    block_sum<7>(a, sh);
    const double S11 = 1.0 / l1 + a[0], S12 = a[1], S22 = 1.0 / l2 + a[2];
    const double det = S11 * S22 - S12 * S12;
    // S^-1 v and S^-1 u,  u = M^T C^-1 m = (a0, a1)
    const double x1 = (S22 * a[3] - S12 * a[4]) / det, x2 = (S11 * a[4] - S12 * a[3]) / det;
    const double y1 = (S22 * a[0] - S12 * a[1]) / det, y2 = (S11 * a[1] - S12 * a[0]) / det;
    if (threadIdx.x == 0)
        nll_out[c] = 0.5 * (a[5] - (a[3] * x1 + a[4] * x2)) + 0.5 * (a[6] + log(l1) + log(l2) + log(det));
    if (!grad_out) return;
    const double* dAc = dA + (size_t)c * n_ep * 7;
    double g[15];                                // m.alpha, P_k = sum alpha_i dA_ik, Q_k = sum bm_i dA_ik
#pragma unroll
    for (int k = 0; k < 15; ++k) g[k] = 0.0;
    for (int i = threadIdx.x; i < n_ep; i += blockDim.x) {
        const double m = Ac[i] - 1.0, iw = 1.0 / (sigma[i] * sigma[i]);
        const double r = flux[i] - m * mu1 - mu2;
        const double al = (r - (m * x1 + x2)) * iw, bm = (m - (m * y1 + y2)) * iw;
        g[0] += m * al;
#pragma unroll
        for (int k = 0; k < 7; ++k) { const double d = dAc[(size_t)i * 7 + k]; g[1 + k] += al * d; g[8 + k] += bm * d; }
    }
    block_sum<15>(g, sh);
    if (threadIdx.x < 7) {
        const int k = threadIdx.x;
        grad_out[(size_t)c * 7 + k] = -(mu1 + l1 * g[0]) * g[1 + k] + l1 * g[8 + k];
    }
}

// FP64 FMA peak: 8 independent chains per thread
__global__ void k_dfma_peak(int iters, double* out)
{
    double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const double m = 1.0000001, b = 1e-9;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            a0 = fma(a0, m, b); a1 = fma(a1, m, b); a2 = fma(a2, m, b); a3 = fma(a3, m, b);
            a4 = fma(a4, m, b); a5 = fma(a5, m, b); a6 = fma(a6, m, b); a7 = fma(a7, m, b);
        }
    }
    double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (s == 12345.678) out[0] = s;
}

// FP32 FMA peak: 8 independent chains per thread
__global__ void k_ffma_peak(int iters, float* out)
{
    float a0 = threadIdx.x * 1e-9f, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const float m = 1.0000001f, b = 1e-9f;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            a0 = fmaf(a0, m, b); a1 = fmaf(a1, m, b); a2 = fmaf(a2, m, b); a3 = fmaf(a3, m, b);
            a4 = fmaf(a4, m, b); a5 = fmaf(a5, m, b); a6 = fmaf(a6, m, b); a7 = fmaf(a7, m, b);
        }
    }
    float s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (s == 12345.678f) out[0] = s;
}

// ------------------------------------------------------------------------------------------------ C ABI

extern "C" const char* ulens_strerror(int code)
{
    switch (code) {
        case ULENS_OK: return "ok";
        case ULENS_EINVAL: return "invalid argument";
        case ULENS_ECUDA: return "CUDA error";
        case ULENS_ENOMEM: return "out of memory";
        case ULENS_EUNSUPPORTED: return "unsupported";
        case ULENS_ELIMIT: return "size beyond the fixed scratch of the no-allocation entry (ULENS_STATIC_MAX_POINTS)";
        default: return "unknown error";
    }
}

extern "C" const char* ulens_last_cuda_error(ulens_ctx* ctx) { return ctx ? ctx->cuda_err : ""; }

extern "C" int ulens_create(ulens_ctx** out, int cuda_device, const ulens_options* opt)
{
    if (!out) return ULENS_EINVAL;
    *out = nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || cuda_device < 0 || cuda_device >= ndev) return ULENS_ECUDA;
    ulens_ctx* ctx = new (std::nothrow) ulens_ctx();
    if (!ctx) return ULENS_ENOMEM;
    memset(ctx, 0, sizeof *ctx);
    ctx->device = cuda_device;
    ctx->timed = new (std::nothrow) std::vector<ulens_ctx::TimedLaunch>();
    ctx->last_lenses = new (std::nothrow) std::vector<ulens_lens>();
    ctx->last_rho = new (std::nothrow) std::vector<double>();
    ctx->last_u1 = new (std::nothrow) std::vector<double>();
    if (!ctx->timed || !ctx->last_lenses || !ctx->last_rho || !ctx->last_u1) {
        delete ctx->timed; delete ctx->last_lenses; delete ctx->last_rho; delete ctx->last_u1; delete ctx;
        return ULENS_ENOMEM;
    }
    ulens_options o; memset(&o, 0, sizeof o);
    if (opt) o = *opt;
    if (o.n_limb <= 0) o.n_limb = 512;
    o.n_limb = (o.n_limb + 31) & ~31;
    if (o.n_limb > 8192) o.n_limb = 8192;
    if (o.n_r <= 0) o.n_r = 96;
    if (o.n_theta <= 0) o.n_theta = 48;
    if (!(o.rel_tol > 0.0)) o.rel_tol = 1e-4;
    if (o.chunk_pts <= 0) o.chunk_pts = 65536;
    if (o.chunk_pts > (1 << 21) / UL_MAXP) o.chunk_pts = (1 << 21) / UL_MAXP;
    if (o.chunk_pts > 0x7fffff00 / 1024) o.chunk_pts = 0x7fffff00 / 1024;
    ctx->opt = o;
    ctx->rp.n_limb = o.n_limb; ctx->rp.n_r = o.n_r; ctx->rp.n_theta = o.n_theta;
    ctx->rp.max_nr = 8192; ctx->rp.max_nth = 32768; ctx->rp.max_units_pt = 1024;
    ctx->chunk = o.chunk_pts;
    ctx->cap_units = (size_t)ctx->chunk * ctx->rp.max_units_pt;     // a full chunk of points at the per-point cap fits: no overflow
    if (ctx->cap_units > 0x7fffff00u) ctx->cap_units = 0x7fffff00u;
    cudaError_t e = cudaSetDevice(cuda_device);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->patches, sizeof(Patch) * UL_MAXP * (size_t)ctx->chunk);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->n_patch, sizeof(int) * (size_t)ctx->chunk);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->status_ws, sizeof(unsigned) * (size_t)ctx->chunk);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->c_zr, sizeof(double) * 10 * (size_t)ctx->chunk);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->c_zi, sizeof(double) * 10 * (size_t)ctx->chunk);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->c_mask, sizeof(unsigned) * (size_t)ctx->chunk);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->n_boxes, sizeof(int) * (size_t)ctx->chunk);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->quiet, (size_t)ctx->chunk);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->limb_list, sizeof(int) * (size_t)ctx->chunk);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->quiet_drho, sizeof(double) * (size_t)ctx->chunk);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->unit_desc, sizeof(unsigned) * ctx->cap_units);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->unit_sum, sizeof(double) * ctx->cap_units);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->unit_odd, sizeof(double) * ctx->cap_units);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->cc, sizeof(ChunkCounters));
    if (e == cudaSuccess) e = cudaMalloc(&ctx->counters, sizeof(DevCounters));
    if (e == cudaSuccess) e = cudaMemset(ctx->counters, 0, sizeof(DevCounters));
    if (e != cudaSuccess) { ulens_destroy(ctx); return e == cudaErrorMemoryAllocation ? ULENS_ENOMEM : ULENS_ECUDA; }
    *out = ctx;
    return ULENS_OK;
}

extern "C" void ulens_destroy(ulens_ctx* ctx)
{
    if (!ctx) return;
    cudaSetDevice(ctx->device);
    cudaDeviceSynchronize();
    cudaFree(ctx->c_zr); cudaFree(ctx->c_zi); cudaFree(ctx->c_mask);
    cudaFree(ctx->boxes); cudaFree(ctx->exts); cudaFree(ctx->n_boxes); cudaFree(ctx->quiet); cudaFree(ctx->limb_list); cudaFree(ctx->quiet_drho);
    cudaFree(ctx->ptans); cudaFree(ctx->unit_tan); cudaFree(ctx->grad5); cudaFree(ctx->tan_dev);
    cudaFree(ctx->patches); cudaFree(ctx->n_patch); cudaFree(ctx->status_ws); cudaFree(ctx->unit_desc);
    cudaFree(ctx->unit_sum); cudaFree(ctx->unit_odd); cudaFree(ctx->cc); cudaFree(ctx->counters);
    cudaFree(ctx->cfg_dev); cudaFree(ctx->poly_dev); cudaFree(ctx->traj_w); cudaFree(ctx->io_buf);
    cudaFree(ctx->ext_flag); cudaFree(ctx->ext_map); cudaFree(ctx->ext_blk); cudaFree(ctx->st_all);
    if (ctx->timed) {
        for (auto& t : *ctx->timed) { cudaEventDestroy(t.a); cudaEventDestroy(t.b); }
        delete ctx->timed;
    }
    for (int k = 0; k < UL_N_STAGE; ++k) {
        if (ctx->stage[k].host) cudaFreeHost(ctx->stage[k].host);
        if (ctx->stage[k].ev) cudaEventDestroy(ctx->stage[k].ev);
    }
    delete ctx->last_lenses; delete ctx->last_rho; delete ctx->last_u1;
    delete ctx;
}

// copy `bytes` from ordinary host memory to the device through a pinned staging slot, stream-ordered, no sync
static int stage_upload(ulens_ctx* ctx, void* dst_dev, const void* src_host, size_t bytes, cudaStream_t st)
{
    if (bytes == 0) return ULENS_OK;
    ulens_ctx::Stage& S = ctx->stage[ctx->stage_next];
    ctx->stage_next = (ctx->stage_next + 1) % UL_N_STAGE;
    if (S.used) CK(cudaEventSynchronize(S.ev));          // the copy issued UL_N_STAGE uploads ago: long finished
    if (!S.ev) CK(cudaEventCreateWithFlags(&S.ev, cudaEventDisableTiming));
    if (bytes > S.cap) {
        if (S.host) cudaFreeHost(S.host);
        S.host = nullptr; S.cap = 0;
        size_t cap = bytes + bytes / 4 + 4096;
        if (cudaHostAlloc(&S.host, cap, cudaHostAllocDefault) != cudaSuccess) return ULENS_ENOMEM;
        S.cap = cap;
    }
    memcpy(S.host, src_host, bytes);
    CK(cudaMemcpyAsync(dst_dev, S.host, bytes, cudaMemcpyHostToDevice, st));
    CK(cudaEventRecord(S.ev, st));
    S.used = true;
    return ULENS_OK;
}

static int upload_cfgs(ulens_ctx* ctx, int n_cfg, const ulens_lens* lenses, const double* rho, const double* u1,
                       cudaStream_t st, int* n_lens_out, bool* any_ld)
{
    int N = lenses[0].n_lens;
    if (N < 1 || N > 3) return ULENS_EINVAL;
    // same tables as the last call (an HMC chain re-evaluates the same lens array many times): nothing to do
    if (ctx->last_lenses->size() == (size_t)n_cfg && ctx->cfg_dev &&
        memcmp(ctx->last_lenses->data(), lenses, sizeof(ulens_lens) * n_cfg) == 0 &&
        memcmp(ctx->last_rho->data(), rho, sizeof(double) * n_cfg) == 0 &&
        memcmp(ctx->last_u1->data(), u1, sizeof(double) * n_cfg) == 0) {
        *n_lens_out = ctx->last_N; *any_ld = ctx->last_ld;
        return ULENS_OK;
    }
    ctx->last_lenses->clear(); ctx->last_tan_valid = false;
    std::vector<PointCfg> cfg(n_cfg);
    std::vector<LensPoly> poly(n_cfg);
    *any_ld = false;
    for (int c = 0; c < n_cfg; ++c) {
        const ulens_lens& L = lenses[c];
        if (L.n_lens != N) return ULENS_EUNSUPPORTED;       // one lens multiplicity per call
        double tot = 0.0;
        for (int a = 0; a < N; ++a) {
            if (!isfinite(L.eps[a]) || !(L.eps[a] >= 0.0) || !isfinite(L.ax[a]) || !isfinite(L.ay[a])) return ULENS_EINVAL;
            tot += L.eps[a];
        }
        if (fabs(tot - 1.0) > 1e-9) return ULENS_EINVAL;
        if (!finite_pos(rho[c]) || !(u1[c] >= 0.0 && u1[c] <= 1.0)) return ULENS_EINVAL;
        memset(&cfg[c], 0, sizeof(PointCfg));
        cfg[c].lens.n = N;
        for (int a = 0; a < N; ++a) { cfg[c].lens.eps[a] = L.eps[a]; cfg[c].lens.ax[a] = L.ax[a]; cfg[c].lens.ay[a] = L.ay[a]; }
        cfg[c].rho = rho[c]; cfg[c].u1 = u1[c];
        if (u1[c] > 0.0) *any_ld = true;
        lens_poly_basis(L.n_lens, L.eps, L.ax, L.ay, &poly[c]);
    }
    if ((size_t)n_cfg > ctx->cfg_cap) {
        cudaFree(ctx->cfg_dev); cudaFree(ctx->poly_dev); ctx->cfg_dev = nullptr; ctx->poly_dev = nullptr; ctx->cfg_cap = 0;
        size_t cap = (size_t)n_cfg + 64;
        if (cudaMalloc(&ctx->cfg_dev, sizeof(PointCfg) * cap) != cudaSuccess) return ULENS_ENOMEM;
        if (cudaMalloc(&ctx->poly_dev, sizeof(LensPoly) * cap) != cudaSuccess) return ULENS_ENOMEM;
        ctx->cfg_cap = cap;
    }
    int rc = stage_upload(ctx, ctx->cfg_dev, cfg.data(), sizeof(PointCfg) * n_cfg, st);
    if (rc == ULENS_OK) rc = stage_upload(ctx, ctx->poly_dev, poly.data(), sizeof(LensPoly) * n_cfg, st);
    if (rc != ULENS_OK) return rc;
    ctx->last_lenses->assign(lenses, lenses + n_cfg);
    ctx->last_rho->assign(rho, rho + n_cfg); ctx->last_u1->assign(u1, u1 + n_cfg);
    ctx->last_N = N; ctx->last_ld = *any_ld;
    *n_lens_out = N;
    return ULENS_OK;
}

template <int N>
static int run_chunks(ulens_ctx* ctx, long long n_total, int n_pts, bool ld, const double* w_re, const double* w_im,
                      double* A_out, double* err_out, unsigned* status_out, cudaStream_t st, double* grad5_out = nullptr,
                      const int* pmap = nullptr, const unsigned* n_dev = nullptr, const RegionParams* rp_override = nullptr,
                      unsigned st_or = 0)
{
    const RegionParams rp = rp_override ? *rp_override : ctx->rp;
    constexpr int DEG = N * N + 1;
    const bool dual = grad5_out != nullptr;
    const TangentTable* tans = dual ? ctx->tan_dev : nullptr;
    constexpr int NT = TanDirs<N>::NT;
    if (dual && !ctx->ptans) {
        if (cudaMalloc(&ctx->ptans, sizeof(PatchTan) * UL_MAXP * (size_t)ctx->chunk) != cudaSuccess) return ULENS_ENOMEM;
    }
    if (dual && ctx->unit_tan_nt < NT) {                 // [cap_units][NT]: sized for the widest tangent set seen so far
        cudaFree(ctx->unit_tan); ctx->unit_tan = nullptr; ctx->unit_tan_nt = 0;
        if (cudaMalloc(&ctx->unit_tan, sizeof(double) * NT * ctx->cap_units) != cudaSuccess) return ULENS_ENOMEM;
        ctx->unit_tan_nt = NT;
    }
    // box lists of one chunk, sized for the widest lens multiplicity seen so far (first use only)
    constexpr int BCAP = BoxCap<N>::value;
    if (ctx->boxes_cap < BCAP) {
        cudaFree(ctx->boxes); ctx->boxes = nullptr; ctx->boxes_cap = 0;
        if (cudaMalloc(&ctx->boxes, sizeof(SubBox) * BCAP * (size_t)ctx->chunk) != cudaSuccess) return ULENS_ENOMEM;
        ctx->boxes_cap = BCAP;
    }
    if (dual && ctx->exts_cap < BCAP) {
        cudaFree(ctx->exts); ctx->exts = nullptr; ctx->exts_cap = 0;
        if (cudaMalloc(&ctx->exts, sizeof(BoxExt) * BCAP * (size_t)ctx->chunk) != cudaSuccess) return ULENS_ENOMEM;
        ctx->exts_cap = BCAP;
    }
    int sm_count = 148;
    cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, ctx->device);
    for (long long base = 0; base < n_total; base += ctx->chunk) {
        int n = (int)((n_total - base < ctx->chunk) ? (n_total - base) : ctx->chunk);
        CK(cudaMemsetAsync(ctx->cc, 0, sizeof(ChunkCounters), st));
        {
            KTimer kt(ctx, ULENS_K_ROOTS, st);
            k_roots<N><<<(n + 127) / 128, 128, 0, st>>>(n, (int)base, n_pts, ctx->cfg_dev, ctx->poly_dev, w_re, w_im,
                                                        nullptr, nullptr, nullptr, ctx->status_ws, ctx->c_zr, ctx->c_zi, ctx->c_mask, nullptr, nullptr, pmap, n_dev);
        }
        // quiet source points take the coarse limb sampling (first pass only: the retry pass is for doubtful points)
        // (whatever the size of the call or the chunk: a point's result must not depend on what it is batched with)
        const bool use_quiet = !(ctx->opt.flags & ULENS_OPT_NO_QUIET) && st_or == 0 && ctx->quiet != nullptr;
        if (use_quiet) {
            KTimer kt(ctx, ULENS_K_ROOTS, st);
            k_quiet<N><<<(n + 127) / 128, 128, 0, st>>>(n, (int)base, n_pts, ctx->cfg_dev, ctx->poly_dev, w_re, w_im, UL_QUIET_TOL, ctx->quiet, ctx->quiet_drho, ctx->limb_list, ctx->cc, pmap, n_dev);
            ctx->last_launches += 1;
        }
        const unsigned char* quiet = use_quiet ? ctx->quiet : nullptr;
        {
            KTimer kt(ctx, ULENS_K_LIMB, st);
            CK(cudaMemsetAsync(ctx->n_boxes, 0, sizeof(int) * (size_t)n, st));
            const unsigned limb_grid = (unsigned)(((long long)n * LimbGeom<N>::WARPS + 3) / 4);
            if (dual)
                k_limb<N, true><<<limb_grid, 128, 0, st>>>(n, (int)base, n_pts, ctx->cfg_dev, ctx->poly_dev, w_re, w_im, rp,
                                                                    ctx->boxes, ctx->exts, ctx->n_boxes, ctx->status_ws, ctx->counters,
                                                                    ctx->c_zr, ctx->c_zi, ctx->c_mask, pmap, n_dev, quiet,
                                                                    quiet ? ctx->limb_list : nullptr, ctx->cc);
            else
                k_limb<N, false><<<limb_grid, 128, 0, st>>>(n, (int)base, n_pts, ctx->cfg_dev, ctx->poly_dev, w_re, w_im, rp,
                                                                     ctx->boxes, ctx->exts, ctx->n_boxes, ctx->status_ws, ctx->counters,
                                                                     ctx->c_zr, ctx->c_zi, ctx->c_mask, pmap, n_dev, quiet,
                                                                     quiet ? ctx->limb_list : nullptr, ctx->cc);
        }
        {
            KTimer kt(ctx, ULENS_K_SECTORS, st);
            k_sectors<N><<<(n + 127) / 128, 128, 0, st>>>(n, (int)base, n_pts, ctx->cfg_dev, w_re, w_im, rp, ctx->boxes, ctx->exts,
                                                           ctx->n_boxes, ctx->patches, ctx->n_patch, ctx->status_ws, ctx->unit_desc,
                                                           (unsigned)ctx->cap_units, ctx->cc, ctx->counters, tans, ctx->ptans, pmap, n_dev, quiet,
                                                           ctx->c_zr, ctx->c_zi, ctx->c_mask);
        }
        // persistent grid: as many CTAs as are resident at once (occupancy API; 4-6 per SM by register count)
        int per_sm = 4;
        if (dual) {
            if (ld) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_shoot_dual<N, true>, 128, 0);
            else cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_shoot_dual<N, false>, 128, 0);
        } else if (ctx->opt.flags & ULENS_OPT_F32_SHOOT) {
            if (ld) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_shoot_f32<N, true>, 128, 0);
            else cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_shoot_f32<N, false>, 128, 0);
        } else {
            if (ld) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_shoot<N, true>, 128, 0);
            else cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_shoot<N, false>, 128, 0);
        }
        if (per_sm < 1) per_sm = 1;
        int grid = sm_count * per_sm;
        {
            KTimer kt(ctx, ULENS_K_SHOOT, st);
            if (dual && ld)
                k_shoot_dual<N, true><<<grid, 128, 0, st>>>((int)base, n_pts, ctx->cfg_dev, tans, w_re, w_im, ctx->patches, ctx->ptans,
                                                            ctx->unit_desc, ctx->unit_sum, ctx->unit_odd, ctx->unit_tan, ctx->status_ws,
                                                            ctx->cc, ctx->counters, (unsigned)ctx->cap_units, pmap);
            else if (dual)
                k_shoot_dual<N, false><<<grid, 128, 0, st>>>((int)base, n_pts, ctx->cfg_dev, tans, w_re, w_im, ctx->patches, ctx->ptans,
                                                             ctx->unit_desc, ctx->unit_sum, ctx->unit_odd, ctx->unit_tan, ctx->status_ws,
                                                             ctx->cc, ctx->counters, (unsigned)ctx->cap_units, pmap);
            else if (ctx->opt.flags & ULENS_OPT_F32_SHOOT) {
                if (ld)
                    k_shoot_f32<N, true><<<grid, 128, 0, st>>>((int)base, n_pts, ctx->cfg_dev, w_re, w_im, ctx->patches, ctx->unit_desc,
                                                               ctx->unit_sum, ctx->unit_odd, ctx->status_ws, ctx->cc, ctx->counters, (unsigned)ctx->cap_units, pmap);
                else
                    k_shoot_f32<N, false><<<grid, 128, 0, st>>>((int)base, n_pts, ctx->cfg_dev, w_re, w_im, ctx->patches, ctx->unit_desc,
                                                                ctx->unit_sum, ctx->unit_odd, ctx->status_ws, ctx->cc, ctx->counters, (unsigned)ctx->cap_units, pmap);
            }
            else if (ld)
                k_shoot<N, true><<<grid, 128, 0, st>>>((int)base, n_pts, ctx->cfg_dev, w_re, w_im, ctx->patches, ctx->unit_desc,
                                                       ctx->unit_sum, ctx->unit_odd, ctx->status_ws, ctx->cc, ctx->counters, (unsigned)ctx->cap_units, pmap);
            else
                k_shoot<N, false><<<grid, 128, 0, st>>>((int)base, n_pts, ctx->cfg_dev, w_re, w_im, ctx->patches, ctx->unit_desc,
                                                        ctx->unit_sum, ctx->unit_odd, ctx->status_ws, ctx->cc, ctx->counters, (unsigned)ctx->cap_units, pmap);
        }
        {
            KTimer kt(ctx, ULENS_K_FINALIZE, st);
            k_finalize<<<(n + 127) / 128, 128, 0, st>>>(n, (int)base, n_pts, ctx->cfg_dev, ctx->patches, ctx->n_patch,
                                                        ctx->unit_sum, ctx->unit_odd, ctx->status_ws, ctx->opt.rel_tol,
                                                        A_out, err_out, status_out, ctx->counters, pmap, n_dev, st_or);
            if (dual) {
                k_finalize_dual<NT><<<(n + 127) / 128, 128, 0, st>>>(n, (int)base, n_pts, ctx->cfg_dev, tans, ctx->patches, ctx->n_patch,
                                                                 ctx->unit_sum, ctx->unit_tan, grad5_out, pmap, n_dev, st_or ? status_out : nullptr,
                                                                 quiet, ctx->quiet_drho);
                ctx->last_launches += 1;
            }
        }
        ctx->last_launches += 5;
        CK(cudaGetLastError());
    }
    return ULENS_OK;
}

static int ensure_ext_buffers(ulens_ctx* ctx, size_t n)
{
    if (n <= ctx->ext_cap) return ULENS_OK;
    cudaFree(ctx->ext_flag); cudaFree(ctx->ext_map); cudaFree(ctx->ext_blk);
    ctx->ext_flag = nullptr; ctx->ext_map = nullptr; ctx->ext_blk = nullptr; ctx->ext_cap = 0;
    if (cudaMalloc(&ctx->ext_flag, n) != cudaSuccess) return ULENS_ENOMEM;
    if (cudaMalloc(&ctx->ext_map, sizeof(int) * n) != cudaSuccess) return ULENS_ENOMEM;
    if (cudaMalloc(&ctx->ext_blk, sizeof(unsigned) * ((n + 1023) / 1024 + 1)) != cudaSuccess) return ULENS_ENOMEM;
    ctx->ext_cap = n;
    return ULENS_OK;
}

// Retry pass. The points whose finite-source result came back doubtful (UL_ST_RETRY_MASK: an inside
// ray on a sector border, self-check above rel_tol, sector cap, EA cap, no image-limb point) are gathered and
// integrated once more with twice the limb samples (Eq. 8), which moves every sector border; the new result and
// status (| ULENS_ST_RETRIED) replace the old ones. Their number stays on the device -- the launches are sized for
// the worst case (one chunk; further flagged points keep their first result) -- so nothing synchronises.
template <int N>
static int retry_flagged(ulens_ctx* ctx, long long n_total, int n_pts, bool ld, const double* w_re, const double* w_im,
                         double* A_out, double* err_out, unsigned* status, cudaStream_t st, double* grad5_out)
{
    if (ctx->opt.flags & ULENS_OPT_NO_RETRY) return ULENS_OK;
    int rc = ensure_ext_buffers(ctx, (size_t)n_total);
    if (rc != ULENS_OK) return rc;
    const int n = (int)n_total, n_blk = (int)((n_total + 1023) / 1024);
    k_retry_flag<<<(unsigned)((n_total + 255) / 256), 256, 0, st>>>(n, status, ctx->ext_flag);
    k_ext_count<<<n_blk, 1024, 0, st>>>(n, ctx->ext_flag, ctx->ext_blk);
    k_ext_scan<<<1, 1024, 0, st>>>(n_blk, ctx->ext_blk);
    k_ext_scatter<<<n_blk, 1024, 0, st>>>(n, ctx->ext_flag, ctx->ext_blk, ctx->ext_map);
    ctx->last_launches += 4;
    CK(cudaGetLastError());
    RegionParams rp2 = ctx->rp;
    rp2.n_limb = ctx->rp.n_limb * 2 > 8192 ? 8192 : ctx->rp.n_limb * 2;
    // launches are sized for two chunks of doubtful points (their number stays on the device); any beyond that keep
    // their first result and status, without ULENS_ST_RETRIED
    const long long n_max = n_total < 2LL * ctx->chunk ? n_total : 2LL * ctx->chunk;
    return run_chunks<N>(ctx, n_max, n_pts, ld, w_re, w_im, A_out, err_out, status, st, grad5_out, ctx->ext_map,
                         ctx->ext_blk + n_blk, &rp2, UL_ST_RETRIED);
}

// Tangent tables of the intrinsic directions (ulens_dual.cuh): binary / single (w_cx, w_cy, s, q, rho), triple
// (w_cx, w_cy, s, q, q3, r3, psi, rho). The lens-parameter directions exist in the geometry of ulens_lens_binary
// (G4: s = a_2 - a_1, q = eps_2 / eps_1, barycentre of M1, M2 at the origin) and ulens_lens_triple (G5: q3 = eps_3 / eps_1,
// a_3 = midpoint of M1-M2 + r3 e^{i psi}); (s, q, q3, r3, psi) are recovered from the lens and the geometry is checked.
static int upload_tangents(ulens_ctx* ctx, int n_cfg, const ulens_lens* lenses, cudaStream_t st)
{
    if (ctx->last_tan_valid && ctx->tan_dev) return ULENS_OK;       // same lens array as the last call (upload_cfgs checked)
    std::vector<TangentTable> tt(n_cfg);
    for (int c = 0; c < n_cfg; ++c) {
        TangentTable& T = tt[c];
        memset(&T, 0, sizeof T);
        const ulens_lens& L = lenses[c];
        const int NT = L.n_lens == 3 ? 8 : 5;
        T.dwx[0] = 1.0; T.dwy[1] = 1.0; T.drho[NT - 1] = 1.0;
        if (L.n_lens >= 2) {
            const double s = L.ax[1] - L.ax[0], q = L.eps[1] / L.eps[0];
            if (L.ay[0] != 0.0 || L.ay[1] != 0.0 || fabs(L.eps[0] * L.ax[0] + L.eps[1] * L.ax[1]) > 1e-12 * (1.0 + fabs(s)))
                return ULENS_EUNSUPPORTED;               // not the ulens_lens_binary / ulens_lens_triple geometry
            const double o = 1.0 / (1.0 + q);
            T.dax[2][0] = -q * o; T.dax[2][1] = o;                       // d/ds
            T.dax[3][0] = -s * o * o; T.dax[3][1] = -s * o * o;          // d/dq: positions
            if (L.n_lens == 2) {
                T.deps[3][0] = -o * o; T.deps[3][1] = o * o;             // d/dq: masses
            } else {
                const double q3 = L.eps[2] / L.eps[0], tot = 1.0 + q + q3, it2 = 1.0 / (tot * tot);
                const double mid = 0.5 * (L.ax[0] + L.ax[1]);
                const double r3x = L.ax[2] - mid, r3y = L.ay[2], r3 = sqrt(r3x * r3x + r3y * r3y);
                if (!(r3 > 0.0)) return ULENS_EUNSUPPORTED;
                T.dax[2][2] = 0.5 * (1.0 - q) * o;                       // the midpoint moves with s ...
                T.dax[3][2] = -s * o * o;                                // ... and with q
                T.deps[3][0] = -it2; T.deps[3][1] = (1.0 + q3) * it2; T.deps[3][2] = -q3 * it2;      // d/dq
                T.deps[4][0] = -it2; T.deps[4][1] = -q * it2; T.deps[4][2] = (1.0 + q) * it2;        // d/dq3
                T.dax[5][2] = r3x / r3; T.day[5][2] = r3y / r3;          // d/dr3
                T.dax[6][2] = -r3y; T.day[6][2] = r3x;                   // d/dpsi
            }
        }
    }
    if ((size_t)n_cfg > ctx->tan_cap) {
        cudaFree(ctx->tan_dev); ctx->tan_dev = nullptr; ctx->tan_cap = 0;
        if (cudaMalloc(&ctx->tan_dev, sizeof(TangentTable) * ((size_t)n_cfg + 64)) != cudaSuccess) return ULENS_ENOMEM;
        ctx->tan_cap = (size_t)n_cfg + 64;
    }
    int rc = stage_upload(ctx, ctx->tan_dev, tt.data(), sizeof(TangentTable) * n_cfg, st);
    if (rc != ULENS_OK) return rc;
    ctx->last_tan_valid = true;
    return ULENS_OK;
}

static int mag_device(ulens_ctx* ctx, int n_cfg, int n_pts, const ulens_lens* lenses, const double* rho, const double* u1,
                      const double* w_re, const double* w_im, double* A_out, double* err_out, unsigned* status_out,
                      cudaStream_t st, double* grad5_out = nullptr)
{
    int N = 0; bool ld = false;
    int rc = upload_cfgs(ctx, n_cfg, lenses, rho, u1, st, &N, &ld);
    if (rc != ULENS_OK) return rc;
    if (grad5_out) {
        rc = upload_tangents(ctx, n_cfg, lenses, st);
        if (rc != ULENS_OK) return rc;
    }
    long long n_total = (long long)n_cfg * n_pts;
    if (n_total > UL_MAX_POINTS) return ULENS_EUNSUPPORTED;
    ctx->last_launches = 0;
    if (!status_out) {                                   // the retry pass needs every point's status
        if ((size_t)n_total > ctx->st_all_cap) {
            cudaFree(ctx->st_all); ctx->st_all = nullptr; ctx->st_all_cap = 0;
            if (cudaMalloc(&ctx->st_all, sizeof(unsigned) * (size_t)n_total) != cudaSuccess) return ULENS_ENOMEM;
            ctx->st_all_cap = (size_t)n_total;
        }
        status_out = ctx->st_all;
    }
    switch (N) {
        case 1: rc = run_chunks<1>(ctx, n_total, n_pts, ld, w_re, w_im, A_out, err_out, status_out, st, grad5_out);
                if (rc == ULENS_OK) rc = retry_flagged<1>(ctx, n_total, n_pts, ld, w_re, w_im, A_out, err_out, status_out, st, grad5_out);
                break;
        case 2: rc = run_chunks<2>(ctx, n_total, n_pts, ld, w_re, w_im, A_out, err_out, status_out, st, grad5_out);
                if (rc == ULENS_OK) rc = retry_flagged<2>(ctx, n_total, n_pts, ld, w_re, w_im, A_out, err_out, status_out, st, grad5_out);
                break;
        default: rc = run_chunks<3>(ctx, n_total, n_pts, ld, w_re, w_im, A_out, err_out, status_out, st, grad5_out);
                if (rc == ULENS_OK) rc = retry_flagged<3>(ctx, n_total, n_pts, ld, w_re, w_im, A_out, err_out, status_out, st, grad5_out);
                break;
    }
    return rc;
}

extern "C" int ulens_mag(ulens_ctx* ctx, int n_cfg, int n_pts, const ulens_lens* lenses_host, const double* rho_host,
                         const double* u1_host, const double* w_re, const double* w_im, double* A_out, double* err_out,
                         uint32_t* status_out, void* stream)
{
    if (!ctx || n_cfg < 0 || n_pts < 0) return ULENS_EINVAL;
    if (n_cfg == 0 || n_pts == 0) return ULENS_OK;
    if (!lenses_host || !rho_host || !u1_host || !w_re || !w_im || !A_out) return ULENS_EINVAL;
    CK(cudaSetDevice(ctx->device));
    return mag_device(ctx, n_cfg, n_pts, lenses_host, rho_host, u1_host, w_re, w_im, A_out, err_out, status_out,
                      (cudaStream_t)stream);
}

extern "C" int ulens_mag_grad(ulens_ctx* ctx, int n_cfg, int n_pts, const ulens_lens* lenses_host, const double* rho_host,
                              const double* u1_host, const double* w_re, const double* w_im, double* A_out, double* dA5_out,
                              double* err_out, uint32_t* status_out, void* stream)
{
    if (!ctx || n_cfg < 0 || n_pts < 0) return ULENS_EINVAL;
    if (n_cfg == 0 || n_pts == 0) return ULENS_OK;
    if (!lenses_host || !rho_host || !u1_host || !w_re || !w_im || !A_out || !dA5_out) return ULENS_EINVAL;
    CK(cudaSetDevice(ctx->device));
    return mag_device(ctx, n_cfg, n_pts, lenses_host, rho_host, u1_host, w_re, w_im, A_out, err_out, status_out,
                      (cudaStream_t)stream, dA5_out);
}

extern "C" int ulens_mag_host(ulens_ctx* ctx, int n_cfg, int n_pts, const ulens_lens* lenses_host, const double* rho_host,
                              const double* u1_host, const double* w_re_host, const double* w_im_host, double* A_out_host,
                              double* err_out_host, uint32_t* status_out_host, void* stream)
{
    if (!ctx || n_cfg < 0 || n_pts < 0) return ULENS_EINVAL;
    if (n_cfg == 0 || n_pts == 0) return ULENS_OK;
    if (!lenses_host || !rho_host || !u1_host || !w_re_host || !w_im_host || !A_out_host) return ULENS_EINVAL;
    CK(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    size_t n = (size_t)n_cfg * n_pts;
    size_t need = n * 5;                                 // w_re, w_im, A, err, status (as 8-byte slots)
    if (need > ctx->io_cap) {
        cudaFree(ctx->io_buf); ctx->io_buf = nullptr; ctx->io_cap = 0;
        if (cudaMalloc(&ctx->io_buf, sizeof(double) * need) != cudaSuccess) return ULENS_ENOMEM;
        ctx->io_cap = need;
    }
    double* d_wre = ctx->io_buf; double* d_wim = d_wre + n; double* d_A = d_wim + n; double* d_err = d_A + n;
    unsigned* d_st = reinterpret_cast<unsigned*>(d_err + n);
    CK(cudaMemcpyAsync(d_wre, w_re_host, sizeof(double) * n, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(d_wim, w_im_host, sizeof(double) * n, cudaMemcpyHostToDevice, st));
    int rc = mag_device(ctx, n_cfg, n_pts, lenses_host, rho_host, u1_host, d_wre, d_wim, d_A, d_err, d_st, st);
    if (rc != ULENS_OK) return rc;
    CK(cudaMemcpyAsync(A_out_host, d_A, sizeof(double) * n, cudaMemcpyDeviceToHost, st));
    if (err_out_host) CK(cudaMemcpyAsync(err_out_host, d_err, sizeof(double) * n, cudaMemcpyDeviceToHost, st));
    if (status_out_host) CK(cudaMemcpyAsync(status_out_host, d_st, sizeof(unsigned) * n, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return ULENS_OK;
}

extern "C" int ulens_trajectory(ulens_ctx* ctx, int n_cfg, int n_epochs, const double* theta_host, const double* t,
                                double* w_re_out, double* w_im_out, void* stream)
{
    if (!ctx || n_cfg < 0 || n_epochs < 0) return ULENS_EINVAL;
    if (n_cfg == 0 || n_epochs == 0) return ULENS_OK;
    if (!theta_host || !t || !w_re_out || !w_im_out) return ULENS_EINVAL;
    for (int c = 0; c < n_cfg; ++c) {
        const double* th = theta_host + 7 * c;
        if (!isfinite(th[0]) || !isfinite(th[1]) || !isfinite(th[6]) || !finite_pos(th[2])) return ULENS_EINVAL;
    }
    CK(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n = (size_t)n_cfg * n_epochs;
    if (n > (size_t)UL_MAX_POINTS) return ULENS_EUNSUPPORTED;
    const size_t need = 7 * (size_t)n_cfg;
    if (need > ctx->traj_cap) {
        cudaFree(ctx->traj_w); ctx->traj_w = nullptr; ctx->traj_cap = 0;
        if (cudaMalloc(&ctx->traj_w, sizeof(double) * need) != cudaSuccess) return ULENS_ENOMEM;
        ctx->traj_cap = need;
    }
    int rc = stage_upload(ctx, ctx->traj_w, theta_host, sizeof(double) * 7 * n_cfg, st);
    if (rc != ULENS_OK) return rc;
    k_traj<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n_cfg, n_epochs, ctx->traj_w, t, w_re_out, w_im_out);
    ctx->last_launches = 1;
    CK(cudaGetLastError());
    return ULENS_OK;
}

extern "C" int ulens_lightcurve_binary(ulens_ctx* ctx, int n_cfg, int n_epochs, const double* theta_host, double u1,
                                       const double* t, double* A_out, double* dA_out, double* err_out,
                                       uint32_t* status_out, void* stream)
{
    if (!ctx || n_cfg < 0 || n_epochs < 0) return ULENS_EINVAL;
    if (n_cfg == 0 || n_epochs == 0) return ULENS_OK;
    if (!theta_host || !t || !A_out || !(u1 >= 0.0 && u1 <= 1.0)) return ULENS_EINVAL;
    CK(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    std::vector<ulens_lens> lenses(n_cfg);
    std::vector<double> rho(n_cfg), u1v(n_cfg, u1);
    for (int c = 0; c < n_cfg; ++c) {
        const double* th = theta_host + 7 * c;
        for (int k = 0; k < 7; ++k) if (!isfinite(th[k])) return ULENS_EINVAL;
        if (!(th[2] > 0.0)) return ULENS_EINVAL;
        int rc = ulens_lens_binary(&lenses[c], th[3], th[4]);
        if (rc != ULENS_OK) return rc;
        rho[c] = th[5];
    }
    size_t n = (size_t)n_cfg * n_epochs;
    size_t need = 2 * n + 7 * (size_t)n_cfg + (dA_out ? UL_NT * n : 0);
    if (need > ctx->traj_cap) {
        cudaFree(ctx->traj_w); ctx->traj_w = nullptr; ctx->traj_cap = 0;
        if (cudaMalloc(&ctx->traj_w, sizeof(double) * need) != cudaSuccess) return ULENS_ENOMEM;
        ctx->traj_cap = need;
    }
    double* w_re = ctx->traj_w; double* w_im = w_re + n; double* th_dev = w_im + n;
    double* g5 = dA_out ? th_dev + 7 * (size_t)n_cfg : nullptr;
    {
        int rcu = stage_upload(ctx, th_dev, theta_host, sizeof(double) * 7 * n_cfg, st);
        if (rcu != ULENS_OK) return rcu;
    }
    {
        KTimer kt(ctx, ULENS_K_TRAJ, st);
        k_traj<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n_cfg, n_epochs, th_dev, t, w_re, w_im);
    }
    CK(cudaGetLastError());
    int rc = mag_device(ctx, n_cfg, n_epochs, lenses.data(), rho.data(), u1v.data(), w_re, w_im, A_out, err_out, status_out, st, g5);
    ctx->last_launches += 1;
    if (rc != ULENS_OK) return rc;
    if (dA_out) {
        k_chain7<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n_cfg, n_epochs, th_dev, t, w_re, w_im, g5, dA_out);
        ctx->last_launches += 1;
        CK(cudaGetLastError());
    }
    return rc;
}

extern "C" int ulens_lightcurve_triple(ulens_ctx* ctx, int n_cfg, int n_epochs, const double* theta_host, double u1,
                                       const double* t, double* A_out, double* dA_out, double* err_out,
                                       uint32_t* status_out, void* stream)
{
    if (!ctx || n_cfg < 0 || n_epochs < 0) return ULENS_EINVAL;
    if (n_cfg == 0 || n_epochs == 0) return ULENS_OK;
    if (!theta_host || !t || !A_out || !(u1 >= 0.0 && u1 <= 1.0)) return ULENS_EINVAL;
    CK(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    std::vector<ulens_lens> lenses(n_cfg);
    std::vector<double> rho(n_cfg), u1v(n_cfg, u1);
    for (int c = 0; c < n_cfg; ++c) {
        const double* th = theta_host + 10 * c;
        for (int k = 0; k < 10; ++k) if (!isfinite(th[k])) return ULENS_EINVAL;
        if (!(th[2] > 0.0)) return ULENS_EINVAL;
        int rc = ulens_lens_triple(&lenses[c], th[3], th[4], th[7], th[8], th[9]);
        if (rc != ULENS_OK) return rc;
        rho[c] = th[5];
    }
    size_t n = (size_t)n_cfg * n_epochs;
    if (n > (size_t)UL_MAX_POINTS) return ULENS_EUNSUPPORTED;
    size_t need = 2 * n + 10 * (size_t)n_cfg + (dA_out ? 8 * n : 0);
    if (need > ctx->traj_cap) {
        cudaFree(ctx->traj_w); ctx->traj_w = nullptr; ctx->traj_cap = 0;
        if (cudaMalloc(&ctx->traj_w, sizeof(double) * need) != cudaSuccess) return ULENS_ENOMEM;
        ctx->traj_cap = need;
    }
    double* w_re = ctx->traj_w; double* w_im = w_re + n; double* th_dev = w_im + n;
    double* g8 = dA_out ? th_dev + 10 * (size_t)n_cfg : nullptr;
    {
        int rcu = stage_upload(ctx, th_dev, theta_host, sizeof(double) * 10 * n_cfg, st);
        if (rcu != ULENS_OK) return rcu;
    }
    {
        KTimer kt(ctx, ULENS_K_TRAJ, st);
        k_traj10<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n_cfg, n_epochs, th_dev, t, w_re, w_im);
    }
    CK(cudaGetLastError());
    int rc = mag_device(ctx, n_cfg, n_epochs, lenses.data(), rho.data(), u1v.data(), w_re, w_im, A_out, err_out, status_out, st, g8);
    ctx->last_launches += 1;
    if (rc != ULENS_OK) return rc;
    if (dA_out) {
        k_chain10<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n_cfg, n_epochs, th_dev, t, w_re, w_im, g8, dA_out);
        ctx->last_launches += 1;
        CK(cudaGetLastError());
    }
    return rc;
}

extern "C" int ulens_lightcurve_triple_host(ulens_ctx* ctx, int n_cfg, int n_epochs, const double* theta_host, double u1,
                                            const double* t_host, double* A_out_host, double* dA_out_host,
                                            double* err_out_host, uint32_t* status_out_host, void* stream)
{
    if (!ctx || n_cfg < 0 || n_epochs < 0) return ULENS_EINVAL;
    if (n_cfg == 0 || n_epochs == 0) return ULENS_OK;
    if (!theta_host || !t_host || !A_out_host) return ULENS_EINVAL;
    CK(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n = (size_t)n_cfg * n_epochs;
    const size_t need = (size_t)n_epochs + n * (3 + (dA_out_host ? 10 : 0));   // t, A, err, status (8-byte slots), dA
    if (need > ctx->io_cap) {
        cudaFree(ctx->io_buf); ctx->io_buf = nullptr; ctx->io_cap = 0;
        if (cudaMalloc(&ctx->io_buf, sizeof(double) * need) != cudaSuccess) return ULENS_ENOMEM;
        ctx->io_cap = need;
    }
    double* d_t = ctx->io_buf; double* d_A = d_t + n_epochs; double* d_err = d_A + n;
    unsigned* d_st = reinterpret_cast<unsigned*>(d_err + n);
    double* d_dA = dA_out_host ? d_err + 2 * n : nullptr;
    CK(cudaMemcpyAsync(d_t, t_host, sizeof(double) * n_epochs, cudaMemcpyHostToDevice, st));
    int rc = ulens_lightcurve_triple(ctx, n_cfg, n_epochs, theta_host, u1, d_t, d_A, d_dA, d_err, d_st, stream);
    if (rc != ULENS_OK) return rc;
    CK(cudaMemcpyAsync(A_out_host, d_A, sizeof(double) * n, cudaMemcpyDeviceToHost, st));
    if (dA_out_host) CK(cudaMemcpyAsync(dA_out_host, d_dA, sizeof(double) * 10 * n, cudaMemcpyDeviceToHost, st));
    if (err_out_host) CK(cudaMemcpyAsync(err_out_host, d_err, sizeof(double) * n, cudaMemcpyDeviceToHost, st));
    if (status_out_host) CK(cudaMemcpyAsync(status_out_host, d_st, sizeof(unsigned) * n, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return ULENS_OK;
}

extern "C" int ulens_lightcurve_binary_ext(ulens_ctx* ctx, int n_cfg, int n_epochs, const double* theta_host, double u1,
                                           const double* t, const uint8_t* ext_mask, double sel_tol, double* A_out,
                                           double* dA_out, double* err_out, uint32_t* status_out, int* n_ext_out,
                                           void* stream)
{
    if (n_ext_out) *n_ext_out = 0;
    if (!ctx || n_cfg < 0 || n_epochs < 0) return ULENS_EINVAL;
    if (n_cfg == 0 || n_epochs == 0) return ULENS_OK;
    if (!theta_host || !t || !A_out || !(u1 >= 0.0 && u1 <= 1.0) || !isfinite(sel_tol)) return ULENS_EINVAL;
    if (!(sel_tol > 0.0)) sel_tol = 2e-5;
    CK(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    std::vector<ulens_lens> lenses(n_cfg);
    std::vector<double> rho(n_cfg), u1v(n_cfg, u1);
    for (int c = 0; c < n_cfg; ++c) {
        const double* th = theta_host + 7 * c;
        for (int k = 0; k < 7; ++k) if (!isfinite(th[k])) return ULENS_EINVAL;
        if (!(th[2] > 0.0)) return ULENS_EINVAL;
        int rc = ulens_lens_binary(&lenses[c], th[3], th[4]);
        if (rc != ULENS_OK) return rc;
        rho[c] = th[5];
    }
    const size_t n = (size_t)n_cfg * n_epochs;
    if (n > (size_t)UL_MAX_POINTS) return ULENS_EUNSUPPORTED;
    size_t need = 2 * n + 7 * (size_t)n_cfg + (dA_out ? UL_NT * n : 0);
    if (need > ctx->traj_cap) {
        cudaFree(ctx->traj_w); ctx->traj_w = nullptr; ctx->traj_cap = 0;
        if (cudaMalloc(&ctx->traj_w, sizeof(double) * need) != cudaSuccess) return ULENS_ENOMEM;
        ctx->traj_cap = need;
    }
    const int n_blk = (int)((n + 1023) / 1024);
    {
        int rc = ensure_ext_buffers(ctx, n);
        if (rc != ULENS_OK) return rc;
    }
    if (!status_out) {
        if (n > ctx->st_all_cap) {
            cudaFree(ctx->st_all); ctx->st_all = nullptr; ctx->st_all_cap = 0;
            if (cudaMalloc(&ctx->st_all, sizeof(unsigned) * n) != cudaSuccess) return ULENS_ENOMEM;
            ctx->st_all_cap = n;
        }
        status_out = ctx->st_all;
    }
    double* w_re = ctx->traj_w; double* w_im = w_re + n; double* th_dev = w_im + n;
    double* g5 = dA_out ? th_dev + 7 * (size_t)n_cfg : nullptr;
    {
        int rcu = stage_upload(ctx, th_dev, theta_host, sizeof(double) * 7 * n_cfg, st);
        if (rcu != ULENS_OK) return rcu;
    }
    {
        KTimer kt(ctx, ULENS_K_TRAJ, st);
        k_traj<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n_cfg, n_epochs, th_dev, t, w_re, w_im);
    }
    CK(cudaGetLastError());
    int N = 0; bool ld = false;
    int rc = upload_cfgs(ctx, n_cfg, lenses.data(), rho.data(), u1v.data(), st, &N, &ld);
    if (rc != ULENS_OK) return rc;
    if (dA_out) {
        rc = upload_tangents(ctx, n_cfg, lenses.data(), st);
        if (rc != ULENS_OK) return rc;
    }
    ctx->last_launches = 1;
    // every epoch: point-source value (and tangents) + the decision; then the ordered gather map of the N_ext epochs
    {
        KTimer kt(ctx, ULENS_K_ROOTS, st);
        k_point_ext<2><<<(unsigned)((n + 127) / 128), 128, 0, st>>>((int)n, n_epochs, ctx->cfg_dev, ctx->poly_dev,
                                                                    dA_out ? ctx->tan_dev : nullptr, w_re, w_im, ext_mask, sel_tol,
                                                                    A_out, err_out, status_out, g5, ctx->ext_flag);
    }
    k_ext_count<<<n_blk, 1024, 0, st>>>((int)n, ctx->ext_flag, ctx->ext_blk);
    k_ext_scan<<<1, 1024, 0, st>>>(n_blk, ctx->ext_blk);
    k_ext_scatter<<<n_blk, 1024, 0, st>>>((int)n, ctx->ext_flag, ctx->ext_blk, ctx->ext_map);
    ctx->last_launches += 4;
    CK(cudaGetLastError());
    unsigned n_ext = 0;
    CK(cudaMemcpyAsync(&n_ext, ctx->ext_blk + n_blk, sizeof(unsigned), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    if (n_ext_out) *n_ext_out = (int)n_ext;
    if (n_ext > 0) {
        rc = run_chunks<2>(ctx, (long long)n_ext, n_epochs, ld, w_re, w_im, A_out, err_out, status_out, st, g5, ctx->ext_map);
        if (rc == ULENS_OK) rc = retry_flagged<2>(ctx, (long long)n, n_epochs, ld, w_re, w_im, A_out, err_out, status_out, st, g5);
        if (rc != ULENS_OK) return rc;
    }
    if (dA_out) {
        k_chain7<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n_cfg, n_epochs, th_dev, t, w_re, w_im, g5, dA_out);
        ctx->last_launches += 1;
        CK(cudaGetLastError());
    }
    return ULENS_OK;
}

extern "C" int ulens_lightcurve_binary_host(ulens_ctx* ctx, int n_cfg, int n_epochs, const double* theta_host, double u1,
                                            const double* t_host, double* A_out_host, double* dA_out_host,
                                            double* err_out_host, uint32_t* status_out_host, void* stream)
{
    if (!ctx || n_cfg < 0 || n_epochs < 0) return ULENS_EINVAL;
    if (n_cfg == 0 || n_epochs == 0) return ULENS_OK;
    if (!theta_host || !t_host || !A_out_host) return ULENS_EINVAL;
    CK(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n = (size_t)n_cfg * n_epochs;
    const size_t need = (size_t)n_epochs + n * (3 + (dA_out_host ? 7 : 0));   // t, A, err, status (8-byte slots), dA
    if (need > ctx->io_cap) {
        cudaFree(ctx->io_buf); ctx->io_buf = nullptr; ctx->io_cap = 0;
        if (cudaMalloc(&ctx->io_buf, sizeof(double) * need) != cudaSuccess) return ULENS_ENOMEM;
        ctx->io_cap = need;
    }
    double* d_t = ctx->io_buf; double* d_A = d_t + n_epochs; double* d_err = d_A + n;
    unsigned* d_st = reinterpret_cast<unsigned*>(d_err + n);
    double* d_dA = dA_out_host ? d_err + 2 * n : nullptr;
    CK(cudaMemcpyAsync(d_t, t_host, sizeof(double) * n_epochs, cudaMemcpyHostToDevice, st));
    int rc = ulens_lightcurve_binary(ctx, n_cfg, n_epochs, theta_host, u1, d_t, d_A, d_dA, d_err, d_st, stream);
    if (rc != ULENS_OK) return rc;
    CK(cudaMemcpyAsync(A_out_host, d_A, sizeof(double) * n, cudaMemcpyDeviceToHost, st));
    if (dA_out_host) CK(cudaMemcpyAsync(dA_out_host, d_dA, sizeof(double) * 7 * n, cudaMemcpyDeviceToHost, st));
    if (err_out_host) CK(cudaMemcpyAsync(err_out_host, d_err, sizeof(double) * n, cudaMemcpyDeviceToHost, st));
    if (status_out_host) CK(cudaMemcpyAsync(status_out_host, d_st, sizeof(unsigned) * n, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return ULENS_OK;
}

extern "C" int ulens_lightcurve_binary_ext_host(ulens_ctx* ctx, int n_cfg, int n_epochs, const double* theta_host, double u1,
                                                const double* t_host, const uint8_t* ext_mask_host, double sel_tol,
                                                double* A_out_host, double* dA_out_host, double* err_out_host,
                                                uint32_t* status_out_host, int* n_ext_out, void* stream)
{
    if (n_ext_out) *n_ext_out = 0;
    if (!ctx || n_cfg < 0 || n_epochs < 0) return ULENS_EINVAL;
    if (n_cfg == 0 || n_epochs == 0) return ULENS_OK;
    if (!theta_host || !t_host || !A_out_host) return ULENS_EINVAL;
    CK(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n = (size_t)n_cfg * n_epochs;
    // t, A, err, status (8-byte slots), dA, mask (bytes, rounded up to 8-byte slots)
    const size_t need = (size_t)n_epochs + n * (3 + (dA_out_host ? 7 : 0)) + (ext_mask_host ? (n + 7) / 8 : 0);
    if (need > ctx->io_cap) {
        cudaFree(ctx->io_buf); ctx->io_buf = nullptr; ctx->io_cap = 0;
        if (cudaMalloc(&ctx->io_buf, sizeof(double) * need) != cudaSuccess) return ULENS_ENOMEM;
        ctx->io_cap = need;
    }
    double* d_t = ctx->io_buf; double* d_A = d_t + n_epochs; double* d_err = d_A + n;
    unsigned* d_st = reinterpret_cast<unsigned*>(d_err + n);
    double* d_dA = dA_out_host ? d_err + 2 * n : nullptr;
    uint8_t* d_mask = ext_mask_host ? reinterpret_cast<uint8_t*>(d_err + 2 * n + (dA_out_host ? 7 * n : 0)) : nullptr;
    CK(cudaMemcpyAsync(d_t, t_host, sizeof(double) * n_epochs, cudaMemcpyHostToDevice, st));
    if (d_mask) CK(cudaMemcpyAsync(d_mask, ext_mask_host, n, cudaMemcpyHostToDevice, st));
    int rc = ulens_lightcurve_binary_ext(ctx, n_cfg, n_epochs, theta_host, u1, d_t, d_mask, sel_tol, d_A, d_dA, d_err, d_st,
                                         n_ext_out, stream);
    if (rc != ULENS_OK) return rc;
    CK(cudaMemcpyAsync(A_out_host, d_A, sizeof(double) * n, cudaMemcpyDeviceToHost, st));
    if (dA_out_host) CK(cudaMemcpyAsync(dA_out_host, d_dA, sizeof(double) * 7 * n, cudaMemcpyDeviceToHost, st));
    if (err_out_host) CK(cudaMemcpyAsync(err_out_host, d_err, sizeof(double) * n, cudaMemcpyDeviceToHost, st));
    if (status_out_host) CK(cudaMemcpyAsync(status_out_host, d_st, sizeof(unsigned) * n, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return ULENS_OK;
}

extern "C" int ulens_nll_marginal(ulens_ctx* ctx, int n_cfg, int n_epochs, const double* A, const double* dA,
                                  const double* flux, const double* sigma, double mu_fs, double mu_fb, double var_fs,
                                  double var_fb, double* nll_out, double* grad_out, void* stream)
{
    if (!ctx || n_cfg < 0 || n_epochs < 0) return ULENS_EINVAL;
    if (n_cfg == 0) return ULENS_OK;
    if (n_epochs == 0 || !A || !flux || !sigma || !nll_out || (grad_out && !dA)) return ULENS_EINVAL;
    if (!isfinite(mu_fs) || !isfinite(mu_fb) || !finite_pos(var_fs) || !finite_pos(var_fb)) return ULENS_EINVAL;
    CK(cudaSetDevice(ctx->device));
    k_nll<<<n_cfg, 256, 0, (cudaStream_t)stream>>>(n_epochs, A, dA, flux, sigma, mu_fs, mu_fb, var_fs, var_fb, nll_out, grad_out);
    ctx->last_launches = 1;
    CK(cudaGetLastError());
    return ULENS_OK;
}

extern "C" int ulens_mag_point(ulens_ctx* ctx, int n_cfg, int n_pts, const ulens_lens* lenses_host, const double* w_re,
                               const double* w_im, double* A_out, uint32_t* status_out, void* stream)
{
    if (!ctx || n_cfg < 0 || n_pts < 0) return ULENS_EINVAL;
    if (n_cfg == 0 || n_pts == 0) return ULENS_OK;
    if (!lenses_host || !w_re || !w_im || !A_out) return ULENS_EINVAL;
    CK(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    std::vector<double> rho(n_cfg, 1.0), u1(n_cfg, 0.0);       // unused by the point-source sum
    int N = 0; bool ld = false;
    int rc = upload_cfgs(ctx, n_cfg, lenses_host, rho.data(), u1.data(), st, &N, &ld);
    if (rc != ULENS_OK) return rc;
    long long n_total = (long long)n_cfg * n_pts;
    if (n_total > UL_MAX_POINTS) return ULENS_EUNSUPPORTED;
    const int n = (int)n_total, grid = (int)((n_total + 127) / 128);
    switch (N) {
        case 1: k_roots<1><<<grid, 128, 0, st>>>(n, 0, n_pts, ctx->cfg_dev, ctx->poly_dev, w_re, w_im, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, A_out, status_out); break;
        case 2: k_roots<2><<<grid, 128, 0, st>>>(n, 0, n_pts, ctx->cfg_dev, ctx->poly_dev, w_re, w_im, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, A_out, status_out); break;
        default: k_roots<3><<<grid, 128, 0, st>>>(n, 0, n_pts, ctx->cfg_dev, ctx->poly_dev, w_re, w_im, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, A_out, status_out); break;
    }
    ctx->last_launches = 1;
    CK(cudaGetLastError());
    return ULENS_OK;
}

extern "C" int ulens_roots(ulens_ctx* ctx, const ulens_lens* lens_host, int n_pts, const double* w_re, const double* w_im,
                           double* roots_re, double* roots_im, uint8_t* is_image, void* stream)
{
    if (!ctx || n_pts < 0) return ULENS_EINVAL;
    if (n_pts == 0) return ULENS_OK;
    if (!lens_host || !w_re || !w_im || !roots_re || !roots_im || !is_image) return ULENS_EINVAL;
    CK(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    int N = 0; bool ld = false;
    double rho = 1.0, u1 = 0.0;
    int rc = upload_cfgs(ctx, 1, lens_host, &rho, &u1, st, &N, &ld);
    if (rc != ULENS_OK) return rc;
    int grid = (n_pts + 127) / 128;
    switch (N) {
        case 1: k_roots<1><<<grid, 128, 0, st>>>(n_pts, 0, n_pts, ctx->cfg_dev, ctx->poly_dev, w_re, w_im, roots_re, roots_im, is_image, nullptr, nullptr, nullptr, nullptr); break;
        case 2: k_roots<2><<<grid, 128, 0, st>>>(n_pts, 0, n_pts, ctx->cfg_dev, ctx->poly_dev, w_re, w_im, roots_re, roots_im, is_image, nullptr, nullptr, nullptr, nullptr); break;
        default: k_roots<3><<<grid, 128, 0, st>>>(n_pts, 0, n_pts, ctx->cfg_dev, ctx->poly_dev, w_re, w_im, roots_re, roots_im, is_image, nullptr, nullptr, nullptr, nullptr); break;
    }
    ctx->last_launches = 1;
    CK(cudaGetLastError());
    return ULENS_OK;
}

extern "C" int ulens_get_stats(ulens_ctx* ctx, ulens_stats* out)
{
    if (!ctx || !out) return ULENS_EINVAL;
    CK(cudaSetDevice(ctx->device));
    CK(cudaDeviceSynchronize());
    DevCounters h;
    CK(cudaMemcpy(&h, ctx->counters, sizeof h, cudaMemcpyDeviceToHost));
    out->n_points = h.n_points; out->n_rays = h.n_rays; out->n_patches = h.n_patches; out->n_units = h.n_units;
    out->n_limb_solves = h.n_limb_solves; out->n_flagged = h.n_flagged;
    return ULENS_OK;
}

extern "C" int ulens_reset_stats(ulens_ctx* ctx)
{
    if (!ctx) return ULENS_EINVAL;
    CK(cudaSetDevice(ctx->device));
    CK(cudaDeviceSynchronize());
    CK(cudaMemset(ctx->counters, 0, sizeof(DevCounters)));
    return ULENS_OK;
}

// fold finished event pairs into the per-kernel totals (synchronises on each pair)
static int drain_timed(ulens_ctx* ctx)
{
    for (auto& t : *ctx->timed) {
        float ms = 0.f;
        CK(cudaEventSynchronize(t.b));
        CK(cudaEventElapsedTime(&ms, t.a, t.b));
        ctx->k_ms[t.which] += ms; ctx->k_launches[t.which] += 1;
        cudaEventDestroy(t.a); cudaEventDestroy(t.b);
    }
    ctx->timed->clear();
    return ULENS_OK;
}

extern "C" int ulens_set_timing(ulens_ctx* ctx, int on)
{
    if (!ctx) return ULENS_EINVAL;
    CK(cudaSetDevice(ctx->device));
    int rc = drain_timed(ctx);
    if (rc != ULENS_OK) return rc;
    ctx->timing_on = on ? 1 : 0;
    if (on) for (int k = 0; k < ULENS_K_COUNT; ++k) { ctx->k_ms[k] = 0.0; ctx->k_launches[k] = 0; }
    return ULENS_OK;
}

extern "C" int ulens_get_kernel_ms(ulens_ctx* ctx, int which, double* ms_total, int* launches)
{
    if (!ctx || which < 0 || which >= ULENS_K_COUNT || !ms_total) return ULENS_EINVAL;
    CK(cudaSetDevice(ctx->device));
    int rc = drain_timed(ctx);
    if (rc != ULENS_OK) return rc;
    *ms_total = ctx->k_ms[which];
    if (launches) *launches = ctx->k_launches[which];
    return ULENS_OK;
}

extern "C" int ulens_last_launch_count(ulens_ctx* ctx) { return ctx ? ctx->last_launches : ULENS_EINVAL; }

extern "C" int ulens_fp64_peak(ulens_ctx* ctx, double ms, double* dfma_per_s)
{
    if (!ctx || !dfma_per_s || !(ms > 0.0)) return ULENS_EINVAL;
    CK(cudaSetDevice(ctx->device));
    int sm_count = 148;
    cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, ctx->device);
    double* d = nullptr;
    CK(cudaMalloc(&d, sizeof(double)));
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    const int blocks = sm_count * 8, threads = 256;
    int iters = 2000;
    double best = 0.0;
    float el = 0.f;
    // calibrate then run ~ms
    for (int pass = 0; pass < 3; ++pass) {
        CK(cudaEventRecord(e0));
        k_dfma_peak<<<blocks, threads>>>(iters, d);
        CK(cudaEventRecord(e1));
        CK(cudaEventSynchronize(e1));
        CK(cudaEventElapsedTime(&el, e0, e1));
        double rate = (double)blocks * threads * 64.0 * iters / (el * 1e-3);
        if (pass > 0 && rate > best) best = rate;
        if (pass == 0) { double scale = ms / (el > 1e-3 ? el : 1e-3); iters = (int)(iters * scale); if (iters < 100) iters = 100; if (iters > 50000000) iters = 50000000; }
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
    *dfma_per_s = best;
    return ULENS_OK;
}

extern "C" int ulens_fp32_peak(ulens_ctx* ctx, double ms, double* ffma_per_s)
{
    if (!ctx || !ffma_per_s || !(ms > 0.0)) return ULENS_EINVAL;
    CK(cudaSetDevice(ctx->device));
    int sm_count = 148;
    cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, ctx->device);
    float* d = nullptr;
    CK(cudaMalloc(&d, sizeof(float)));
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    const int blocks = sm_count * 8, threads = 256;
    int iters = 2000;
    double best = 0.0;
    float el = 0.f;
    // calibrate then run ~ms
    for (int pass = 0; pass < 3; ++pass) {
        CK(cudaEventRecord(e0));
        k_ffma_peak<<<blocks, threads>>>(iters, d);
        CK(cudaEventRecord(e1));
        CK(cudaEventSynchronize(e1));
        CK(cudaEventElapsedTime(&el, e0, e1));
        double rate = (double)blocks * threads * 64.0 * iters / (el * 1e-3);
        if (pass > 0 && rate > best) best = rate;
        if (pass == 0) { double scale = ms / (el > 1e-3 ? el : 1e-3); iters = (int)(iters * scale); if (iters < 100) iters = 100; if (iters > 50000000) iters = 50000000; }
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
    *ffma_per_s = best;
    return ULENS_OK;
}

// ------------------------------------------------------------------------------------------------ no-allocation entry
//
// ulens_mag_static: the finite-source magnification (steps a2 - a7, as ulens_mag without the retry pass) for callers
// that cannot allocate device memory (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc). The whole
// per-chunk workspace -- configuration tables, roots of the source centres, box lists, sector descriptors, unit queue
// and its sums, counters -- lives in ONE file-scope device array of fixed size; no context is needed. Every GPU that
// loads the library holds the array (UL_STATIC_BYTES, about 6 MiB) until the process exits.
// In host code `g_static_scratch` is only a stand-in for the symbol: its DEVICE address comes from
// cudaGetSymbolAddress, once per device with that device current, and the kernels are given pointers carved from it.

#define UL_STATIC_MAX_DEV 64
constexpr size_t ul_align256(size_t x) { return (x + 255) & ~(size_t)255; }
constexpr size_t UL_STATIC_UNITS   = (size_t)ULENS_STATIC_MAX_POINTS * 1024;          // per-point unit cap x points
constexpr size_t UL_SO_CFG      = 0;
constexpr size_t UL_SO_POLY     = UL_SO_CFG      + ul_align256(sizeof(PointCfg) * ULENS_STATIC_MAX_POINTS);
constexpr size_t UL_SO_PATCHES  = UL_SO_POLY     + ul_align256(sizeof(LensPoly) * ULENS_STATIC_MAX_POINTS);
constexpr size_t UL_SO_NPATCH   = UL_SO_PATCHES  + ul_align256(sizeof(Patch) * UL_MAXP * ULENS_STATIC_MAX_POINTS);
constexpr size_t UL_SO_STATUS   = UL_SO_NPATCH   + ul_align256(sizeof(int) * ULENS_STATIC_MAX_POINTS);
constexpr size_t UL_SO_CZR      = UL_SO_STATUS   + ul_align256(sizeof(unsigned) * ULENS_STATIC_MAX_POINTS);
constexpr size_t UL_SO_CZI      = UL_SO_CZR      + ul_align256(sizeof(double) * 10 * ULENS_STATIC_MAX_POINTS);
constexpr size_t UL_SO_CMASK    = UL_SO_CZI      + ul_align256(sizeof(double) * 10 * ULENS_STATIC_MAX_POINTS);
constexpr size_t UL_SO_NBOXES   = UL_SO_CMASK    + ul_align256(sizeof(unsigned) * ULENS_STATIC_MAX_POINTS);
constexpr size_t UL_SO_BOXES    = UL_SO_NBOXES   + ul_align256(sizeof(int) * ULENS_STATIC_MAX_POINTS);
constexpr size_t UL_SO_UDESC    = UL_SO_BOXES    + ul_align256(sizeof(SubBox) * BoxCap<3>::value * ULENS_STATIC_MAX_POINTS);
constexpr size_t UL_SO_USUM     = UL_SO_UDESC    + ul_align256(sizeof(unsigned) * UL_STATIC_UNITS);
constexpr size_t UL_SO_UODD     = UL_SO_USUM     + ul_align256(sizeof(double) * UL_STATIC_UNITS);
constexpr size_t UL_SO_CC       = UL_SO_UODD     + ul_align256(sizeof(double) * UL_STATIC_UNITS);
constexpr size_t UL_SO_COUNTERS = UL_SO_CC       + ul_align256(sizeof(ChunkCounters));
constexpr size_t UL_SO_QUIET    = UL_SO_COUNTERS + ul_align256(sizeof(DevCounters));
constexpr size_t UL_SO_LIMBLIST = UL_SO_QUIET + ul_align256(ULENS_STATIC_MAX_POINTS);
constexpr size_t UL_SO_QDRHO    = UL_SO_LIMBLIST + ul_align256(sizeof(int) * ULENS_STATIC_MAX_POINTS);
constexpr size_t UL_STATIC_BYTES = UL_SO_QDRHO + ul_align256(sizeof(double) * ULENS_STATIC_MAX_POINTS);
static_assert(UL_STATIC_BYTES <= (size_t)8 << 20, "static scratch is meant to stay modest (<= 8 MiB)");

static __device__ __align__(256) unsigned char g_static_scratch[UL_STATIC_BYTES];

// one workspace descriptor per device, in static host storage (no heap either); device < 0: not set up yet
static ulens_ctx g_static_ctx[UL_STATIC_MAX_DEV];
static bool g_static_ready[UL_STATIC_MAX_DEV];
static PointCfg g_static_cfg_host[ULENS_STATIC_MAX_POINTS];
static LensPoly g_static_poly_host[ULENS_STATIC_MAX_POINTS];
static char g_static_err[256];

extern "C" const char* ulens_static_last_cuda_error(void) { return g_static_err; }
extern "C" int ulens_static_max_points(void) { return ULENS_STATIC_MAX_POINTS; }
extern "C" long long ulens_static_scratch_bytes(void) { return (long long)UL_STATIC_BYTES; }

static int static_setup(int dev)
{
    ulens_ctx* ctx = &g_static_ctx[dev];
    memset(ctx, 0, sizeof *ctx);
    ctx->device = dev;
    CK(cudaSetDevice(dev));
    unsigned char* base = nullptr;
    CK(cudaGetSymbolAddress((void**)&base, g_static_scratch));      // this device's copy of the array
    if (!base) return ULENS_ECUDA;
    ulens_options o; memset(&o, 0, sizeof o);                        // the defaults of ulens_create
    o.n_limb = 512; o.n_r = 96; o.n_theta = 48; o.rel_tol = 1e-4; o.chunk_pts = ULENS_STATIC_MAX_POINTS;
    o.flags = ULENS_OPT_NO_RETRY;
    ctx->opt = o;
    ctx->rp.n_limb = o.n_limb; ctx->rp.n_r = o.n_r; ctx->rp.n_theta = o.n_theta;
    ctx->rp.max_nr = 8192; ctx->rp.max_nth = 32768; ctx->rp.max_units_pt = 1024;
    ctx->chunk = ULENS_STATIC_MAX_POINTS;
    ctx->cap_units = UL_STATIC_UNITS;
    ctx->cfg_dev   = reinterpret_cast<PointCfg*>(base + UL_SO_CFG);
    ctx->poly_dev  = reinterpret_cast<LensPoly*>(base + UL_SO_POLY);
    ctx->cfg_cap   = ULENS_STATIC_MAX_POINTS;
    ctx->patches   = reinterpret_cast<Patch*>(base + UL_SO_PATCHES);
    ctx->n_patch   = reinterpret_cast<int*>(base + UL_SO_NPATCH);
    ctx->status_ws = reinterpret_cast<unsigned*>(base + UL_SO_STATUS);
    ctx->c_zr      = reinterpret_cast<double*>(base + UL_SO_CZR);
    ctx->c_zi      = reinterpret_cast<double*>(base + UL_SO_CZI);
    ctx->c_mask    = reinterpret_cast<unsigned*>(base + UL_SO_CMASK);
    ctx->n_boxes   = reinterpret_cast<int*>(base + UL_SO_NBOXES);
    ctx->boxes     = reinterpret_cast<SubBox*>(base + UL_SO_BOXES);
    ctx->boxes_cap = BoxCap<3>::value;                               // the widest box list: run_chunks never reallocates
    ctx->unit_desc = reinterpret_cast<unsigned*>(base + UL_SO_UDESC);
    ctx->unit_sum  = reinterpret_cast<double*>(base + UL_SO_USUM);
    ctx->unit_odd  = reinterpret_cast<double*>(base + UL_SO_UODD);
    ctx->cc        = reinterpret_cast<ChunkCounters*>(base + UL_SO_CC);
    ctx->counters  = reinterpret_cast<DevCounters*>(base + UL_SO_COUNTERS);
    ctx->quiet     = base + UL_SO_QUIET;
    ctx->limb_list = reinterpret_cast<int*>(base + UL_SO_LIMBLIST);
    ctx->quiet_drho = reinterpret_cast<double*>(base + UL_SO_QDRHO);
    g_static_ready[dev] = true;
    return ULENS_OK;
}

extern "C" int ulens_mag_static(int cuda_device, int n_cfg, int n_pts, const ulens_lens* lenses_host,
                                const double* rho_host, const double* u1_host, const double* w_re, const double* w_im,
                                double* A_out, double* err_out, uint32_t* status_out, void* stream)
{
    g_static_err[0] = 0;
    if (cuda_device < 0 || cuda_device >= UL_STATIC_MAX_DEV || n_cfg < 0 || n_pts < 0) return ULENS_EINVAL;
    if (n_cfg == 0 || n_pts == 0) return ULENS_OK;
    if (!lenses_host || !rho_host || !u1_host || !w_re || !w_im || !A_out) return ULENS_EINVAL;
    const long long n_total = (long long)n_cfg * n_pts;
    if (n_total > ULENS_STATIC_MAX_POINTS) return ULENS_ELIMIT;      // beyond the fixed scratch: use ulens_mag
    ulens_ctx* ctx = &g_static_ctx[cuda_device];
    int rc = ULENS_OK;
    if (!g_static_ready[cuda_device]) {
        int ndev = 0;
        if (cudaGetDeviceCount(&ndev) != cudaSuccess || cuda_device >= ndev) return ULENS_ECUDA;
        rc = static_setup(cuda_device);
    } else {
        cudaError_t e = cudaSetDevice(cuda_device);
        if (e != cudaSuccess) rc = fail_cuda(ctx, e, "cudaSetDevice");
    }
    if (rc != ULENS_OK) { memcpy(g_static_err, ctx->cuda_err, sizeof g_static_err); return rc; }
    cudaStream_t st = (cudaStream_t)stream;
    // configuration tables (the checks and the arithmetic of upload_cfgs), built in static host storage
    const int N = lenses_host[0].n_lens;
    if (N < 1 || N > 3) return ULENS_EINVAL;
    bool ld = false;
    for (int c = 0; c < n_cfg; ++c) {
        const ulens_lens& L = lenses_host[c];
        if (L.n_lens != N) return ULENS_EUNSUPPORTED;
        double tot = 0.0;
        for (int a = 0; a < N; ++a) {
            if (!isfinite(L.eps[a]) || !(L.eps[a] >= 0.0) || !isfinite(L.ax[a]) || !isfinite(L.ay[a])) return ULENS_EINVAL;
            tot += L.eps[a];
        }
        if (fabs(tot - 1.0) > 1e-9) return ULENS_EINVAL;
        if (!finite_pos(rho_host[c]) || !(u1_host[c] >= 0.0 && u1_host[c] <= 1.0)) return ULENS_EINVAL;
        PointCfg& P = g_static_cfg_host[c];
        memset(&P, 0, sizeof P);
        P.lens.n = N;
        for (int a = 0; a < N; ++a) { P.lens.eps[a] = L.eps[a]; P.lens.ax[a] = L.ax[a]; P.lens.ay[a] = L.ay[a]; }
        P.rho = rho_host[c]; P.u1 = u1_host[c];
        if (u1_host[c] > 0.0) ld = true;
        lens_poly_basis(L.n_lens, L.eps, L.ax, L.ay, &g_static_poly_host[c]);
    }
    // pageable source: the runtime stages the bytes before it returns, so the static host tables may be rewritten
    // by the next call; the copies are ordered on `st` ahead of the kernels
    rc = [&]() -> int {
        CK(cudaMemcpyAsync(ctx->cfg_dev, g_static_cfg_host, sizeof(PointCfg) * n_cfg, cudaMemcpyHostToDevice, st));
        CK(cudaMemcpyAsync(ctx->poly_dev, g_static_poly_host, sizeof(LensPoly) * n_cfg, cudaMemcpyHostToDevice, st));
        // the array keeps the previous call's contents: the statistics counters restart at zero (the chunk counters
        // and the per-point box counts are cleared by run_chunks itself; everything else is written before it is read)
        CK(cudaMemsetAsync(ctx->counters, 0, sizeof(DevCounters), st));
        ctx->last_launches = 0;
        switch (N) {
            case 1: return run_chunks<1>(ctx, n_total, n_pts, ld, w_re, w_im, A_out, err_out, status_out, st);
            case 2: return run_chunks<2>(ctx, n_total, n_pts, ld, w_re, w_im, A_out, err_out, status_out, st);
            default: return run_chunks<3>(ctx, n_total, n_pts, ld, w_re, w_im, A_out, err_out, status_out, st);
        }
    }();
    if (rc != ULENS_OK) memcpy(g_static_err, ctx->cuda_err, sizeof g_static_err);
    return rc;
}
