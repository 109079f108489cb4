/*
 * ulens.h -- C ABI of the B200-native image-centred ray-shooting (ICRS) hot path.
 *
 * What is computed (citations are to /root/reference/PAPER.md, "P:<line>"):
 *
 *   finite-source, limb-darkened magnification of an N-point-mass lens (N = 1, 2, 3)
 *
 *       A(w_c, rho, u1) = (1/F0) Int Int Theta(rho - |w(z) - w_c|) I(|w(z) - w_c| / rho) d^2 z   Eqs. 5-6
 *       w(z) = z - sum_i eps_i / conj(z - a_i),  sum_i eps_i = 1                                 Eq. 1,
 *       I(x) = 1 - u1 (1 - sqrt(1 - x^2)),       F0 = pi rho^2 (1 - u1/3)                         Eq. A6,
 *
 *   by the paper's method: Ehrlich-Aberth roots of the lens polynomial (Eq. 4, Eq. 7),
 *   image-limb points (Eq. 8) -> polar (r, theta) sectors -> fixed polar grid of
 *   rays per sector with cubic edge location along theta and a limb-singularity-aware ring quadrature
 *   (Sec. 3.3, App. A), summed over rings and sectors and normalised (Eq. A5).
 *
 * Conventions
 *   - every function returns int: 0 = ULENS_OK, negative = error (below); ulens_strerror() names it.
 *   - "device" pointers are CUDA device memory OWNED BY THE CALLER (e.g. torch tensors); the library
 *     never frees or keeps them beyond the work it enqueues. "host" pointers are ordinary memory, read
 *     (or written, for *_host entry points) before the call returns.
 *   - all device work is enqueued on the caller's stream (a cudaStream_t passed as void*, NULL = the
 *     legacy default stream) and the call does NOT synchronise, except the *_host entry points,
 *     ulens_lightcurve_binary_ext (once, to read N_ext), the stats/peak calls and ulens_destroy, which say so.
 *     Host tables (lenses, rho, u1, theta) are copied into context-owned pinned staging during the call and
 *     uploaded stream-ordered; an array identical to the previous call's is not rebuilt or uploaded again.
 *     (A call that has to GROW a workspace buffer frees the old one, which waits for the device: first calls only.)
 *   - one context = one device = one stream at a time (the context owns the workspace the kernels share).
 *   - lengths are in Einstein radii of the TOTAL lens mass; complex numbers are passed as
 *     separate re / im arrays (SoA); doubles are IEEE binary64.
 *   - per-point trouble (root iteration not converged, patch cap hit, resolution cap hit, image
 *     touching a patch border, ...) is reported in the optional status bitmask, not as an error code.
 *   - there is NO CPU fallback: every step runs in the CUDA kernels of this library.
 */
#ifndef ULENS_H
#define ULENS_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ULENS_OK            0
#define ULENS_EINVAL       -1   /* NULL where not allowed, non-finite or out-of-domain scalar, negative size */
#define ULENS_ECUDA        -2   /* a CUDA runtime call failed (ulens_last_cuda_error has the text) */
#define ULENS_ENOMEM       -3   /* workspace allocation failed */
#define ULENS_EUNSUPPORTED -4   /* valid request that this build does not implement */
#define ULENS_ELIMIT       -5   /* ulens_mag_static: more points than the fixed scratch holds (ULENS_STATIC_MAX_POINTS) */

/* per-point status bits (status_out) */
#define ULENS_ST_EA_NOCONV   0x0001u  /* an Ehrlich-Aberth solve hit its iteration cap (Eq. 7) */
#define ULENS_ST_IMG_PARITY  0x0002u  /* centre image count not congruent N+1 (mod 2) */
#define ULENS_ST_PATCH_CAP   0x0004u  /* more sectors than the cap: merged into one */
#define ULENS_ST_RES_CAP     0x0008u  /* a sector wanted more rings / rays than the cap allows */
#define ULENS_ST_CLIPPED     0x0010u  /* an inside ray sat on a sector border (margin too small) */
#define ULENS_ST_UNIT_OVF    0x0020u  /* work-queue refusal: point not integrated, A = NaN (cannot happen with the built-in
                                         per-point unit cap: the queue holds chunk_pts x that cap) */
#define ULENS_ST_ERR_HIGH    0x0040u  /* half-resolution self-check differs by more than rel_tol */
#define ULENS_ST_NO_IMAGE    0x0080u  /* no image-limb point found (A = NaN) */
#define ULENS_ST_NIMG_SHIFT  8        /* bits 8..11: number of images of the source centre */
#define ULENS_ST_RETRIED     0x2000u  /* the first result was doubtful (EA_NOCONV, PATCH_CAP, CLIPPED, ERR_HIGH or NO_IMAGE) and the retry pass
                                         with twice the limb samples gave a finite result that is no worse (fewer of those bits, or as many
                                         and a smaller self-error): this is the retry's result and status. A doubtful point without this
                                         bit kept its first result (retry not better, or beyond the two chunks the retry pass covers) */
#define ULENS_ST_POINT_SRC   0x1000u  /* ulens_lightcurve_binary_ext: the epoch took the point-source value (Eq. 2-3) */

typedef struct ulens_ctx ulens_ctx;

#define ULENS_OPT_NO_RETRY   0x1      /* ulens_options.flags: do not re-integrate doubtful points (see ULENS_ST_RETRIED) */
#define ULENS_OPT_F32_SHOOT  0x2      /* mixed-precision ray shooting: the rays of ulens_mag / ulens_lightcurve_* WITHOUT
                                         derivatives run on the FP32 pipe in segment-local coordinates (cancellation-free difference
                                         form of Eq. 1); segment constants, edge events and accumulation stay FP64. Same sectors, same
                                         rule, same 1e-4 bar; the forward-mode variant always runs in FP64 */
#define ULENS_OPT_NO_QUIET   0x4      /* do not use the quiet-point shortcut. By default a source point that a 9-probe point-source test
                                         finds far from every caustic (same image count at the centre and at 8 limb points, finite-source
                                         effect below 1e-4) and from every light lens (8 sqrt(eps) + 2 rho around its planetary caustic)
                                         has its limb followed with an eighth of the n_limb samples; a sector that holds one image of its
                                         centre ends at the TRUE extremes of that image (Newton on Eq. 1 along the limb) and is shot
                                         with 3/8 of the scan lines and 3/4 of the nodes per line: on a smooth near-ellipse with exact
                                         ends the rule is all but exact (<= 2.6e-5 from the full treatment over every point of BASELINE
                                         C1-C3, <= 3.3e-5 over 1.4 M random-lens points). Its dA/drho is the quadrupole term of the same
                                         probe. The images are still tracked, the rays still decide; never in the retry pass; a point's
                                         result does not depend on what it is batched with */

/* Tunables; a zeroed struct (or NULL) selects the defaults in brackets. */
typedef struct {
    int    n_limb;        /* source-limb samples per point, multiple of 32 (Eq. 8: ~500) [512]   */
    int    n_r;           /* scan lines per image half-extent across the lines (P:139 N_r)       [96]    */
    int    n_theta;       /* rays per image half-chord along a scan line (P:139 N_theta)         [48]    */
    double rel_tol;       /* self-check threshold for ULENS_ST_ERR_HIGH                          [1e-4]  */
    int    chunk_pts;     /* points processed per internal pass (workspace size)                 [65536] */
    int    flags;         /* ULENS_OPT_* bits                                                    [0]     */
} ulens_options;

/* Lens: n_lens in {1,2,3}; eps sums to 1; positions in Einstein radii of the total mass. */
typedef struct {
    int    n_lens;
    double eps[3];
    double ax[3];
    double ay[3];
} ulens_lens;

typedef struct {
    uint64_t n_points;     /* source points integrated since create / reset */
    uint64_t n_rays;       /* lens-map evaluations in the ray-shooting kernel */
    uint64_t n_patches;    /* sectors integrated */
    uint64_t n_units;      /* 32-ring work units integrated */
    uint64_t n_limb_solves;/* polynomial solves at limb points */
    uint64_t n_flagged;    /* points with any status bit 0x00ff set */
} ulens_stats;

int  ulens_create (ulens_ctx** out, int cuda_device, const ulens_options* opt);
void ulens_destroy(ulens_ctx* ctx);                       /* synchronises the device, frees the workspace */

/* Geometry (Fig. 3 caption P:203; readings G4/G5 in DESIGN.md).
 * binary: origin = barycentre of M1, M2; M1 (eps 1/(1+q)) at x = -s q/(1+q), M2 (eps q/(1+q)) at x = +s/(1+q).
 * triple: q3 = M3/M1, M3 at polar (r3, psi) from the MIDPOINT of M1-M2; eps = (1, q, q3)/(1+q+q3).
 * EINVAL unless s > 0, q > 0, q3 >= 0, r3 > 0, all finite. Host-only helpers. */
int  ulens_lens_binary(ulens_lens* out, double s, double q);
int  ulens_lens_triple(ulens_lens* out, double s, double q, double q3, double r3, double psi);

/* (i) Source positions in -> magnification out.
 * n_cfg lens/source configurations, n_pts source centres each, row-major [cfg][pt].
 *   lenses_host, rho_host, u1_host : host arrays of n_cfg entries, copied during the call
 *                                    (rho > 0, 0 <= u1 <= 1, else EINVAL).
 *   w_re, w_im   : device, n_cfg*n_pts doubles, source centres w_c.
 *   A_out        : device, n_cfg*n_pts doubles, magnification (Eq. 6 / A5).
 *   err_out      : device or NULL, n_cfg*n_pts doubles: |A - A(half radial resolution)| / A.
 *   status_out   : device or NULL, n_cfg*n_pts uint32 bitmasks (ULENS_ST_*).
 * n_cfg == 0 or n_pts == 0 is a successful no-op. */
int  ulens_mag(ulens_ctx* ctx, int n_cfg, int n_pts,
               const ulens_lens* lenses_host, const double* rho_host, const double* u1_host,
               const double* w_re, const double* w_im,
               double* A_out, double* err_out, uint32_t* status_out, void* stream);

/* (i') The same with forward-mode derivatives (Sec. 3.5) with respect to
 * the intrinsic inputs:
 *   n_lens = 1, 2: dA5_out device [n_cfg*n_pts][5] = dA/d(w_cx, w_cy, s, q, rho)   (s, q columns zero for n_lens = 1)
 *   n_lens = 3   : dA5_out device [n_cfg*n_pts][8] = dA/d(w_cx, w_cy, s, q, q3, r3, psi, rho)
 * The lens-parameter columns are defined in the geometry of ulens_lens_binary / ulens_lens_triple (the parameters are
 * recovered from the lens; any other geometry is EUNSUPPORTED).
 * The derivatives are those of the quadrature rule on a ray grid that moves with the image, with one
 * exception: on a quiet source point (see ULENS_OPT_NO_QUIET) the rho column is the quadrupole term of the finite-source
 * expansion, (<A_ps>_limb - A_ps(w_c)) (1 - 7 u1/15)/(1 - u1/3) / rho. Far from caustics dA/drho is the small difference of two
 * terms ~2A/rho and the rule's own value there is cancellation noise of size ~1e-4 A/rho (also with ULENS_OPT_NO_QUIET). */
int  ulens_mag_grad(ulens_ctx* ctx, int n_cfg, int n_pts,
               const ulens_lens* lenses_host, const double* rho_host, const double* u1_host,
               const double* w_re, const double* w_im,
               double* A_out, double* dA5_out, double* err_out, uint32_t* status_out, void* stream);

/* Same with HOST arrays for w_re, w_im, A_out, err_out, status_out: copies in, computes, copies out and
 * synchronises the stream before returning (the end-to-end entry point). */
int  ulens_mag_host(ulens_ctx* ctx, int n_cfg, int n_pts,
               const ulens_lens* lenses_host, const double* rho_host, const double* u1_host,
               const double* w_re_host, const double* w_im_host,
               double* A_out_host, double* err_out_host, uint32_t* status_out_host, void* stream);

/* Step a1 alone: trajectory parameters -> source centres (reading G3). theta_host [n_cfg][7] as below (only t0, u0,
 * tE, alpha are read), t device [n_epochs]; w_re_out, w_im_out device [n_cfg][n_epochs]:
 *   tau = (t - t0)/tE,  w_c = (tau cos a - u0 sin a) + i (tau sin a + u0 cos a).   EINVAL unless tE > 0 and all finite. */
int  ulens_trajectory(ulens_ctx* ctx, int n_cfg, int n_epochs, const double* theta_host, const double* t,
               double* w_re_out, double* w_im_out, void* stream);

/* (ii) Trajectory parameters in -> light curve out (binary lens, reading G3):
 *   theta_host [n_cfg][7] = (t0, u0, tE, s, q, rho, alpha), host; u1 shared; t device [n_epochs].
 *   tau = (t - t0)/tE,  w_c = (tau cos a - u0 sin a) + i (tau sin a + u0 cos a).
 *   A_out device [n_cfg][n_epochs]; dA_out device [n_cfg][n_epochs][7] or NULL (forward-mode
 *   derivatives dA/d(t0,u0,tE,s,q,rho,alpha), Sec. 3.5). */
int  ulens_lightcurve_binary(ulens_ctx* ctx, int n_cfg, int n_epochs,
               const double* theta_host, double u1, const double* t,
               double* A_out, double* dA_out, double* err_out, uint32_t* status_out, void* stream);

/* Same with HOST arrays for t, A_out, dA_out (may be NULL), err_out (may be NULL), status_out (may be NULL):
 * copies t in, computes, copies the results out and synchronises the stream before returning
 * (the end-to-end entry point of the light-curve / derivative path, BASELINE.json configs[4]). */
int  ulens_lightcurve_binary_host(ulens_ctx* ctx, int n_cfg, int n_epochs,
               const double* theta_host, double u1, const double* t_host,
               double* A_out_host, double* dA_out_host, double* err_out_host, uint32_t* status_out_host,
               void* stream);

/* (ii') The triple-lens light curve (the paper's gradient showcase Fig. 2, is this case):
 *   theta_host [n_cfg][10] = (t0, u0, tE, s, q, rho, alpha, q3, r3, psi), host; geometry of ulens_lens_triple; trajectory as above.
 *   A_out device [n_cfg][n_epochs]; dA_out device [n_cfg][n_epochs][10] or NULL: dA/d(theta) in the order of theta.
 * ulens_lightcurve_triple_host: HOST arrays for t and the outputs, copies and synchronises (as ulens_lightcurve_binary_host). */
int  ulens_lightcurve_triple(ulens_ctx* ctx, int n_cfg, int n_epochs,
               const double* theta_host, double u1, const double* t,
               double* A_out, double* dA_out, double* err_out, uint32_t* status_out, void* stream);
int  ulens_lightcurve_triple_host(ulens_ctx* ctx, int n_cfg, int n_epochs,
               const double* theta_host, double u1, const double* t_host,
               double* A_out_host, double* dA_out_host, double* err_out_host, uint32_t* status_out_host,
               void* stream);

/* Light-curve driver with the point-source / finite-source switch (Sec. 3.4 (iii): "For extended-source
 * treatment, only a preselected set of N_ext epochs (e.g., near caustics) are modeled").
 * Every epoch gets the point-source magnification of its source centre (Eq. 2-3; with dA_out its
 * derivatives by implicit differentiation of Eq. 1 at the images); the N_ext selected epochs are then
 * gathered and recomputed by the finite-source path (a2-a8) exactly as ulens_lightcurve_binary does, and
 * scattered back. Arguments as ulens_lightcurve_binary, plus:
 *   ext_mask  device uint8 [n_cfg][n_epochs], non-zero = finite-source epoch (the caller's preselection), or NULL:
 *             the library selects ([proposal]): A_ps at 8 points of the source limb; an epoch keeps
 *             the point-source value when all 8 have as many images as the centre and the quadrupole estimate
 *             |mean_8 - A_c|/2 plus the hexadecapole guard |mean_axes - mean_diagonals| is <= sel_tol * A_c.
 *   sel_tol   tolerance of that test (ignored with ext_mask; <= 0 selects the default 2e-5).
 *   n_ext_out host int*, may be NULL: N_ext, the number of epochs that took the finite-source path.
 * Point-source epochs carry ULENS_ST_POINT_SRC in status_out and 0 in err_out. The call synchronises the stream
 * once (N_ext sizes the finite-source launches); the results are stream-ordered as everywhere else. */
int  ulens_lightcurve_binary_ext(ulens_ctx* ctx, int n_cfg, int n_epochs,
               const double* theta_host, double u1, const double* t,
               const uint8_t* ext_mask, double sel_tol,
               double* A_out, double* dA_out, double* err_out, uint32_t* status_out,
               int* n_ext_out, void* stream);

/* Same with HOST arrays for t, ext_mask (may be NULL), A_out, dA_out (may be NULL), err_out (may be NULL),
 * status_out (may be NULL): copies in, computes, copies out and synchronises the stream before returning. */
int  ulens_lightcurve_binary_ext_host(ulens_ctx* ctx, int n_cfg, int n_epochs,
               const double* theta_host, double u1, const double* t_host,
               const uint8_t* ext_mask_host, double sel_tol,
               double* A_out_host, double* dA_out_host, double* err_out_host, uint32_t* status_out_host,
               int* n_ext_out, void* stream);

/* Marginalised-flux negative log-likelihood of n_cfg model light curves against ONE data set, and its gradient
 * (App. B.2, Eqs. B17-B23). Model (B20): F_i = (A_i - 1) F_S + F_base; the two linear flux
 * parameters carry Gaussian priors N(mu_fs, var_fs), N(mu_fb, var_fb) and are integrated out (B15); the noise is
 * independent Gaussian, C = diag(sigma_i^2). Per light curve c:
 *   NLL_c = 1/2 r^T B^-1 r + 1/2 ln|B|,  r = F - M mu,  B = C + M Lambda M^T,  M_i = (A_ci - 1, 1)        (B17, B21-B23)
 * evaluated through the 2x2 Woodbury forms B18-B19 (the constant n/2 ln 2 pi is left out, as in B17), and
 *   grad_c[k] = sum_i dNLL_c/dA_ci * dA_ci/dtheta_k   for the 7 parameters of dA (forward-mode output of a8).
 * A device [n_cfg][n_epochs]; dA device [n_cfg][n_epochs][7] (needed iff grad_out != NULL); flux, sigma device [n_epochs];
 * nll_out device [n_cfg]; grad_out device [n_cfg][7] or NULL. One CTA per light curve, sums in a fixed order
 * (deterministic). EINVAL: NULL where not allowed, n_epochs == 0 with n_cfg > 0, non-finite means, variances <= 0. */
int  ulens_nll_marginal(ulens_ctx* ctx, int n_cfg, int n_epochs, const double* A, const double* dA,
               const double* flux, const double* sigma, double mu_fs, double mu_fb, double var_fs, double var_fb,
               double* nll_out, double* grad_out, void* stream);

/* Point-source magnification (Eq. 2-3): A = sum over the images of 1/|det J|, det J = 1 - |sum_i eps_i/conj(z - a_i)^2|^2,
 * from the validated, polished images of step a2 (one thread per source position). Layout as ulens_mag
 * (lenses host, w_re/w_im device [n_cfg][n_pts], A_out device, status_out device or NULL: image count in
 * bits 8-11, ULENS_ST_EA_NOCONV / ULENS_ST_IMG_PARITY). On a caustic det J -> 0 and A diverges, as it must.
 * This is the building block of the point-source / finite-source switch for far epochs, SURVEY 8.f-2. */
int  ulens_mag_point(ulens_ctx* ctx, int n_cfg, int n_pts, const ulens_lens* lenses_host,
               const double* w_re, const double* w_im, double* A_out, uint32_t* status_out, void* stream);

/* (iii) Root export (Eq. 4, Eq. 7): all N^2+1 roots of the lens polynomial for
 * each source position and which of them are images (validated on Eq. 1; images are polished
 * on Eq. 1). roots_re/im device [n_pts][n_deg], is_image device [n_pts][n_deg] bytes, n_deg = N^2+1. */
int  ulens_roots(ulens_ctx* ctx, const ulens_lens* lens_host, int n_pts,
               const double* w_re, const double* w_im,
               double* roots_re, double* roots_im, uint8_t* is_image, void* stream);

/* Counters (synchronises the device). ulens_reset_stats zeroes them. */
int  ulens_get_stats(ulens_ctx* ctx, ulens_stats* out);
int  ulens_reset_stats(ulens_ctx* ctx);

/* Names of the kernels a call launches, for launch accounting: number of kernel launches the last
 * ulens_mag / ulens_lightcurve_binary / ulens_roots call on this context enqueued. */
int  ulens_last_launch_count(ulens_ctx* ctx);

/* Per-kernel device time (measurement): while timing is on, every kernel launch of the
 * pipeline is bracketed by a CUDA event pair recorded on the CALLER'S stream (no synchronisation, no
 * serialisation beyond stream order). ulens_get_kernel_ms synchronises those events and returns the
 * total device milliseconds and the launch count of kernel `which` accumulated since the last
 * ulens_set_timing(ctx, 1) call (which also clears the totals). */
#define ULENS_K_TRAJ     0   /* trajectory -> source centres            (step a1) */
#define ULENS_K_ROOTS    1   /* centre roots: polynomial, EA, polish    (step a2) */
#define ULENS_K_LIMB     2   /* limb images -> boxes of the image arcs  (step a3, first half of a4) */
#define ULENS_K_SHOOT    3   /* ray shooting + ring quadrature          (steps a5, a6; the forward-mode kernel for a8) */
#define ULENS_K_FINALIZE 4   /* per-point sum, normalisation            (step a7) */
#define ULENS_K_SECTORS  5   /* boxes -> sectors -> work units          (second half of a4) */
#define ULENS_K_COUNT    6
int  ulens_set_timing(ulens_ctx* ctx, int on);
int  ulens_get_kernel_ms(ulens_ctx* ctx, int which, double* ms_total, int* launches);

/* FP64 FMA roofline denominator: runs a dependent-chain-free DFMA kernel on every SM for about
 * `ms` milliseconds and returns the achieved rate in DFMA/s (one DFMA = 2 flop). Synchronises. */
int  ulens_fp64_peak(ulens_ctx* ctx, double ms, double* dfma_per_s);

/* The same for the FP32 pipe (FFMA/s): denominator of the mixed-precision variant's roofline. Synchronises. */
int  ulens_fp32_peak(ulens_ctx* ctx, double ms, double* ffma_per_s);

/* ---- no-allocation entry ----------------------------------------------------------------------------------------
 * For callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): ulens_mag WITHOUT a context and without any allocation. Same operation as ulens_mag on a context
 * with default options and ULENS_OPT_NO_RETRY (steps a2-a7 of the hot path: Eq. 1-3, 7-8, App. A of the paper; one pass,
 * no retry of doubtful points -- they keep their status bits), same argument meaning and layout:
 *   cuda_device        device ordinal (made current); lenses_host / rho_host / u1_host: HOST arrays [n_cfg]
 *   w_re, w_im         DEVICE [n_cfg][n_pts] source centres;  A_out DEVICE [n_cfg][n_pts]
 *   err_out, status_out DEVICE [n_cfg][n_pts] or NULL;        stream: cudaStream_t (NULL = default stream)
 * The whole workspace (tables, box lists, sector descriptors, unit queue, counters) is one file-scope device array of
 * ulens_static_scratch_bytes() bytes (about 6 MiB) that EVERY GPU touched by this library holds until the process exits;
 * it bounds the call to n_cfg * n_pts <= ULENS_STATIC_MAX_POINTS. A larger request returns ULENS_ELIMIT and does
 * nothing -- use ulens_mag. The entry calls no cudaMalloc / cudaFree / cudaHostAlloc and no allocating library routine;
 * it enqueues two small host-to-device copies (pageable source, staged by the runtime before the call returns), one
 * memset and the five kernels of the path on `stream`, and does not wait for them.
 * All calls (all threads, all streams) on one device SHARE the array, which keeps the last call's contents; what must
 * start at zero is cleared on `stream` by the call itself. Two calls that overlap on the GPU (different streams, or
 * different host threads) RACE on it: issue the calls of one device on one stream, or order them with events. Not
 * thread-safe on the host either (static tables). ulens_static_last_cuda_error() has the text after ULENS_ECUDA. */
#define ULENS_STATIC_MAX_POINTS 128
int  ulens_mag_static(int cuda_device, int n_cfg, int n_pts, const ulens_lens* lenses_host, const double* rho_host,
                      const double* u1_host, const double* w_re, const double* w_im, double* A_out, double* err_out,
                      uint32_t* status_out, void* stream);
int  ulens_static_max_points(void);
long long ulens_static_scratch_bytes(void);
const char* ulens_static_last_cuda_error(void);

const char* ulens_strerror(int code);
const char* ulens_last_cuda_error(ulens_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* ULENS_H */
