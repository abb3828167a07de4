/* few.h -- C ABI of libfew_b200: the interpolated harmonic-mode summation of FastEMRIWaveforms
 * (Katz, Chua, Speri, Warburton, Hughes, arXiv:2104.04582; cited below as PAPER.md:<line>) as hand-written
 * CUDA for NVIDIA B200 (sm_100a), FP64, one GPU per process.
 *
 * The hot path:
 *   S0  few_ylm_modes      per-source harmonic constants  -2Y_{l,+-m}(theta, phi)
 *   S1  few_spline_fit     batched not-a-knot cubic splines of A_lmn(t_k)
 *       few_spline_fit_dd  the same for the two phases, solved and stored in double-double (R13)
 *   S2  few_select_modes   power sort + cumulative sum + eps threshold per sparse step, union over steps
 *                                                                                        PAPER.md:167
 *   S3  few_sum_waveform   h_+ - i h_x = sum_kept A_lmn(t) Y_lm exp(-i(m Phi_phi + n Phi_r)), m<0 folded in by
 *                          A_{l,-m,-n} = (-1)^l conj(A_lmn)                              PAPER.md:155-159, Eq.(9), Eq.(10)
 *   few_waveform / few_waveform_host  chain S0->S2->S1->S3 in the paper's pipeline order
 *
 * Conventions
 *   - Every function returns an int status: FEW_OK (0) or a negative FEW_ERR_*.  No exception crosses the ABI.
 *     few_strerror(code) names a code; few_last_error() returns the calling thread's last detailed message.
 *   - Pointers are DEVICE pointers (on the context's device) unless the name or comment says "host".
 *   - Ownership: the caller owns every input, output and workspace buffer.  The library keeps only a few KB of
 *     state in few_ctx (plus, if few_waveform_host is used, its device arena).  Workspace sizes come from the *_workspace() queries; workspaces need 256-byte alignment.
 *   - All work is ordered on the caller's stream (`stream` is a cudaStream_t passed as void*; NULL = legacy
 *     default stream).  No device-pointer call synchronises; n_keep stays on the device so S2 -> S1 -> S3 chain
 *     without a host round trip.  Only few_waveform_host and few_device_status synchronise.
 *     few_waveform, few_waveform_kerr and few_waveform_ssb run the two spline fits on two internal streams of the
 *     context, forked from and joined back into the caller's stream with events (on every return path, failing or not).
 *   - Threading and devices: a few_ctx serves ONE host thread at a time (its internal streams, events, profiling pair and
 *     host arena are not locked); use one context per thread.  Device-pointer entry points expect the context's device to
 *     be the calling thread's current device; few_create and few_waveform_host switch to it themselves and restore the
 *     caller's current device before returning.
 *   - Shapes are validated on the host (FEW_ERR_INVALID_ARG, FEW_ERR_TOO_FEW_POINTS, FEW_ERR_LIMIT).  Data that
 *     lives on the device (t increasing, (l,m,n) validity) is checked by the kernels, which OR a FEW_DEV_* bit into a
 *     device status word read back by few_device_status().  Outputs are unspecified when a bit is set.
 *   - Layouts are C-contiguous with the LAST index fastest.  Complex numbers are (re, im) pairs of doubles.
 *   - n_samples, t0, dt are uniform across a batch; sources differ in t, amplitudes, phases, angles and kept modes.  n_t is
 *     uniform in the plain entry points (true for every benchmark workload of the paper); the *_ragged entry points take each
 *     source's own knot count in padded arrays (adaptive trajectories), see "Ragged batches" below.
 *   - There is no CPU fallback: without a CUDA device few_create fails with FEW_ERR_CUDA.
 */
#ifndef FEW_H
#define FEW_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FEW_VERSION 100 /* 0.1.0 */

enum {
    FEW_OK = 0,
    FEW_ERR_INVALID_ARG = -1,     /* NULL pointer, non-positive size, bad flag */
    FEW_ERR_TOO_FEW_POINTS = -2,  /* n_t < 4: a not-a-knot cubic spline needs 4 knots; ragged: n_t_src[s] outside [4, n_t] (few_device_status) */
    FEW_ERR_NOT_INCREASING = -3,  /* t not strictly increasing (reported by few_device_status) */
    FEW_ERR_BAD_MODE = -4,        /* l < 2, |m| > l, m < 0, |n| > FEW_MAX_ABS_N, |k| > FEW_MAX_ABS_K, l > FEW_MAX_L (few_device_status / few_ylm) */
    FEW_ERR_WORKSPACE = -5,       /* workspace NULL, misaligned or smaller than the query says */
    FEW_ERR_CUDA = -6,            /* a CUDA runtime call failed; few_last_error() has the text */
    FEW_ERR_LIMIT = -7            /* size beyond a documented limit (FEW_MAX_*) */
};

/* bits of the device status word */
enum { FEW_DEV_NOT_INCREASING = 1, FEW_DEV_BAD_MODE = 2, FEW_DEV_SPARSE_LIST = 4, FEW_DEV_BAD_COUNT = 8 };

#define FEW_MAX_L 16            /* l <= 16: the explicit Wigner-d sum in FP64 is accurate to 5e-15 for l <= 10 (the paper's range) and 1e-12 at l = 16 */
#define FEW_MAX_ABS_N 1023      /* |n| <= 1023: rho^n is stepped by a three-term recurrence whose error after b = |n| / 4 steps is <= b^2 ulp */
#define FEW_MAX_ABS_K 63        /* |k| <= 63 (polar index of Kerr-shaped mode lists, few_sum_waveform_kerr) */
#define FEW_MAX_NT_SPLINE 736   /* n_t limit of few_spline_fit (one shared-memory column per system) */
#define FEW_MAX_SELECT_MODES 131072 /* n_modes limit of few_select_modes (owner bitmap of a row in shared memory) */

typedef struct few_ctx few_ctx;

/* Context: binds a CUDA device, holds the device status word.  `device` = CUDA ordinal. */
int few_create(few_ctx** out, int device);
int few_destroy(few_ctx* ctx);
const char* few_strerror(int code);
const char* few_last_error(void);
int few_version(void);

/* Synchronises `stream`, returns FEW_OK or the FEW_ERR_* of the lowest FEW_DEV_* bit set by kernels since the last
 * call (FEW_DEV_BAD_COUNT first: a wrong knot count makes the kernels read padding, which sets other bits too), and clears the word.  Optional `bits_out` (host) receives the raw bits. */
int few_device_status(few_ctx* ctx, int* bits_out, void* stream);

/* ---- S0: spin-weighted spherical harmonics, s = -2 (Goldberg et al. convention, R11).
 * few_ylm is a HOST helper: out (host) = {Re, Im} of -2Y_lm(theta, phi).  FEW_ERR_BAD_MODE if l < 2, |m| > l, l > FEW_MAX_L.
 * few_ylm_modes: theta, phi [n_src]; l, m [n_modes] int32 (m >= 0) -> ylm_plus[n_src][n_modes][2] = -2Y_{l,m},
 * ylm_minus[n_src][n_modes][2] = -2Y_{l,-m}. */
int few_ylm(int l, int m, double theta, double phi, double* out_host);
int few_ylm_modes(few_ctx* ctx, const double* theta, const double* phi, const int* l, const int* m,
                  int n_src, int n_modes, double* ylm_plus, double* ylm_minus, void* stream);

/* ---- S1: batched not-a-knot cubic spline fit on a per-source shared grid.
 * t[n_src][n_t] strictly increasing; y[n_src][n_t][n_sys] (systems fastest: the amplitude module's [n_t, n_modes]
 * complex array viewed as doubles has n_sys = 2 n_modes).
 * coef[n_src][n_t-1][4][n_sys]: on segment k, S(t) = c0 + c1 dx + c2 dx^2 + c3 dx^3 with dx = t - t_k; c0 = y_k bitwise.
 * workspace: few_spline_fit_workspace(n_src, n_t) bytes; receives each source's factorised tridiagonal matrix (the matrix
 * depends on the grid only, so it is factored once per source, not once per system).
 * Limits: 4 <= n_t <= FEW_MAX_NT_SPLINE. */
size_t few_spline_fit_workspace(int n_src, int n_t);
int few_spline_fit(few_ctx* ctx, const double* t, const double* y, int n_src, int n_t, int n_sys,
                   double* coef, void* workspace, size_t workspace_bytes, void* stream);

/* Same spline, solved and stored in double-double (unevaluated sum hi + lo, |lo| <= ulp(hi)/2) for the orbital phases,
 * whose 1e5..1e6 rad magnitude needs more than 53 bits to reach 1e-10 on the waveform (R13).
 * y[n_src][n_t][n_sys] (FP64 knot values) -> coef_dd[n_src][n_t-1][4][n_sys][2] (hi, lo).  n_sys is small (2: Phi_phi, Phi_r). */
int few_spline_fit_dd(few_ctx* ctx, const double* t, const double* y, int n_src, int n_t, int n_sys,
                      double* coef_dd, void* stream);

/* ---- S2: Mode Selector.  Per source and sparse step k: entries = every mode j (power
 * |A_j(t_k)|^2 |Y+_j|^2) plus, for m_j > 0, its mirror (l,-m,-n) (power |A_j(t_k)|^2 |Y-_j|^2, owner j); sort by power
 * descending (ties: lower entry index first); inclusive cumulative sum C; entry of rank r is kept iff r == 0 or
 * C_{r-1} < (1 - eps) C_last.  Kept set = union over k of the owners.  eps <= 0 keeps every mode.
 * ylm_plus == NULL (then ylm_minus is ignored): power = |A|^2, no mirror entries.
 * amp[n_src][n_t][n_modes][2]; m[n_modes]; ylm_*[n_src][n_modes][2];
 * keep_idx[n_src][n_modes] int32 ascending, padded with -1; n_keep[n_src] int32.
 * Rows of any length up to n_modes <= FEW_MAX_SELECT_MODES (a Kerr-shaped 42 273-mode row has 78 507 entries). */
size_t few_select_modes_workspace(int n_src, int n_t, int n_modes);
int few_select_modes(few_ctx* ctx, const double* amp, const int* m, const double* ylm_plus, const double* ylm_minus,
                     double eps, int n_src, int n_t, int n_modes, int* keep_idx, int* n_keep,
                     void* workspace, size_t workspace_bytes, void* stream);

/* ---- S3: interpolated summation (Eq.(9), Eq.(10)).  For i in [0, n_samples): t_i = t0 + i*dt
 * (product and sum rounded separately); outside [t_0, t_{n_t-1}] h = 0; otherwise with k = max{k: t_k <= t_i} (clamped
 * to n_t-2), dx = t_i - t_k:
 *   h_i = scale * sum_{j kept} [ Y+_j W_j + (m_j > 0) (-1)^{l_j} Y-_j conj(W_j) ],  W_j = A_j(t_i) exp(-i(m_j Phi_phi + n_j Phi_r)).
 * coef_amp[n_src][n_t-1][4][2 n_modes] from few_spline_fit; coef_phase_dd[n_src][n_t-1][4][2][2] from few_spline_fit_dd
 * (system 0 = Phi_phi, 1 = Phi_r); l, m, n [n_modes] int32 shared by the sources, m >= 0;
 * keep_idx[n_src][n_modes] / n_keep[n_src] from few_select_modes, or both NULL = all modes;
 * scale[n_src] or NULL (= 1) is the mu/d_L prefactor of Eq.(10);
 * h[n_src][n_samples][2] = (h_+, -h_x). */
size_t few_sum_waveform_workspace(int n_src, int n_t, int n_modes, long long n_samples);
int few_sum_waveform(few_ctx* ctx, const double* t, const double* coef_amp, const double* coef_phase_dd,
                     const int* l, const int* m, const int* n, const int* keep_idx, const int* n_keep,
                     const double* ylm_plus, const double* ylm_minus, const double* scale,
                     double t0, double dt, long long n_samples, double* h,
                     int n_src, int n_t, int n_modes, void* workspace, size_t workspace_bytes, void* stream);

/* A caller's bound on the summation's STEPS per source, to shrink its workspace.  The summation consumes the kept modes as steps:
 * one step = the kept modes of one (m, k) whose |n| lie in one aligned block of four (4b .. 4b+3).  By default the workspace is laid
 * out for min(n_modes, n_modes / 4 + 64) steps per source, which no kept list of the call can exceed but which is far more than a
 * list on a grid needs: the paper's 3843-mode grid (m = 0..10, |n| <= 30) gives at most 11 x 8 = 88 steps where
 * the default reserves 1024 -- 105 MB of coefficient stages per source at n_t = 100 instead of 9 MB.
 *   few_max_steps_for_modes  HOST helper: the number of distinct (m, k, |n| >> 2) in a mode list (k_host may be NULL = 0), i.e. the
 *                            most steps ANY kept subset of that list can produce.  Returns the count (>= 1) or a negative FEW_ERR_*.
 *   few_set_max_steps        stores the bound in the context (0 = back to the default).  From then on every summation through this
 *                            context (few_sum_waveform*, few_waveform*) lays its workspace out for min(default, max_steps) steps per
 *                            source and expects at least few_*_workspace_ex(..., max_steps) bytes.  A kept list that needs more steps is
 *                            cut at the bound and reported: FEW_DEV_SPARSE_LIST -> few_device_status returns FEW_ERR_LIMIT.
 *   few_*_workspace_ex       the workspace queries for a given bound (max_steps = 0: the plain queries).
 * few_waveform_host(_ragged) has the mode list on the host and applies few_max_steps_for_modes itself for the duration of the call. */
int few_max_steps_for_modes(const int* m_host, const int* k_host, const int* n_host, int n_modes);
int few_set_max_steps(few_ctx* ctx, int max_steps);
size_t few_sum_waveform_workspace_ex(int n_src, int n_t, int n_modes, long long n_samples, int max_steps);
size_t few_waveform_workspace_ex(int n_src, int n_t, int n_modes, long long n_samples, int max_steps);

/* Extended form of S3.  Adds
 *   factor[n_src][2] or NULL: a complex per-source prefactor (few_frame_constants: the detector-frame transformation of
 *     Eq. (4)-(8) and mu/d_L).  h is linear in the harmonic constants, so the factor is folded into them before the sample
 *     loop and the transformation costs nothing per sample.  Multiplies with `scale` if both are given.
 *   d[n_src][n_samples][2] or NULL, inner[n_src][3] or NULL: with inner != NULL the kernel also reduces, per source, the
 *     PSD = 1 inner products of PAPER.md:283-296 Eq. (15)-(17) (Parseval, both polarisations, R23):
 *       inner[s][0] = <d|h> = 2 dt Re sum_i conj(d_i) h_i,  inner[s][1] = 2 dt Im sum_i conj(d_i) h_i,  inner[s][2] = <h|h>
 *     ([0], [1] are 0 when d == NULL).  h may then be NULL: nothing but three doubles per source is written, which is what a
 *     likelihood evaluation consumes (NEXT-2).  The reduction order is fixed: results are bit-reproducible.
 * Everything else as few_sum_waveform (same workspace query). */
int few_sum_waveform_ex(few_ctx* ctx, const double* t, const double* coef_amp, const double* coef_phase_dd,
                        const int* l, const int* m, const int* n, const int* keep_idx, const int* n_keep,
                        const double* ylm_plus, const double* ylm_minus, const double* scale, const double* factor,
                        double t0, double dt, long long n_samples, double* h, const double* d, double* inner,
                        int n_src, int n_t, int n_modes, void* workspace, size_t workspace_bytes, void* stream);

/* ---- NEXT-4: the summation for Kerr-shaped mode lists, Eq. (1) "Phi_mkn = m Phi_phi + k Phi_theta + n Phi_r",
 * PAPER.md:438-444 Eq. (19) (spheroidal harmonics projected on -2Y_lm, so the harmonic constants stay S0's), Eq. (9) in full:
 *   h_i = scale * factor * sum_{j kept} [ Y+_j W_j + (m_j > 0) (-1)^{l_j + k_j} Y-_j conj(W_j) ],
 *   W_j = A_j(t_i) exp(-i(m_j Phi_phi + k_j Phi_theta + n_j Phi_r)).
 * n_phase = 3: coef_phase_dd[n_src][n_t-1][4][3][2] from few_spline_fit_dd with n_sys = 3, systems (Phi_phi, Phi_theta, Phi_r);
 * k[n_modes] int32, |k| <= FEW_MAX_ABS_K, or NULL (= 0).  n_phase = 2, k = NULL is few_sum_waveform_ex exactly.
 * Kept lists longer than 16384 modes are ordered in the workspace instead of shared memory (same result).
 * All other arguments, the workspace query and the error behaviour as few_sum_waveform_ex. */
int few_sum_waveform_kerr(few_ctx* ctx, const double* t, const double* coef_amp, const double* coef_phase_dd, int n_phase,
                          const int* l, const int* m, const int* k, const int* n, const int* keep_idx, const int* n_keep,
                          const double* ylm_plus, const double* ylm_minus, const double* scale, const double* factor,
                          double t0, double dt, long long n_samples, double* h, const double* d, double* inner,
                          int n_src, int n_t, int n_modes, void* workspace, size_t workspace_bytes, void* stream);

/* ---- NEXT-1: detector (solar-system-barycentre) frame, sec. II A.
 * few_frame_constants: sky[n_src][4] = (theta_S, phi_S, theta_K, phi_K) (sky position, MBH spin direction; Eq. (4), (5));
 * mu_over_dl[n_src] or NULL (= 1) -> theta[n_src] with cos(theta) = -R.S and phi[n_src] = -pi/2, the viewing
 * angles the harmonics take, and factor[n_src][2] = -(mu/d_L) e^{2 i psi}, tan(psi) given by Eq. (8) (the minus sign is the
 * "phase shift of pi" of PAPER.md:98; readings: DESIGN.md R22).
 * few_frame_rotate: h_out[n_src][n_samples][2] = factor[src] * h_in (may alias): the transformation as a separate pass over an
 * existing source-frame waveform. */
int few_frame_constants(few_ctx* ctx, const double* sky, const double* mu_over_dl, int n_src,
                        double* theta, double* phi, double* factor, void* stream);
int few_frame_rotate(few_ctx* ctx, const double* h_in, const double* factor, int n_src, long long n_samples,
                     double* h_out, void* stream);

/* ---- NEXT-2: PSD = 1 inner products of two stored series: inner[n_src][3] as in few_sum_waveform_ex,
 * d, h [n_src][n_samples][2].  Two passes (per-chunk partials in the workspace, then a fixed-order sum): bit-reproducible. */
size_t few_inner_products_workspace(int n_src, long long n_samples);
int few_inner_products(few_ctx* ctx, const double* d, const double* h, int n_src, long long n_samples, double dt,
                       double* inner, void* workspace, size_t workspace_bytes, void* stream);

/* few_inner_products for callers that cannot allocate device memory.  few_inner_products wants a workspace, so somebody has to
 * call an allocator first.  Not every caller may: host code running where the CUDA runtime rejects allocation calls, a sampler
 * whose whole device-memory budget sits in a pool it must not grow, a plug-in that is handed device pointers by its host
 * application and has no allocator of its own.  This variant takes inputs and outputs only and keeps its per-chunk partial sums
 * in an array that is part of the library's device image.  It calls no cudaMalloc, cudaFree or allocating library routine.
 *   - Result: inner[n_src][3], bit-identical to few_inner_products on the same d, h, dt (same kernels, same reduction order).
 *   - Limit: n_src * ceil(n_samples / 2048) <= FEW_INNER_STATIC_MAX_CHUNKS (one source of up to 33 554 432 samples -- 10 years at
 *     10 s -- or e.g. 16 sources of 2 097 152); beyond it the call fails with FEW_ERR_LIMIT before touching the GPU, and
 *     few_last_error() says so.  The array costs FEW_INNER_STATIC_MAX_CHUNKS * 32 B = 512 KB of device memory on every GPU that
 *     loads the library, from load to process exit, whether this function is called or not.
 *   - ctx may be NULL (few_create allocates, so a caller that cannot allocate may have no context); if given it must belong to
 *     the current device and only counts the two launches.  d, h, inner and stream must belong to the calling thread's CURRENT
 *     device: the scratch array used is the current device's copy.
 *   - Set-up: the first call made on each device asks the CUDA runtime for the device address of the array (cudaGetSymbolAddress,
 *     return code checked, cached per device under a lock).  Make that first call outside any stream capture.
 *   - The array is shared by every call in the process and keeps the previous call's contents.  Nothing in it needs clearing:
 *     each call overwrites every slot it later reads.  For the same reason two calls whose kernels can overlap on one GPU
 *     (different streams, or different host threads) race on it and give garbage: keep calls on one device ordered, on one stream
 *     or with events.  Calls on different GPUs are independent.
 *   - n_samples = 0 zeroes inner (cudaMemsetAsync) as few_inner_products does.  Other errors as few_inner_products. */
#define FEW_INNER_STATIC_MAX_CHUNKS 16384
int few_inner_products_static(few_ctx* ctx, const double* d, const double* h, int n_src, long long n_samples, double dt,
                              double* inner, void* stream);

/* ---- NEXT-3: direct (non-interpolated) summation: amplitudes and phases given at every output sample.
 *   h_i = scale * factor * sum_j [ Y+_j W_ij + (m_j > 0) (-1)^{l_j} Y-_j conj(W_ij) ],  W_ij = A_ij exp(-i(m_j Phi_phi,i + n_j Phi_r,i)).
 * amp[n_src][n_samples][n_modes][2] (modes fastest: the amplitude module's layout); phase[n_src][n_samples][2] =
 * (Phi_phi, Phi_r) in FP64 (reduced mod 2 pi exactly, per sample); l, m, n [n_modes] int32, m >= 0, any order (the grid's
 * natural order -- n fastest -- is the fast case); ylm_*[n_src][n_modes][2]; scale[n_src] / factor[n_src][2] or NULL;
 * h[n_src][n_samples][2].  Every mode given is summed (select by passing fewer columns).  HBM-bound: 16 B per sample*mode. */
size_t few_sum_direct_workspace(int n_src, int n_modes);
int few_sum_direct(few_ctx* ctx, const double* amp, const double* phase, const int* l, const int* m, const int* n,
                   const double* ylm_plus, const double* ylm_minus, const double* scale, const double* factor,
                   long long n_samples, int n_src, int n_modes, double* h,
                   void* workspace, size_t workspace_bytes, void* stream);

/* ---- Whole path on device buffers: S0 -> S2 -> S1 -> S3, no host synchronisation.
 * t[n_src][n_t], phase[n_src][n_t][2] (Phi_phi, Phi_r), amp[n_src][n_t][n_modes][2], theta/phi[n_src], l/m/n[n_modes].
 * Outputs: h[n_src][n_samples][2]; optional keep_idx[n_src][n_modes], n_keep[n_src] (NULL: kept inside the workspace). */
size_t few_waveform_workspace(int n_src, int n_t, int n_modes, long long n_samples);
int few_waveform(few_ctx* ctx, const double* t, const double* phase, const double* amp,
                 const int* l, const int* m, const int* n, const double* theta, const double* phi, const double* scale,
                 double eps, double t0, double dt, long long n_samples, int n_src, int n_t, int n_modes,
                 double* h, int* keep_idx, int* n_keep, void* workspace, size_t workspace_bytes, void* stream);

/* Whole path for Kerr-shaped mode lists (NEXT-4): phase[n_src][n_t][3] = (Phi_phi, Phi_theta, Phi_r), k[n_modes] the polar
 * index; selection on rows of any length (streamed), three double-double phase fits, few_sum_waveform_kerr.  Everything else
 * as few_waveform, same workspace query. */
int few_waveform_kerr(few_ctx* ctx, const double* t, const double* phase, const double* amp,
                      const int* l, const int* m, const int* k, const int* n, const double* theta, const double* phi,
                      const double* scale, double eps, double t0, double dt, long long n_samples, int n_src, int n_t, int n_modes,
                      double* h, int* keep_idx, int* n_keep, void* workspace, size_t workspace_bytes, void* stream);

/* Whole path in the detector frame: few_frame_constants -> S0 -> S2 -> S1 -> S3 with the frame factor folded in, and
 * optionally the fused inner products against a resident data stream d (h may be NULL when inner is given).
 * sky[n_src][4], mu_over_dl[n_src] or NULL as in few_frame_constants; d, inner as in few_sum_waveform_ex.  Same workspace
 * query as few_waveform. */
int few_waveform_ssb(few_ctx* ctx, const double* t, const double* phase, const double* amp,
                     const int* l, const int* m, const int* n, const double* sky, const double* mu_over_dl,
                     double eps, double t0, double dt, long long n_samples, int n_src, int n_t, int n_modes,
                     double* h, const double* d, double* inner, int* keep_idx, int* n_keep,
                     void* workspace, size_t workspace_bytes, void* stream);

/* ---- Ragged batches: every source with its own number of sparse points.  The trajectory module steps adaptively ("~100"
 * points) and stops where the inspiral ends, so the sources of a batch of parameter draws differ in
 * length and end time.  All arrays keep the PADDED layouts documented above, with n_t = the largest count of the batch (the row
 * stride); n_t_src[n_src] int32 (device; host for few_waveform_host_ragged) is source s's count, 4 <= n_t_src[s] <= n_t -- a
 * count outside that range sets FEW_DEV_BAD_COUNT (few_device_status: FEW_ERR_TOO_FEW_POINTS), outputs then unspecified but
 * in bounds.  For source s only rows k < n_t_src[s] of t, y, amp, phase are read (the padding may hold anything, NaN included);
 * the fits write coefficient rows k < n_t_src[s] - 1 and leave the others untouched; selection takes the union over the steps
 * k < n_t_src[s]; the summation gives h = 0 after t[s][n_t_src[s] - 1], which is how sources end at different samples inside the
 * uniform n_samples.  n_t_src == NULL is the uniform call.  Workspace queries are the uniform ones with the padded n_t.
 * Otherwise each function is its namesake: few_spline_fit, few_spline_fit_dd, few_select_modes, few_sum_waveform_kerr (the most
 * general summation: n_phase = 2, k = NULL, factor = d = inner = NULL give few_sum_waveform), few_waveform, few_waveform_host. */
int few_spline_fit_ragged(few_ctx* ctx, const double* t, const double* y, const int* n_t_src, int n_src, int n_t, int n_sys,
                          double* coef, void* workspace, size_t workspace_bytes, void* stream);
int few_spline_fit_dd_ragged(few_ctx* ctx, const double* t, const double* y, const int* n_t_src, int n_src, int n_t, int n_sys,
                             double* coef_dd, void* stream);
int few_select_modes_ragged(few_ctx* ctx, const double* amp, const int* m, const double* ylm_plus, const double* ylm_minus,
                            const int* n_t_src, double eps, int n_src, int n_t, int n_modes, int* keep_idx, int* n_keep,
                            void* workspace, size_t workspace_bytes, void* stream);
int few_sum_waveform_ragged(few_ctx* ctx, const double* t, const int* n_t_src, const double* coef_amp, const double* coef_phase_dd,
                            int n_phase, const int* l, const int* m, const int* k, const int* n, const int* keep_idx,
                            const int* n_keep, const double* ylm_plus, const double* ylm_minus, const double* scale,
                            const double* factor, double t0, double dt, long long n_samples, double* h, const double* d,
                            double* inner, int n_src, int n_t, int n_modes, void* workspace, size_t workspace_bytes, void* stream);
int few_waveform_ragged(few_ctx* ctx, const double* t, const int* n_t_src, const double* phase, const double* amp,
                        const int* l, const int* m, const int* n, const double* theta, const double* phi, const double* scale,
                        double eps, double t0, double dt, long long n_samples, int n_src, int n_t, int n_modes,
                        double* h, int* keep_idx, int* n_keep, void* workspace, size_t workspace_bytes, void* stream);
int few_waveform_host_ragged(few_ctx* ctx, const double* t_host, const int* n_t_src_host, const double* phase_host,
                             const double* amp_host, const int* l_host, const int* m_host, const int* n_host,
                             const double* theta_host, const double* phi_host, const double* scale_host, double eps, double t0,
                             double dt, long long n_samples, int n_src, int n_t, int n_modes,
                             double* h_host, int* keep_idx_host, int* n_keep_host);

/* ---- Whole path on HOST buffers (same shapes, all pointers host; pinned memory recommended): copies inputs host->device
 * into a device arena the context keeps between calls (grow-only, released by few_destroy), runs few_waveform and delivers h
 * (and keep_idx/n_keep if not NULL) to the host, then synchronises.  If h_host is page-locked (cudaHostAlloc /
 * cudaHostRegister / torch pin_memory) the summation kernel stores into it directly, so the device->host transfer overlaps
 * the computation; pageable h_host is filled by a copy after the kernels.  Like every call, not re-entrant on one context.  `scale_host` may
 * be NULL.  Returns the device status as well. */
int few_waveform_host(few_ctx* ctx, const double* t_host, const double* phase_host, const double* amp_host,
                      const int* l_host, const int* m_host, const int* n_host, const double* theta_host,
                      const double* phi_host, const double* scale_host, double eps, double t0, double dt,
                      long long n_samples, int n_src, int n_t, int n_modes,
                      double* h_host, int* keep_idx_host, int* n_keep_host);

/* ==== The four entry points below are MEASUREMENT AIDS for bench.py, not part of the method: nothing on the hot path calls them. ==== */

/* ---- Measurement aid: register-resident DFMA chains on every SM (the FP64 roofline denominator).
 * Launches `blocks` x `threads` threads, each doing `iters` x 16 dependent-chain-free DFMAs; writes one double per thread
 * to sink[blocks*threads].  FLOPs = 2 * 16 * iters * blocks * threads. */
int few_fp64_peak_probe(few_ctx* ctx, int blocks, int threads, int iters, double* sink, void* stream);

/* ---- Measurement aid: with profiling on, few_sum_waveform (also inside few_waveform) brackets its hot kernel
 * (few_sum_kernel, the dominant launch of the path) with two CUDA events on the caller's stream.  few_profile_sum_ms
 * waits for the closing event of the most recent launch and writes its duration in milliseconds to ms_host.
 * FEW_ERR_INVALID_ARG if profiling is off or nothing was launched since it was switched on. */
int few_profile_enable(few_ctx* ctx, int on);
int few_profile_sum_ms(few_ctx* ctx, float* ms_host);

/* ---- Measurement aid: number of kernels this library has launched through `ctx` since few_create (every launch site
 * counts itself), written to count_host.  bench.py reports the difference over its timed region as `gpu_launches`. */
int few_launch_count(few_ctx* ctx, long long* count_host);

#ifdef __cplusplus
}
#endif
#endif /* FEW_H */
