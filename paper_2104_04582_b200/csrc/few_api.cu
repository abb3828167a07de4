// few_api.cu -- context, error reporting, the chained whole-path entry points and the FP64 peak probe.
#include <stdarg.h>
#include <string.h>
#include <new>
#include "few_common.cuh"

static thread_local char g_last_error[512] = "";

void few_set_error(const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_last_error, sizeof(g_last_error), fmt, ap);
    va_end(ap);
}

extern "C" const char* few_last_error(void) { return g_last_error; }
extern "C" int few_version(void) { return FEW_VERSION; }

extern "C" const char* few_strerror(int code)
{
    switch (code) {
        case FEW_OK: return "FEW_OK";
        case FEW_ERR_INVALID_ARG: return "FEW_ERR_INVALID_ARG: NULL pointer, non-positive size or bad flag";
        case FEW_ERR_TOO_FEW_POINTS: return "FEW_ERR_TOO_FEW_POINTS: a not-a-knot cubic spline needs n_t >= 4";
        case FEW_ERR_NOT_INCREASING: return "FEW_ERR_NOT_INCREASING: sparse times are not strictly increasing";
        case FEW_ERR_BAD_MODE: return "FEW_ERR_BAD_MODE: need 2 <= l <= FEW_MAX_L, 0 <= m <= l, |n| <= FEW_MAX_ABS_N";
        case FEW_ERR_WORKSPACE: return "FEW_ERR_WORKSPACE: workspace NULL, misaligned or too small";
        case FEW_ERR_CUDA: return "FEW_ERR_CUDA: CUDA runtime error";
        case FEW_ERR_LIMIT: return "FEW_ERR_LIMIT: size beyond a documented FEW_MAX_* limit";
        default: return "unknown FEW status code";
    }
}

extern "C" int few_create(few_ctx** out, int device)
{
    FEW_REQUIRE(out != nullptr, FEW_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    int count = 0;
    FEW_CUDA_CHECK(cudaGetDeviceCount(&count));
    FEW_REQUIRE(device >= 0 && device < count, FEW_ERR_INVALID_ARG, "no such CUDA device");
    int prev_device = 0;
    FEW_CUDA_CHECK(cudaGetDevice(&prev_device));
    FEW_CUDA_CHECK(cudaSetDevice(device));
    few_ctx* c = new (std::nothrow) few_ctx();          // value-initialised: every handle starts as NULL
    if (c == nullptr) { cudaSetDevice(prev_device); few_set_error("few_create: out of host memory"); return FEW_ERR_INVALID_ARG; }
    c->device = device;
    cudaError_t e = cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, device);
    if (e == cudaSuccess) e = cudaMalloc(&c->d_status, sizeof(int));
    if (e == cudaSuccess) e = cudaMemset(c->d_status, 0, sizeof(int));
    if (e == cudaSuccess) e = cudaEventCreate(&c->ev_sum[0]);
    if (e == cudaSuccess) e = cudaEventCreate(&c->ev_sum[1]);
    for (int i = 0; i < 2 && e == cudaSuccess; ++i) {
        e = cudaStreamCreateWithFlags(&c->side[i], cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_join[i], cudaEventDisableTiming);
    }
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming);
    if (e != cudaSuccess) {
        few_set_error("few_create: %s", cudaGetErrorString(e));
        few_destroy(c);                                 // releases whatever was created (the rest is NULL)
        cudaSetDevice(prev_device);
        return FEW_ERR_CUDA;
    }
    cudaSetDevice(prev_device);                         // the caller's current device is left as it was
    *out = c;
    return FEW_OK;
}

extern "C" int few_destroy(few_ctx* ctx)
{
    if (!ctx) return FEW_OK;
    cudaFree(ctx->d_status);
    if (ctx->ev_sum[0]) cudaEventDestroy(ctx->ev_sum[0]);
    if (ctx->ev_sum[1]) cudaEventDestroy(ctx->ev_sum[1]);
    for (int i = 0; i < 2; ++i) {
        if (ctx->side[i]) cudaStreamDestroy(ctx->side[i]);
        if (ctx->ev_join[i]) cudaEventDestroy(ctx->ev_join[i]);
    }
    if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
    if (ctx->host_stream) cudaStreamDestroy(ctx->host_stream);
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    for (int g = 0; g < kHostGroups; ++g) if (ctx->ev_group[g]) cudaEventDestroy(ctx->ev_group[g]);
    cudaFree(ctx->host_arena);
    if (ctx->host_stage) cudaFreeHost(ctx->host_stage);
    delete ctx;
    return FEW_OK;
}

extern "C" int few_profile_enable(few_ctx* ctx, int on)
{
    FEW_REQUIRE(ctx != nullptr, FEW_ERR_INVALID_ARG, "ctx is NULL");
    ctx->profile = on ? 1 : 0;
    ctx->profile_valid = 0;
    return FEW_OK;
}

extern "C" int few_profile_sum_ms(few_ctx* ctx, float* ms_host)
{
    FEW_REQUIRE(ctx && ms_host, FEW_ERR_INVALID_ARG, "NULL argument");
    FEW_REQUIRE(ctx->profile && ctx->profile_valid, FEW_ERR_INVALID_ARG, "profiling is off or no summation was launched");
    FEW_CUDA_CHECK(cudaEventSynchronize(ctx->ev_sum[1]));
    FEW_CUDA_CHECK(cudaEventElapsedTime(ms_host, ctx->ev_sum[0], ctx->ev_sum[1]));
    return FEW_OK;
}

extern "C" int few_launch_count(few_ctx* ctx, long long* count_host)
{
    FEW_REQUIRE(ctx && count_host, FEW_ERR_INVALID_ARG, "NULL argument");
    *count_host = ctx->launches;
    return FEW_OK;
}

extern "C" int few_device_status(few_ctx* ctx, int* bits_out, void* stream)
{
    FEW_REQUIRE(ctx != nullptr, FEW_ERR_INVALID_ARG, "ctx is NULL");
    int bits = 0;
    cudaStream_t st = (cudaStream_t)stream;
    FEW_CUDA_CHECK(cudaMemcpyAsync(&bits, ctx->d_status, sizeof(int), cudaMemcpyDeviceToHost, st));
    FEW_CUDA_CHECK(cudaMemsetAsync(ctx->d_status, 0, sizeof(int), st));
    FEW_CUDA_CHECK(cudaStreamSynchronize(st));
    if (bits_out) *bits_out = bits;
    if (bits & FEW_DEV_BAD_COUNT) { few_set_error("device check: a source's knot count n_t_src[s] is outside [4, n_t]"); return FEW_ERR_TOO_FEW_POINTS; }
    if (bits & FEW_DEV_NOT_INCREASING) { few_set_error("device check: sparse times not strictly increasing"); return FEW_ERR_NOT_INCREASING; }
    if (bits & FEW_DEV_BAD_MODE) { few_set_error("device check: invalid (l, m, n) or kept-mode index"); return FEW_ERR_BAD_MODE; }
    if (bits & FEW_DEV_SPARSE_LIST) { few_set_error("device check: kept-mode list too sparse in (m, k, |n|) for the summation's step capacity"); return FEW_ERR_LIMIT; }
    return FEW_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// Whole path: S0 -> S2 -> S1 -> S3 ("combined with the spin-weighted spherical harmonics and then put through
// mode selection ... Following mode selection, the waveform is built using the interpolated summation").
// ---------------------------------------------------------------------------------------------------------------
namespace {
struct wf_layout {
    double *ylm_plus, *ylm_minus, *coef_amp, *coef_phase;
    double *theta_src, *phi_src, *factor;      // few_waveform_ssb: source-frame viewing angles and the frame factor
    int *keep_idx, *n_keep;
    void *sel_ws, *sum_ws, *spl_ws;
    size_t sel_bytes, sum_bytes, spl_bytes;
};

wf_layout wf_carve(void* ws, int n_src, int n_t, int n_modes, long long n_samples, int max_steps, size_t* bytes)
{
    few_carver c(ws);
    wf_layout L;
    L.ylm_plus = c.take<double>((size_t)n_src * n_modes * 2);
    L.ylm_minus = c.take<double>((size_t)n_src * n_modes * 2);
    L.coef_amp = c.take<double>((size_t)n_src * (n_t - 1) * 4 * 2 * n_modes);
    L.coef_phase = c.take<double>((size_t)n_src * (n_t - 1) * 4 * 3 * 2);      // up to three phases (Kerr-shaped lists)
    L.keep_idx = c.take<int>((size_t)n_src * n_modes);
    L.n_keep = c.take<int>(n_src);
    L.theta_src = c.take<double>(n_src);
    L.phi_src = c.take<double>(n_src);
    L.factor = c.take<double>((size_t)n_src * 2);
    L.sel_bytes = few_select_modes_workspace(n_src, n_t, n_modes);
    L.sum_bytes = few_sum_waveform_workspace_ex(n_src, n_t, n_modes, n_samples, max_steps);
    L.spl_bytes = few_spline_fit_workspace(n_src, n_t);
    L.spl_ws = c.take<char>(L.spl_bytes);
    L.sel_ws = c.take<char>(L.sel_bytes);
    L.sum_ws = c.take<char>(L.sum_bytes);
    if (bytes) *bytes = c.off;
    return L;
}
}  // namespace

extern "C" size_t few_waveform_workspace_ex(int n_src, int n_t, int n_modes, long long n_samples, int max_steps)
{
    if (n_src <= 0 || n_t < 4 || n_modes <= 0) return 0;
    size_t bytes = 0;
    wf_carve(nullptr, n_src, n_t, n_modes, n_samples, max_steps, &bytes);
    return bytes;
}

extern "C" size_t few_waveform_workspace(int n_src, int n_t, int n_modes, long long n_samples)
{
    return few_waveform_workspace_ex(n_src, n_t, n_modes, n_samples, 0);
}

namespace {
// theta/phi: source-frame viewing angles, or (sky != NULL) computed from the detector-frame angles by few_frame_constants.
int waveform_impl(few_ctx* ctx, const double* t, const int* n_t_src, const double* phase, int n_phase, const double* amp, const int* l, const int* m,
                  const int* k, const int* n, const double* theta, const double* phi, const double* sky, const double* scale, double eps, double t0, double dt,
                  long long n_samples, int n_src, int n_t, int n_modes, double* h, const double* d, double* inner, int* keep_idx,
                  int* n_keep, void* workspace, size_t workspace_bytes, void* stream)
{
    FEW_REQUIRE(ctx && t && phase && amp && l && m && n && ((theta && phi) || sky), FEW_ERR_INVALID_ARG, "NULL argument");
    FEW_REQUIRE(n_src > 0 && n_modes > 0 && n_samples >= 0, FEW_ERR_INVALID_ARG, "sizes must be positive");
    FEW_REQUIRE(n_t >= 4, FEW_ERR_TOO_FEW_POINTS, "n_t < 4");
    FEW_REQUIRE(workspace && ((uintptr_t)workspace % 256) == 0 &&
                    workspace_bytes >= few_waveform_workspace_ex(n_src, n_t, n_modes, n_samples, ctx->max_steps),
                FEW_ERR_WORKSPACE, "workspace NULL, misaligned or too small");
    // every limit a sub-call checks is checked HERE, before anything is enqueued: once the side streams are forked, an early
    // return would leave them running into a workspace the caller is free to release
    FEW_REQUIRE(n_src <= 65535 && n_t <= 65535, FEW_ERR_LIMIT, "n_src or n_t > 65535");
    FEW_REQUIRE(n_t <= FEW_MAX_NT_SPLINE, FEW_ERR_LIMIT, "n_t > FEW_MAX_NT_SPLINE");
    FEW_REQUIRE(n_modes <= FEW_MAX_SELECT_MODES, FEW_ERR_LIMIT, "n_modes > FEW_MAX_SELECT_MODES");
    FEW_REQUIRE(dt > 0.0 && isfinite(dt) && isfinite(t0), FEW_ERR_INVALID_ARG, "dt must be positive and finite");
    FEW_REQUIRE(d == nullptr || inner != nullptr, FEW_ERR_INVALID_ARG, "d given but inner is NULL");
    if (n_samples > 0) {
        const int lim = few_sum_check_limits(ctx, n_src, n_t, n_modes, n_samples, n_phase);
        if (lim != FEW_OK) return lim;
    }
    wf_layout L = wf_carve(workspace, n_src, n_t, n_modes, n_samples, ctx->max_steps, nullptr);
    int* kidx = keep_idx ? keep_idx : L.keep_idx;
    int* nk = n_keep ? n_keep : L.n_keep;
    // The spline fits depend on the inputs only, so they run on two side streams beside harmonics + mode selection and
    // join before the summation (fork/join with events: nothing synchronises the host, and the pattern is graph-capturable).
    // A few_ctx serves ONE host thread at a time: the side streams and the fork/join events are the context's (few.h).
    cudaStream_t st = (cudaStream_t)stream;
    FEW_CUDA_CHECK(cudaEventRecord(ctx->ev_fork, st));
    FEW_CUDA_CHECK(cudaStreamWaitEvent(ctx->side[0], ctx->ev_fork, 0));
    FEW_CUDA_CHECK(cudaStreamWaitEvent(ctx->side[1], ctx->ev_fork, 0));
    // from here on every path, failing or not, joins the side streams back into the caller's stream before returning
    int rc = few_spline_fit_ragged(ctx, t, amp, n_t_src, n_src, n_t, 2 * n_modes, L.coef_amp, L.spl_ws, L.spl_bytes, ctx->side[0]);
    if (rc == FEW_OK) rc = few_spline_fit_dd_ragged(ctx, t, phase, n_t_src, n_src, n_t, n_phase, L.coef_phase, ctx->side[1]);
    const double* factor = nullptr;
    if (rc == FEW_OK && sky) {      // Eq. (4)-(8): viewing angles for the harmonics, one complex constant per source for the summation
        rc = few_frame_constants(ctx, sky, scale, n_src, L.theta_src, L.phi_src, L.factor, stream);
        theta = L.theta_src; phi = L.phi_src; factor = L.factor; scale = nullptr;
    }
    if (rc == FEW_OK) rc = few_ylm_modes(ctx, theta, phi, l, m, n_src, n_modes, L.ylm_plus, L.ylm_minus, stream);
    if (rc == FEW_OK) rc = few_select_modes_ragged(ctx, amp, m, L.ylm_plus, L.ylm_minus, n_t_src, eps, n_src, n_t, n_modes, kidx, nk, L.sel_ws, L.sel_bytes, stream);
    cudaError_t je = cudaEventRecord(ctx->ev_join[0], ctx->side[0]);
    if (je == cudaSuccess) je = cudaEventRecord(ctx->ev_join[1], ctx->side[1]);
    if (je == cudaSuccess) je = cudaStreamWaitEvent(st, ctx->ev_join[0], 0);
    if (je == cudaSuccess) je = cudaStreamWaitEvent(st, ctx->ev_join[1], 0);
    if (rc != FEW_OK) return rc;
    if (je != cudaSuccess) { few_set_error("few_waveform: joining the spline-fit streams failed: %s", cudaGetErrorString(je)); return FEW_ERR_CUDA; }
    return few_sum_waveform_ragged(ctx, t, n_t_src, L.coef_amp, L.coef_phase, n_phase, l, m, k, n, kidx, nk, L.ylm_plus, L.ylm_minus, scale,
                                   factor, t0, dt, n_samples, h, d, inner, n_src, n_t, n_modes, L.sum_ws, L.sum_bytes, stream);
}
}  // namespace

extern "C" int few_waveform(few_ctx* ctx, const double* t, const double* phase, const double* amp,
                            const int* l, const int* m, const int* n, const double* theta, const double* phi, const double* scale,
                            double eps, double t0, double dt, long long n_samples, int n_src, int n_t, int n_modes,
                            double* h, int* keep_idx, int* n_keep, void* workspace, size_t workspace_bytes, void* stream)
{
    FEW_REQUIRE(theta && phi, FEW_ERR_INVALID_ARG, "theta or phi is NULL");
    FEW_REQUIRE(n_samples == 0 || h, FEW_ERR_INVALID_ARG, "h is NULL");
    return waveform_impl(ctx, t, nullptr, phase, 2, amp, l, m, nullptr, n, theta, phi, nullptr, scale, eps, t0, dt, n_samples, n_src, n_t, n_modes, h,
                         nullptr, nullptr, keep_idx, n_keep, workspace, workspace_bytes, stream);
}

extern "C" int few_waveform_ragged(few_ctx* ctx, const double* t, const int* n_t_src, const double* phase, const double* amp,
                                   const int* l, const int* m, const int* n, const double* theta, const double* phi, const double* scale,
                                   double eps, double t0, double dt, long long n_samples, int n_src, int n_t, int n_modes,
                                   double* h, int* keep_idx, int* n_keep, void* workspace, size_t workspace_bytes, void* stream)
{
    FEW_REQUIRE(theta && phi, FEW_ERR_INVALID_ARG, "theta or phi is NULL");
    FEW_REQUIRE(n_samples == 0 || h, FEW_ERR_INVALID_ARG, "h is NULL");
    return waveform_impl(ctx, t, n_t_src, phase, 2, amp, l, m, nullptr, n, theta, phi, nullptr, scale, eps, t0, dt, n_samples, n_src, n_t, n_modes,
                         h, nullptr, nullptr, keep_idx, n_keep, workspace, workspace_bytes, stream);
}

extern "C" int few_waveform_kerr(few_ctx* ctx, const double* t, const double* phase, const double* amp,
                                 const int* l, const int* m, const int* k, const int* n, const double* theta, const double* phi,
                                 const double* scale, double eps, double t0, double dt, long long n_samples, int n_src, int n_t,
                                 int n_modes, double* h, int* keep_idx, int* n_keep, void* workspace, size_t workspace_bytes, void* stream)
{
    FEW_REQUIRE(theta && phi && k, FEW_ERR_INVALID_ARG, "theta, phi or k is NULL");
    FEW_REQUIRE(n_samples == 0 || h, FEW_ERR_INVALID_ARG, "h is NULL");
    return waveform_impl(ctx, t, nullptr, phase, 3, amp, l, m, k, n, theta, phi, nullptr, scale, eps, t0, dt, n_samples, n_src, n_t, n_modes, h,
                         nullptr, nullptr, keep_idx, n_keep, workspace, workspace_bytes, stream);
}

extern "C" int few_waveform_ssb(few_ctx* ctx, const double* t, const double* phase, const double* amp,
                                const int* l, const int* m, const int* n, const double* sky, const double* mu_over_dl,
                                double eps, double t0, double dt, long long n_samples, int n_src, int n_t, int n_modes,
                                double* h, const double* d, double* inner, int* keep_idx, int* n_keep,
                                void* workspace, size_t workspace_bytes, void* stream)
{
    FEW_REQUIRE(sky != nullptr, FEW_ERR_INVALID_ARG, "sky is NULL");
    FEW_REQUIRE(n_samples == 0 || h || inner, FEW_ERR_INVALID_ARG, "h and inner are both NULL");
    return waveform_impl(ctx, t, nullptr, phase, 2, amp, l, m, nullptr, n, nullptr, nullptr, sky, mu_over_dl, eps, t0, dt, n_samples, n_src, n_t, n_modes,
                         h, d, inner, keep_idx, n_keep, workspace, workspace_bytes, stream);
}

extern "C" int few_waveform_host_ragged(few_ctx* ctx, const double* t_host, const int* n_t_src_host, const double* phase_host,
                                        const double* amp_host, const int* l_host, const int* m_host, const int* n_host,
                                        const double* theta_host, const double* phi_host, const double* scale_host, double eps, double t0,
                                        double dt, long long n_samples, int n_src, int n_t, int n_modes,
                                        double* h_host, int* keep_idx_host, int* n_keep_host)
{
    FEW_REQUIRE(ctx && t_host && phase_host && amp_host && l_host && m_host && n_host && theta_host && phi_host,
                FEW_ERR_INVALID_ARG, "NULL argument");
    FEW_REQUIRE(n_src > 0 && n_modes > 0 && n_samples >= 0, FEW_ERR_INVALID_ARG, "sizes must be positive");
    FEW_REQUIRE(n_t >= 4, FEW_ERR_TOO_FEW_POINTS, "n_t < 4");
    FEW_REQUIRE(n_samples == 0 || h_host, FEW_ERR_INVALID_ARG, "h_host is NULL");
    // Everything that can be refused from the arguments alone is refused here, before a copy is enqueued: a host->device copy
    // still in flight when the call returns would read buffers the caller is free to release.
    FEW_REQUIRE(dt > 0.0 && isfinite(dt) && isfinite(t0), FEW_ERR_INVALID_ARG, "dt must be positive and finite");
    FEW_REQUIRE(n_t <= FEW_MAX_NT_SPLINE, FEW_ERR_LIMIT, "n_t > FEW_MAX_NT_SPLINE");
    FEW_REQUIRE(n_modes <= FEW_MAX_SELECT_MODES, FEW_ERR_LIMIT, "n_modes > FEW_MAX_SELECT_MODES");
    if (n_t_src_host)      // the counts are on the host: validated here (device-pointer calls report them through few_device_status)
        for (int s = 0; s < n_src; ++s)
            FEW_REQUIRE(n_t_src_host[s] >= 4 && n_t_src_host[s] <= n_t, FEW_ERR_TOO_FEW_POINTS, "a source's knot count n_t_src_host[s] is outside [4, n_t]");
    {
        const int per_call = n_src < kHostGroups ? 1 : (n_src + kHostGroups - 1) / kHostGroups;       // sources per few_waveform call below
        FEW_REQUIRE(per_call <= 65535, FEW_ERR_LIMIT, "n_src > 8 * 65535");
        if (n_samples > 0) {
            const int lim = few_sum_check_limits(ctx, per_call, n_t, n_modes, n_samples, 2);
            if (lim != FEW_OK) return lim;
        }
    }
    struct device_guard {           // the context's device is current inside the call; the caller's is restored on every return
        int prev = -1;
        ~device_guard() { if (prev >= 0) cudaSetDevice(prev); }
    } guard;
    FEW_CUDA_CHECK(cudaGetDevice(&guard.prev));
    FEW_CUDA_CHECK(cudaSetDevice(ctx->device));
    const size_t b_t = (size_t)n_src * n_t * 8, b_ph = b_t * 2, b_amp = (size_t)n_src * n_t * n_modes * 16;
    const size_t b_lmn = (size_t)n_modes * 4, b_ang = (size_t)n_src * 8, b_h = (size_t)n_src * n_samples * 16;
    const size_t b_keep = (size_t)n_src * n_modes * 4, b_nk = (size_t)n_src * 4;
    const int group_max = (n_src + kHostGroups - 1) / kHostGroups > 1 ? (n_src + kHostGroups - 1) / kHostGroups : 1;
    // The mode list is on the host here, so the summation's workspace is sized for the steps this list can produce at most (the
    // distinct (m, |n| >> 2): 88 on the paper's grid) instead of the default capacity (1024 there): 12 x less device memory per
    // source.  A bound the caller set with few_set_max_steps is kept if it is lower; the context's setting is restored on return.
    struct cap_guard {
        few_ctx* c; int saved;
        ~cap_guard() { c->max_steps = saved; }
    } cap{ctx, ctx->max_steps};
    {
        const int bound = few_max_steps_for_modes(m_host, nullptr, n_host, n_modes);
        if (bound > 0 && (ctx->max_steps == 0 || bound < ctx->max_steps)) ctx->max_steps = bound;
    }
    const size_t ws_bytes = few_waveform_workspace_ex(n_src < kHostGroups ? 1 : group_max, n_t, n_modes, n_samples, ctx->max_steps);
    // If h_host is pinned (page-locked, hence device-accessible under unified addressing) the summation kernel stores the
    // waveform straight into it: the device->host transfer then rides on the kernel's own coalesced streaming stores and
    // overlaps the FP64 work, instead of following it as a separate copy.  Pageable memory takes the staged path.
    double* h_mapped = nullptr;
    if (n_samples) {
        cudaPointerAttributes attr;
        if (cudaPointerGetAttributes(&attr, h_host) == cudaSuccess && attr.type == cudaMemoryTypeHost && attr.devicePointer)
            h_mapped = static_cast<double*>(attr.devicePointer);
        else
            (void)cudaGetLastError();
    }
    const size_t b_h_dev = h_mapped ? 0 : b_h;
    // one device allocation, carved: the small inputs first and contiguous (they travel as one block), then amp, h, outputs
    size_t total = 0;
    few_carver sz(nullptr);
    sz.take<char>(b_lmn); sz.take<char>(b_lmn); sz.take<char>(b_lmn); sz.take<char>(b_t); sz.take<char>(b_ph);
    sz.take<char>(b_ang); sz.take<char>(b_ang); sz.take<char>(b_ang); sz.take<char>(b_nk);
    const size_t small_bytes = sz.off;
    sz.take<char>(b_amp); sz.take<char>(b_h_dev); sz.take<char>(b_keep); sz.take<char>(b_nk);
    sz.take<char>(ws_bytes);
    total = sz.off;
    // device arena and stream are kept in the context between calls (grow-only), so a steady-state call allocates nothing
    if (total > ctx->host_arena_bytes) {
        if (ctx->host_arena) { FEW_CUDA_CHECK(cudaFree(ctx->host_arena)); ctx->host_arena = nullptr; ctx->host_arena_bytes = 0; }
        FEW_CUDA_CHECK(cudaMalloc(&ctx->host_arena, total));
        ctx->host_arena_bytes = total;
    }
    if (small_bytes > ctx->host_stage_bytes) {
        if (ctx->host_stage) { FEW_CUDA_CHECK(cudaFreeHost(ctx->host_stage)); ctx->host_stage = nullptr; ctx->host_stage_bytes = 0; }
        FEW_CUDA_CHECK(cudaHostAlloc(&ctx->host_stage, small_bytes, cudaHostAllocDefault));
        ctx->host_stage_bytes = small_bytes;
    }
    if (!ctx->host_stream) {
        FEW_CUDA_CHECK(cudaStreamCreateWithFlags(&ctx->host_stream, cudaStreamNonBlocking));
        FEW_CUDA_CHECK(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
        for (int g = 0; g < kHostGroups; ++g) FEW_CUDA_CHECK(cudaEventCreateWithFlags(&ctx->ev_group[g], cudaEventDisableTiming));
    }
    void* dev = ctx->host_arena;
    cudaStream_t st = ctx->host_stream;
    int rc = FEW_OK;
    cudaError_t e = cudaSuccess;
    few_carver c(dev);
    int* d_l = (int*)c.take<char>(b_lmn); int* d_m = (int*)c.take<char>(b_lmn); int* d_n = (int*)c.take<char>(b_lmn);
    double* d_t = (double*)c.take<char>(b_t); double* d_ph = (double*)c.take<char>(b_ph);
    double* d_th = (double*)c.take<char>(b_ang); double* d_phi = (double*)c.take<char>(b_ang); double* d_sc = (double*)c.take<char>(b_ang);
    int* d_nts = (int*)c.take<char>(b_nk);      // per-source knot counts of a ragged batch
    double* d_amp = (double*)c.take<char>(b_amp);
    double* d_h = (double*)c.take<char>(b_h_dev); int* d_keep = (int*)c.take<char>(b_keep); int* d_nk = (int*)c.take<char>(b_nk);
    void* d_ws = c.take<char>(ws_bytes);
    // The small inputs (mode indices, sparse times, phases, angles: tens of KB) are gathered into a pinned staging block
    // with the arena's own layout and go up as ONE copy; the amplitudes follow source group by source group.
    // Sources are independent, so a batch is cut into up to kHostGroups groups: group g's kernels start as soon as ITS
    // amplitudes have landed, i.e. while later groups are still in flight over PCIe.  (One source: one group.)
    {
        char* hs = static_cast<char*>(ctx->host_stage);
        few_carver hc(hs);
        memcpy(hc.take<char>(b_lmn), l_host, b_lmn); memcpy(hc.take<char>(b_lmn), m_host, b_lmn); memcpy(hc.take<char>(b_lmn), n_host, b_lmn);
        memcpy(hc.take<char>(b_t), t_host, b_t); memcpy(hc.take<char>(b_ph), phase_host, b_ph);
        memcpy(hc.take<char>(b_ang), theta_host, b_ang); memcpy(hc.take<char>(b_ang), phi_host, b_ang);
        char* sc = hc.take<char>(b_ang);
        if (scale_host) memcpy(sc, scale_host, b_ang);
        char* nts = hc.take<char>(b_nk);
        if (n_t_src_host) memcpy(nts, n_t_src_host, b_nk);
    }
    const int n_groups = n_src < kHostGroups ? n_src : kHostGroups;
    cudaStream_t cs = ctx->copy_stream;
    // the staging block is reused by the next call: that call's memcpy must not overtake this copy, which the final
    // synchronisation of this call guarantees
    e = cudaMemcpyAsync(dev, ctx->host_stage, small_bytes, cudaMemcpyHostToDevice, cs);
    for (int g = 0; g < n_groups && e == cudaSuccess; ++g) {
        const size_t s0 = (size_t)n_src * g / n_groups, s1 = (size_t)n_src * (g + 1) / n_groups, ns = s1 - s0;
        e = cudaMemcpyAsync(d_amp + s0 * n_t * n_modes * 2, amp_host + s0 * n_t * n_modes * 2, ns * n_t * n_modes * 16,
                            cudaMemcpyHostToDevice, cs);
        if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_group[g], cs);
    }
    double* h_out = h_mapped ? h_mapped : d_h;
    for (int g = 0; g < n_groups && e == cudaSuccess && rc == FEW_OK; ++g) {
        const size_t s0 = (size_t)n_src * g / n_groups, s1 = (size_t)n_src * (g + 1) / n_groups, ns = s1 - s0;
        e = cudaStreamWaitEvent(st, ctx->ev_group[g], 0);
        if (e != cudaSuccess) break;
        rc = few_waveform_ragged(ctx, d_t + s0 * n_t, n_t_src_host ? d_nts + s0 : nullptr, d_ph + s0 * n_t * 2, d_amp + s0 * n_t * n_modes * 2,
                                 d_l, d_m, d_n, d_th + s0, d_phi + s0, scale_host ? d_sc + s0 : nullptr, eps, t0, dt, n_samples, (int)ns,
                                 n_t, n_modes, h_out + s0 * (size_t)n_samples * 2, d_keep + s0 * n_modes, d_nk + s0, d_ws, ws_bytes, st);
        if (rc == FEW_OK && n_samples && !h_mapped)
            e = cudaMemcpyAsync(h_host + s0 * (size_t)n_samples * 2, d_h + s0 * (size_t)n_samples * 2, ns * (size_t)n_samples * 16,
                                cudaMemcpyDeviceToHost, st);
    }
    if (e == cudaSuccess && rc == FEW_OK) {
        if (keep_idx_host) e = cudaMemcpyAsync(keep_idx_host, d_keep, b_keep, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess && n_keep_host) e = cudaMemcpyAsync(n_keep_host, d_nk, b_nk, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) rc = few_device_status(ctx, nullptr, st);   // synchronises
    }
    if (e != cudaSuccess) { few_set_error("few_waveform_host: %s", cudaGetErrorString(e)); rc = FEW_ERR_CUDA; }
    // On every path, failing or not, nothing of this call is in flight when it returns: the kernels' stream and the copy stream
    // (whose host->device copies read the caller's amp_host and the staging block the next call overwrites) are both drained.
    cudaStreamSynchronize(st);
    cudaStreamSynchronize(cs);
    return rc;
}

extern "C" int few_waveform_host(few_ctx* ctx, const double* t_host, const double* phase_host, const double* amp_host,
                                 const int* l_host, const int* m_host, const int* n_host, const double* theta_host,
                                 const double* phi_host, const double* scale_host, double eps, double t0, double dt,
                                 long long n_samples, int n_src, int n_t, int n_modes,
                                 double* h_host, int* keep_idx_host, int* n_keep_host)
{
    return few_waveform_host_ragged(ctx, t_host, nullptr, phase_host, amp_host, l_host, m_host, n_host, theta_host, phi_host, scale_host, eps,
                                    t0, dt, n_samples, n_src, n_t, n_modes, h_host, keep_idx_host, n_keep_host);
}

// ---------------------------------------------------------------------------------------------------------------
// FP64 peak probe: 16 independent DFMA chains per thread, all in registers.
// ---------------------------------------------------------------------------------------------------------------
__global__ void few_fp64_peak_kernel(int iters, double* sink)
{
    double a[16];
    const double x = 1.0 + 1e-9 * threadIdx.x, y = 1e-12 * (blockIdx.x + 1);
#pragma unroll
    for (int i = 0; i < 16; ++i) a[i] = 1.0 + i * 1e-3;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) a[i] = fma(a[i], x, y);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += a[i];
    sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

extern "C" int few_fp64_peak_probe(few_ctx* ctx, int blocks, int threads, int iters, double* sink, void* stream)
{
    FEW_REQUIRE(ctx && sink, FEW_ERR_INVALID_ARG, "NULL argument");
    FEW_REQUIRE(blocks > 0 && threads > 0 && threads <= 1024 && iters > 0, FEW_ERR_INVALID_ARG, "bad launch shape");
    few_fp64_peak_kernel<<<blocks, threads, 0, (cudaStream_t)stream>>>(iters, sink);
    FEW_LAUNCHED(ctx);
    return FEW_OK;
}
