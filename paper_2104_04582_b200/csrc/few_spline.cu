// few_spline.cu -- S1: batched not-a-knot cubic spline fit (sec. III C: "not-a-knot" end
// conditions, "tridiagonal banded matrix representation", "all arrays to be interpolated exist on the same sparse
// time grid", "~1e2 - 1e4 separate splines").
//
// Unknowns are the knot slopes s_i = S'(t_i):
//   interior rows  h_i s_{i-1} + 2(h_{i-1}+h_i) s_i + h_{i-1} s_{i+1} = 3(h_i d_{i-1} + h_{i-1} d_i),  d_i = (y_{i+1}-y_i)/h_i
//   first row      h_1 s_0 + (h_0+h_1) s_1 = [(3h_0+2h_1) h_1 d_0 + h_0^2 d_1] / (h_0+h_1)      (not-a-knot at t_1, s_2 eliminated)
//   last row       mirror image at t_{n-2}.
// The matrix depends on the grid only, which every system of a source shares.
//
// few_spline_fit_kernel (FP64, thousands of systems): one thread per system, systems fastest in memory so every global
// access of a warp is a contiguous row.  A block first streams its [n_t x W] tile of y into shared memory with cp.async
// (all rows in flight at once: the kernel is HBM-bound, 8 B read + 32 B written per knot and system), while thread 0
// factors the tridiagonal matrix (Thomas, no pivoting) into per-knot multipliers.  The forward and backward substitutions
// are then single-FMA recurrences out of shared memory, and the four coefficient planes are written as coalesced rows.
// No cuSPARSE, no global scratch.
//
// few_spline_fit_dd_kernel (double-double, the two phases): the serial recurrences stay in FP64 and the extra precision
// comes from iterative refinement: solve in FP64, form the residual of the EXACT system (grid spacings and right-hand
// side as hi+lo pairs) in double-double -- parallel over knots --, solve for the correction in FP64, add it in
// double-double; twice.  Each pass shrinks the error by ~cond * 2^-53, so two passes reach the double-double level.
#include "few_common.cuh"

namespace {

constexpr int kConstArrays = 7;   // inv_h, w, inv_d, u = up*inv_d, rA, rB, (spare for alignment)

__device__ __forceinline__ void cp_async_8(void* smem_dst, const void* gmem_src)
{
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// Grid-only part shared by both kernels: 1/h, rhs weights, Thomas factorisation in FP64 (thread 0).
__device__ void factor_grid(const double* __restrict__ t, int n, double* inv_h, double* wm, double* inv_d, double* um,
                            double* rA, double* rB, int* status)
{
    const int tid = threadIdx.x, W = blockDim.x;
    for (int i = tid; i < n - 1; i += W) {
        double h = t[i + 1] - t[i];
        if (!(h > 0.0)) atomicOr(status, FEW_DEV_NOT_INCREASING);
        inv_h[i] = 1.0 / h;
    }
    for (int i = tid; i < n; i += W) {
        if (i >= 1 && i <= n - 2) {
            double hm = t[i] - t[i - 1], hp = t[i + 1] - t[i];
            rA[i] = 3.0 * hp; rB[i] = 3.0 * hm;
        } else if (i == 0) {
            double h0 = t[1] - t[0], h1 = t[2] - t[1];
            rA[0] = (3.0 * h0 + 2.0 * h1) * h1 / (h0 + h1); rB[0] = h0 * h0 / (h0 + h1);
        } else {
            double ha = t[n - 2] - t[n - 3], hb = t[n - 1] - t[n - 2];   // h_{n-3}, h_{n-2}
            rA[i] = hb * hb / (ha + hb); rB[i] = (2.0 * ha + 3.0 * hb) * ha / (ha + hb);
        }
    }
    if (tid == 0) {
        double di = t[2] - t[1];                      // row 0: diagonal h_1, super-diagonal h_0 + h_1
        double up_prev = t[2] - t[0];
        wm[0] = 0.0; inv_d[0] = 1.0 / di; um[0] = up_prev * inv_d[0];
        for (int i = 1; i < n; ++i) {
            double lo, dg, up;
            if (i < n - 1) { lo = t[i + 1] - t[i]; dg = 2.0 * (t[i + 1] - t[i - 1]); up = t[i] - t[i - 1]; }
            else { lo = t[n - 1] - t[n - 3]; dg = t[n - 2] - t[n - 3]; up = 0.0; }
            double w = lo * inv_d[i - 1];
            di = fma(-w, up_prev, dg);
            double id = 1.0 / di;
            wm[i] = w; inv_d[i] = id; um[i] = up * id;
            up_prev = up;
        }
    }
}

template <bool kTwoTiles>
__global__ void few_spline_fit_kernel(const double* __restrict__ t_all, const double* __restrict__ y_all,
                                      int n_t, int n_sys, double* __restrict__ coef_all, int* status)
{
    extern __shared__ double smem[];
    const int W = blockDim.x, tid = threadIdx.x, n = n_t;
    double* inv_h = smem;             // [n]   1/h_i
    double* wm = inv_h + n;           // [n]   elimination multiplier lo_i / di'_{i-1}
    double* inv_d = wm + n;           // [n]   1 / di'_i
    double* um = inv_d + n;           // [n]   up_i / di'_i
    double* rA = um + n;              // [n]   rhs_i = rA_i * d_{ia} + rB_i * d_{ib}
    double* rB = rA + n;              // [n]
    double* Y = rB + 2 * n;           // [n][W] knot values (later overwritten by the forward-swept rhs if !kTwoTiles)
    double* D = kTwoTiles ? Y + (size_t)n * W : Y;

    const int src = blockIdx.y;
    const double* t = t_all + (size_t)src * n;
    const double* y = y_all + (size_t)src * n * n_sys;
    double* coef = coef_all + (size_t)src * (n - 1) * 4 * n_sys;
    const int q = blockIdx.x * W + tid;
    const bool active = q < n_sys;

    // ---- stream the tile in: n rows of W doubles, every row in flight at once
    if (active) {
        const double* yq = y + q;
        for (int i = 0; i < n; ++i) cp_async_8(&Y[i * W + tid], yq + (size_t)i * n_sys);
    }
    factor_grid(t, n, inv_h, wm, inv_d, um, rA, rB, status);
    cp_async_wait_all();
    __syncthreads();
    if (!active) return;

    // ---- forward substitution: d'_i = rhs_i - w_i d'_{i-1}  (one dependent FMA per knot)
    double y_cur = Y[tid], y_nxt = Y[W + tid];
    double dl_prev = (y_nxt - y_cur) * inv_h[0];                 // d_0
    y_cur = y_nxt; y_nxt = Y[2 * W + tid];
    double dl = (y_nxt - y_cur) * inv_h[1];                      // d_1
    double d = rA[0] * dl_prev + rB[0] * dl;
    if (!kTwoTiles) coef[q] = Y[tid];                            // c0 of segment 0 leaves before its slot is reused
    D[tid] = d;
#pragma unroll 4
    for (int i = 1; i <= n - 2; ++i) {
        // here: dl_prev = d_{i-1}, dl = d_i, y_cur = y_i, y_nxt = y_{i+1}
        d = fma(-wm[i], d, fma(rA[i], dl_prev, rB[i] * dl));
        if (!kTwoTiles) coef[(size_t)i * 4 * n_sys + q] = y_cur;
        D[i * W + tid] = d;
        if (i < n - 2) {
            y_cur = y_nxt; y_nxt = Y[(i + 2) * W + tid];
            dl_prev = dl; dl = (y_nxt - y_cur) * inv_h[i + 1];
        }
    }
    // now dl = d_{n-2}, dl_prev = d_{n-3} (n >= 4), y_nxt = y_{n-1}
    d = fma(-wm[n - 1], d, fma(rA[n - 1], dl_prev, rB[n - 1] * dl));

    // ---- back substitution + coefficients, written segment by segment (coalesced rows of n_sys)
    double s_nxt = d * inv_d[n - 1];
    double y_hi = y_nxt;                                         // y_{n-1}
#pragma unroll 4
    for (int i = n - 2; i >= 0; --i) {
        const double s = fma(-um[i], s_nxt, D[i * W + tid] * inv_d[i]);
        double* c = coef + (size_t)i * 4 * n_sys + q;
        const double y_lo = kTwoTiles ? Y[i * W + tid] : c[0];   // !kTwoTiles: re-read what this thread wrote (L1/L2 hit)
        const double ih = inv_h[i];
        const double dli = (y_hi - y_lo) * ih;
        if (kTwoTiles) c[0] = y_lo;
        c[n_sys] = s;
        c[(size_t)2 * n_sys] = (3.0 * dli - 2.0 * s - s_nxt) * ih;
        c[(size_t)3 * n_sys] = (s + s_nxt - 2.0 * dli) * (ih * ih);
        s_nxt = s; y_hi = y_lo;
    }
}

// ------------------------------------------------------------------------------------------------------------------
// Double-double fit by iterative refinement.  One block per (source, chunk of <= kDdSys systems).
// ------------------------------------------------------------------------------------------------------------------
constexpr int kDdSys = 4;         // systems per block (each needs its own serial FP64 sweeps: lanes 0..3 of warp 0)
constexpr int kDdThreads = 128;
constexpr int kDdRefine = 2;

__global__ void __launch_bounds__(kDdThreads)
few_spline_fit_dd_kernel(const double* __restrict__ t_all, const double* __restrict__ y_all,
                         int n_t, int n_sys, double* __restrict__ coef_all, int* status)
{
    extern __shared__ double smem[];
    const int n = n_t, tid = threadIdx.x;
    double* inv_h = smem;                 // FP64 preconditioner (factor_grid)
    double* wm = inv_h + n;
    double* inv_d = wm + n;
    double* um = inv_d + n;
    double* rA = um + n;
    double* rB = rA + n;
    dd* hh = reinterpret_cast<dd*>(rB + 2 * n);   // [n]   exact spacings h_i = t_{i+1} - t_i
    dd* ihh = hh + n;                             // [n]   1 / h_i
    dd* rhs = ihh + n;                            // [kDdSys][n]  exact right-hand side
    dd* sl = rhs + (size_t)kDdSys * n;            // [kDdSys][n]  slopes, refined in place
    double* wk = reinterpret_cast<double*>(sl + (size_t)kDdSys * n);   // [kDdSys][n]  FP64 work vector of the sweeps

    const int src = blockIdx.y, q0 = blockIdx.x * kDdSys;
    const int ns = min(kDdSys, n_sys - q0);
    const double* t = t_all + (size_t)src * n;
    const double* y = y_all + (size_t)src * n * n_sys + q0;
    dd* coef = reinterpret_cast<dd*>(coef_all) + (size_t)src * (n - 1) * 4 * n_sys + q0;

    factor_grid(t, n, inv_h, wm, inv_d, um, rA, rB, status);
    for (int i = tid; i < n - 1; i += kDdThreads) {
        dd h = dd_from_diff(t[i + 1], t[i]);
        hh[i] = h;
        ihh[i] = dd_div(dd_make(1.0), h);
    }
    __syncthreads();

    auto delta = [&](int q, int i) { return dd_mul(dd_from_diff(y[(size_t)(i + 1) * n_sys + q], y[(size_t)i * n_sys + q]), ihh[i]); };
    // exact matrix rows (lo, dg, up) and right-hand side, all double-double, parallel over knots
    auto row = [&](int i, dd& lo, dd& dg, dd& up) {
        if (i == 0) { lo = dd_make(0.0); dg = hh[1]; up = dd_add(hh[0], hh[1]); }
        else if (i < n - 1) { lo = hh[i]; dg = dd_mul_d(dd_add(hh[i - 1], hh[i]), 2.0); up = hh[i - 1]; }
        else { lo = dd_add(hh[n - 2], hh[n - 3]); dg = hh[n - 3]; up = dd_make(0.0); }
    };
    for (int idx = tid; idx < ns * n; idx += kDdThreads) {
        const int q = idx / n, i = idx - q * n;
        dd r;
        if (i == 0) {
            dd h0 = hh[0], h1 = hh[1], sum = dd_add(h0, h1);
            dd a = dd_div(dd_mul(dd_add(dd_mul_d(h0, 3.0), dd_mul_d(h1, 2.0)), h1), sum), b = dd_div(dd_mul(h0, h0), sum);
            r = dd_add(dd_mul(a, delta(q, 0)), dd_mul(b, delta(q, 1)));
        } else if (i < n - 1) {
            r = dd_mul_d(dd_add(dd_mul(hh[i], delta(q, i - 1)), dd_mul(hh[i - 1], delta(q, i))), 3.0);
        } else {
            dd ha = hh[n - 3], hb = hh[n - 2], sum = dd_add(ha, hb);
            dd a = dd_div(dd_mul(hb, hb), sum), b = dd_div(dd_mul(dd_add(dd_mul_d(ha, 2.0), dd_mul_d(hb, 3.0)), ha), sum);
            r = dd_add(dd_mul(a, delta(q, n - 3)), dd_mul(b, delta(q, n - 2)));
        }
        rhs[(size_t)q * n + i] = r;
        sl[(size_t)q * n + i] = dd_make(0.0);
        wk[(size_t)q * n + i] = r.hi;                        // first pass solves M s = rhs in FP64
    }
    __syncthreads();

    for (int pass = 0; pass <= kDdRefine; ++pass) {
        if (tid < ns) {                                      // serial FP64 sweeps, one lane per system
            double* v = wk + (size_t)tid * n;
            double d = v[0];
            for (int i = 1; i < n; ++i) { d = fma(-wm[i], d, v[i]); v[i] = d; }
            double s = v[n - 1] * inv_d[n - 1];
            v[n - 1] = s;
            for (int i = n - 2; i >= 0; --i) { s = fma(-um[i], s, v[i] * inv_d[i]); v[i] = s; }
        }
        __syncthreads();
        for (int idx = tid; idx < ns * n; idx += kDdThreads)                 // s += correction (double-double)
            sl[idx] = dd_add_d(sl[idx], wk[idx]);
        __syncthreads();
        if (pass == kDdRefine) break;
        for (int idx = tid; idx < ns * n; idx += kDdThreads) {               // residual of the exact system
            const int q = idx / n, i = idx - q * n;
            const dd* s = sl + (size_t)q * n;
            dd lo, dg, up;
            row(i, lo, dg, up);
            dd acc = dd_sub(rhs[idx], dd_mul(dg, s[i]));
            if (i > 0) acc = dd_sub(acc, dd_mul(lo, s[i - 1]));
            if (i < n - 1) acc = dd_sub(acc, dd_mul(up, s[i + 1]));
            wk[idx] = acc.hi;
        }
        __syncthreads();
    }

    for (int idx = tid; idx < ns * (n - 1); idx += kDdThreads) {              // coefficients, parallel over segments
        const int q = idx / (n - 1), i = idx - q * (n - 1);
        const dd s = sl[(size_t)q * n + i], s_nxt = sl[(size_t)q * n + i + 1];
        const dd dli = delta(q, i), ih = ihh[i];
        dd* c = coef + (size_t)i * 4 * n_sys + q;
        c[0] = dd_make(y[(size_t)i * n_sys + q]);
        c[n_sys] = s;
        c[(size_t)2 * n_sys] = dd_mul(dd_sub(dd_sub(dd_mul_d(dli, 3.0), dd_mul_d(s, 2.0)), s_nxt), ih);
        c[(size_t)3 * n_sys] = dd_mul(dd_sub(dd_add(s, s_nxt), dd_mul_d(dli, 2.0)), dd_mul(ih, ih));
    }
}

}  // namespace

static int few_spline_check(few_ctx* ctx, const void* t, const void* y, const void* coef, int n_src, int n_t, int n_sys)
{
    FEW_REQUIRE(ctx && t && y && coef, FEW_ERR_INVALID_ARG, "NULL argument");
    FEW_REQUIRE(n_src > 0 && n_sys > 0, FEW_ERR_INVALID_ARG, "n_src and n_sys must be positive");
    FEW_REQUIRE(n_t >= 4, FEW_ERR_TOO_FEW_POINTS, "a not-a-knot cubic spline needs n_t >= 4");
    FEW_REQUIRE(n_src <= 65535, FEW_ERR_LIMIT, "n_src > 65535");
    return FEW_OK;
}

extern "C" int few_spline_fit(few_ctx* ctx, const double* t, const double* y, int n_src, int n_t, int n_sys,
                              double* coef, void* stream)
{
    int rc = few_spline_check(ctx, t, y, coef, n_src, n_t, n_sys);
    if (rc) return rc;
    FEW_REQUIRE(n_t <= FEW_MAX_NT_SPLINE, FEW_ERR_LIMIT, "n_t > FEW_MAX_NT_SPLINE");
    // Block width W (systems per block): keep every SM busy (>= 2 blocks per SM when the batch allows) and at least two
    // blocks resident per SM; prefer two shared-memory tiles (y and the swept rhs), fall back to one.
    auto bytes = [&](int w, bool two) { return (size_t)(kConstArrays + (two ? 2 : 1) * w) * n_t * sizeof(double); };
    const size_t cap = (size_t)ctx->smem_optin, half = cap / 2;
    int W = 128;
    const long long total = (long long)n_sys * n_src;
    while (W > 32 && (bytes(W, true) > half || total / W < 2LL * ctx->sm_count)) W >>= 1;
    bool two = bytes(W, true) <= cap;
    if (!two) { W = 128; while (W > 32 && bytes(W, false) > half) W >>= 1; }
    FEW_REQUIRE(bytes(W, two) <= cap, FEW_ERR_LIMIT, "n_t too large for shared memory");
    dim3 grid((n_sys + W - 1) / W, n_src);
    const size_t sm = bytes(W, two);
    if (two) {
        FEW_CUDA_CHECK(cudaFuncSetAttribute(few_spline_fit_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
        few_spline_fit_kernel<true><<<grid, W, sm, (cudaStream_t)stream>>>(t, y, n_t, n_sys, coef, ctx->d_status);
    } else {
        FEW_CUDA_CHECK(cudaFuncSetAttribute(few_spline_fit_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
        few_spline_fit_kernel<false><<<grid, W, sm, (cudaStream_t)stream>>>(t, y, n_t, n_sys, coef, ctx->d_status);
    }
    FEW_CUDA_CHECK(cudaGetLastError());
    return FEW_OK;
}

extern "C" int few_spline_fit_dd(few_ctx* ctx, const double* t, const double* y, int n_src, int n_t, int n_sys,
                                 double* coef_dd, void* stream)
{
    int rc = few_spline_check(ctx, t, y, coef_dd, n_src, n_t, n_sys);
    if (rc) return rc;
    const size_t bytes = ((size_t)(kConstArrays + 1) + 2 * 2 + kDdSys * (2 + 2 + 1)) * n_t * sizeof(double);
    FEW_REQUIRE(bytes <= (size_t)ctx->smem_optin, FEW_ERR_LIMIT, "n_t too large for shared memory");
    FEW_CUDA_CHECK(cudaFuncSetAttribute(few_spline_fit_dd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    dim3 grid((n_sys + kDdSys - 1) / kDdSys, n_src);
    few_spline_fit_dd_kernel<<<grid, kDdThreads, bytes, (cudaStream_t)stream>>>(t, y, n_t, n_sys, coef_dd, ctx->d_status);
    FEW_CUDA_CHECK(cudaGetLastError());
    return FEW_OK;
}
