// few_spline.cu -- S1: batched not-a-knot cubic spline fit (sec. III C: "not-a-knot" end
// conditions, "tridiagonal banded matrix representation", "all arrays to be interpolated exist on the same sparse
// time grid", "~1e2 - 1e4 separate splines").
//
// Unknowns are the knot slopes s_i = S'(t_i):
//   interior rows  h_i s_{i-1} + 2(h_{i-1}+h_i) s_i + h_{i-1} s_{i+1} = 3(h_i d_{i-1} + h_{i-1} d_i),  d_i = (y_{i+1}-y_i)/h_i
//   first row      h_1 s_0 + (h_0+h_1) s_1 = [(3h_0+2h_1) h_1 d_0 + h_0^2 d_1] / (h_0+h_1)      (not-a-knot at t_1, s_2 eliminated)
//   last row       mirror image at t_{n-2}.
// The matrix depends on the grid only, which every system of a source shares, so each block factors it ONCE (thread 0,
// Thomas without pivoting) into per-knot multipliers held in shared memory; every thread then owns one system and runs the
// forward and backward substitutions as pure FMA chains.  Systems are the fastest index of y and coef, so all global
// accesses of a warp are 256-byte contiguous rows.  No cuSPARSE, no global scratch: the forward-swept right-hand side
// lives in a shared-memory column per thread.
#include "few_common.cuh"

namespace {

constexpr int kConstArrays = 6;   // inv_h, w, inv_d, up, rA, rB

__global__ void few_spline_fit_kernel(const double* __restrict__ t_all, const double* __restrict__ y_all,
                                      int n_t, int n_sys, double* __restrict__ coef_all, int* status)
{
    extern __shared__ double smem[];
    const int W = blockDim.x, tid = threadIdx.x, n = n_t;
    double* inv_h = smem;             // [n]   1/h_i
    double* wm = inv_h + n;           // [n]   elimination multiplier lo_i / di'_{i-1}
    double* inv_d = wm + n;           // [n]   1 / di'_i
    double* up = inv_d + n;           // [n]   super-diagonal
    double* rA = up + n;              // [n]   rhs_i = rA_i * d_{ia} + rB_i * d_{ib}
    double* rB = rA + n;              // [n]
    double* D = rB + n;               // [n][W] forward-swept rhs, one column per thread

    const int src = blockIdx.y;
    const double* t = t_all + (size_t)src * n;
    const double* y = y_all + (size_t)src * n * n_sys;
    double* coef = coef_all + (size_t)src * (n - 1) * 4 * n_sys;
    const int q = blockIdx.x * W + tid;
    const bool active = q < n_sys;

    // ---- grid-only part: h, 1/h, rhs weights (parallel), then the serial factorisation by thread 0
    for (int i = tid; i < n - 1; i += W) {
        double h = t[i + 1] - t[i];
        if (!(h > 0.0)) atomicOr(status, FEW_DEV_NOT_INCREASING);
        inv_h[i] = 1.0 / h;
    }
    for (int i = tid; i < n; i += W) {
        if (i >= 1 && i <= n - 2) {
            double hm = t[i] - t[i - 1], hp = t[i + 1] - t[i];
            rA[i] = 3.0 * hp; rB[i] = 3.0 * hm; up[i] = hm;
        } else if (i == 0) {
            double h0 = t[1] - t[0], h1 = t[2] - t[1];
            rA[0] = (3.0 * h0 + 2.0 * h1) * h1 / (h0 + h1); rB[0] = h0 * h0 / (h0 + h1); up[0] = h0 + h1;
        } else {
            double ha = t[n - 2] - t[n - 3], hb = t[n - 1] - t[n - 2];   // h_{n-3}, h_{n-2}
            rA[i] = hb * hb / (ha + hb); rB[i] = (2.0 * ha + 3.0 * hb) * ha / (ha + hb); up[i] = 0.0;
        }
    }
    __syncthreads();
    if (tid == 0) {
        double di = t[2] - t[1];                      // row 0 diagonal h_1
        wm[0] = 0.0; inv_d[0] = 1.0 / di;
        for (int i = 1; i < n; ++i) {
            double lo, dg;
            if (i < n - 1) { lo = t[i + 1] - t[i]; dg = 2.0 * (t[i + 1] - t[i - 1]); }
            else { lo = t[n - 1] - t[n - 3]; dg = t[n - 2] - t[n - 3]; }
            double w = lo / di;
            di = dg - w * up[i - 1];
            wm[i] = w; inv_d[i] = 1.0 / di;
        }
    }
    __syncthreads();
    if (!active) return;

    // ---- forward substitution: d'_i = rhs_i - w_i d'_{i-1}
    const double* yq = y + q;
    double y_cur = yq[0], y_nxt = yq[n_sys];
    double dl_prev = (y_nxt - y_cur) * inv_h[0];                 // d_0
    y_cur = y_nxt; y_nxt = yq[(size_t)2 * n_sys];
    double dl = (y_nxt - y_cur) * inv_h[1];                      // d_1
    double d = rA[0] * dl_prev + rB[0] * dl;
    D[tid] = d;
    double dl_pp = dl_prev;                                      // d_{i-2} once i advances
#pragma unroll 4
    for (int i = 1; i <= n - 2; ++i) {
        // here: dl_prev = d_{i-1}, dl = d_i, y_nxt = y_{i+1}
        d = fma(-wm[i], d, fma(rA[i], dl_prev, rB[i] * dl));
        D[i * W + tid] = d;
        if (i < n - 2) {
            y_cur = y_nxt; y_nxt = yq[(size_t)(i + 2) * n_sys];
            dl_pp = dl_prev; dl_prev = dl; dl = (y_nxt - y_cur) * inv_h[i + 1];
        }
    }
    // now dl = d_{n-2}, dl_prev = d_{n-3} (n >= 4)
    (void)dl_pp;
    d = fma(-wm[n - 1], d, fma(rA[n - 1], dl_prev, rB[n - 1] * dl));

    // ---- back substitution + coefficients, written segment by segment (coalesced rows of n_sys)
    double s_nxt = d * inv_d[n - 1];
    double y_hi = y_nxt;                                         // y_{n-1}
#pragma unroll 4
    for (int i = n - 2; i >= 0; --i) {
        double s = (D[i * W + tid] - up[i] * s_nxt) * inv_d[i];
        double y_lo = yq[(size_t)i * n_sys];
        double ih = inv_h[i];
        double dli = (y_hi - y_lo) * ih;
        double* c = coef + (size_t)i * 4 * n_sys + q;
        c[0] = y_lo;
        c[n_sys] = s;
        c[(size_t)2 * n_sys] = (3.0 * dli - 2.0 * s - s_nxt) * ih;
        c[(size_t)3 * n_sys] = (s + s_nxt - 2.0 * dli) * (ih * ih);
        s_nxt = s; y_hi = y_lo;
    }
}

// Double-double variant for the phases: few systems (2 per source), every quantity -- grid spacings, factorisation,
// right-hand sides, slopes, coefficients -- carried as hi+lo pairs.  The forward-swept rhs is parked in the c1 slot of the
// output (each thread re-reads only what it wrote).  Thread 0 of each block factors the grid into shared memory.
__global__ void few_spline_fit_dd_kernel(const double* __restrict__ t_all, const double* __restrict__ y_all,
                                         int n_t, int n_sys, double* __restrict__ coef_all, int* status)
{
    extern __shared__ double smem[];
    const int n = n_t, tid = threadIdx.x;
    dd* inv_h = reinterpret_cast<dd*>(smem);   // [n]
    dd* wm = inv_h + n;
    dd* inv_d = wm + n;
    dd* up = inv_d + n;
    dd* rA = up + n;
    dd* rB = rA + n;
    dd* hh = rB + n;                           // [n] h_i
    const int src = blockIdx.y;
    const double* t = t_all + (size_t)src * n;
    const double* y = y_all + (size_t)src * n * n_sys;
    dd* coef = reinterpret_cast<dd*>(coef_all) + (size_t)src * (n - 1) * 4 * n_sys;
    const int q = blockIdx.x * blockDim.x + tid;

    for (int i = tid; i < n - 1; i += blockDim.x) {
        dd h = dd_from_diff(t[i + 1], t[i]);
        if (!(h.hi > 0.0)) atomicOr(status, FEW_DEV_NOT_INCREASING);
        hh[i] = h;
        inv_h[i] = dd_div(dd_make(1.0), h);
    }
    __syncthreads();
    for (int i = tid; i < n; i += blockDim.x) {
        if (i >= 1 && i <= n - 2) {
            rA[i] = dd_mul_d(hh[i], 3.0); rB[i] = dd_mul_d(hh[i - 1], 3.0); up[i] = hh[i - 1];
        } else if (i == 0) {
            dd h0 = hh[0], h1 = hh[1], sum = dd_add(h0, h1);
            rA[0] = dd_div(dd_mul(dd_add(dd_mul_d(h0, 3.0), dd_mul_d(h1, 2.0)), h1), sum);
            rB[0] = dd_div(dd_mul(h0, h0), sum);
            up[0] = sum;
        } else {
            dd ha = hh[n - 3], hb = hh[n - 2], sum = dd_add(ha, hb);
            rA[i] = dd_div(dd_mul(hb, hb), sum);
            rB[i] = dd_div(dd_mul(dd_add(dd_mul_d(ha, 2.0), dd_mul_d(hb, 3.0)), ha), sum);
            up[i] = dd_make(0.0);
        }
    }
    __syncthreads();
    if (tid == 0) {
        dd di = hh[1];
        wm[0] = dd_make(0.0); inv_d[0] = dd_div(dd_make(1.0), di);
        for (int i = 1; i < n; ++i) {
            dd lo, dg;
            if (i < n - 1) { lo = hh[i]; dg = dd_mul_d(dd_add(hh[i - 1], hh[i]), 2.0); }
            else { lo = dd_add(hh[n - 2], hh[n - 3]); dg = hh[n - 3]; }
            dd w = dd_div(lo, di);
            di = dd_sub(dg, dd_mul(w, up[i - 1]));
            wm[i] = w; inv_d[i] = dd_div(dd_make(1.0), di);
        }
    }
    __syncthreads();
    if (q >= n_sys) return;

    const double* yq = y + q;
    auto delta = [&](int i) { return dd_mul(dd_from_diff(yq[(size_t)(i + 1) * n_sys], yq[(size_t)i * n_sys]), inv_h[i]); };
    auto park = [&](int i) -> dd& { return coef[((size_t)i * 4 + 1) * n_sys + q]; };   // c1 slot of segment i as scratch

    dd dl_prev = delta(0), dl = delta(1);
    dd d = dd_add(dd_mul(rA[0], dl_prev), dd_mul(rB[0], dl));
    park(0) = d;
    for (int i = 1; i <= n - 2; ++i) {
        d = dd_sub(dd_add(dd_mul(rA[i], dl_prev), dd_mul(rB[i], dl)), dd_mul(wm[i], d));
        park(i) = d;
        if (i < n - 2) { dl_prev = dl; dl = delta(i + 1); }
    }
    d = dd_sub(dd_add(dd_mul(rA[n - 1], dl_prev), dd_mul(rB[n - 1], dl)), dd_mul(wm[n - 1], d));
    dd s_nxt = dd_mul(d, inv_d[n - 1]);
    for (int i = n - 2; i >= 0; --i) {
        dd s = dd_mul(dd_sub(park(i), dd_mul(up[i], s_nxt)), inv_d[i]);
        dd dli = delta(i), ih = inv_h[i];
        dd* c = coef + (size_t)i * 4 * n_sys + q;
        c[0] = dd_make(yq[(size_t)i * n_sys]);
        c[n_sys] = s;
        c[(size_t)2 * n_sys] = dd_mul(dd_sub(dd_sub(dd_mul_d(dli, 3.0), dd_mul_d(s, 2.0)), s_nxt), ih);
        c[(size_t)3 * n_sys] = dd_mul(dd_sub(dd_add(s, s_nxt), dd_mul_d(dli, 2.0)), dd_mul(ih, ih));
        s_nxt = s;
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
    // widest block whose D column tile fits: prefer >= 2 resident blocks per SM
    int W = 128;
    auto bytes = [&](int w) { return (size_t)(kConstArrays + w) * n_t * sizeof(double); };
    while (W > 32 && bytes(W) > (size_t)ctx->smem_optin / 2) W >>= 1;
    FEW_REQUIRE(bytes(W) <= (size_t)ctx->smem_optin, FEW_ERR_LIMIT, "n_t too large for shared memory");
    FEW_CUDA_CHECK(cudaFuncSetAttribute(few_spline_fit_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes(W)));
    dim3 grid((n_sys + W - 1) / W, n_src);
    few_spline_fit_kernel<<<grid, W, bytes(W), (cudaStream_t)stream>>>(t, y, n_t, n_sys, coef, ctx->d_status);
    FEW_CUDA_CHECK(cudaGetLastError());
    return FEW_OK;
}

extern "C" int few_spline_fit_dd(few_ctx* ctx, const double* t, const double* y, int n_src, int n_t, int n_sys,
                                 double* coef_dd, void* stream)
{
    int rc = few_spline_check(ctx, t, y, coef_dd, n_src, n_t, n_sys);
    if (rc) return rc;
    size_t bytes = (size_t)7 * n_t * sizeof(dd);
    FEW_REQUIRE(bytes <= (size_t)ctx->smem_optin, FEW_ERR_LIMIT, "n_t too large for shared memory");
    FEW_CUDA_CHECK(cudaFuncSetAttribute(few_spline_fit_dd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    const int W = 32;
    dim3 grid((n_sys + W - 1) / W, n_src);
    few_spline_fit_dd_kernel<<<grid, W, bytes, (cudaStream_t)stream>>>(t, y, n_t, n_sys, coef_dd, ctx->d_status);
    FEW_CUDA_CHECK(cudaGetLastError());
    return FEW_OK;
}
