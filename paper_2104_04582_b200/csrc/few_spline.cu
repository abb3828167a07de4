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
// few_spline_factor_kernel (one block per source): the matrix depends on the grid only, so its Thomas factorisation (no
// pivoting) is done ONCE per source into six per-knot arrays in the caller's workspace -- a serial chain of n_t divisions
// that would otherwise sit on the critical path of every block of the fit kernel (it cost as much as the block's whole
// HBM time: 0.477 ms before, 0.372 ms with the pre-kernel on config 3; the capture of this version is in profiles/r01c_kernels.md, section few_spline_fit_kernel).
// few_spline_fit_kernel (FP64, thousands of systems): one thread per system, systems fastest in memory so every global
// access of a warp is a contiguous row.  The kernel is HBM-bound (8 B read + 32 B written per knot and system); see the
// comment at the kernel.  No cuSPARSE.
//
// few_spline_fit_dd_kernel (double-double, the two phases): the serial recurrences stay in FP64 and the extra precision
// comes from iterative refinement: solve in FP64, form the residual of the EXACT system (grid spacings and right-hand
// side as hi+lo pairs) in double-double -- parallel over knots --, solve for the correction in FP64, add it in
// double-double; twice.  Each pass shrinks the error by ~cond * 2^-53, so two passes reach the double-double level.
#include "few_common.cuh"

namespace {


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

// Factorisation of every source's grid into the workspace: fac[src][6][n_t] = inv_h, w, inv_d, u, rA, rB.
__global__ void __launch_bounds__(128)
few_spline_factor_kernel(const double* __restrict__ t_all, const int* __restrict__ n_t_src, int n_t, double* __restrict__ fac_all, int* status)
{
    extern __shared__ double smem[];
    const int n = few_knots(n_t_src, blockIdx.x, n_t, status);      // the source's knots; n_t is the stride of the padded arrays
    factor_grid(t_all + (size_t)blockIdx.x * n_t, n, smem, smem + n, smem + 2 * n, smem + 3 * n, smem + 4 * n, smem + 5 * n, status);
    __syncthreads();
    double* fac = fac_all + (size_t)blockIdx.x * 6 * n_t;
    for (int i = threadIdx.x; i < 6 * n; i += blockDim.x) fac[i] = smem[i];
}

// One thread per system.  Shared memory holds the source's factorisation and ONE tile, the forward-swept right-hand
// side D[n_t][W] (8 B per knot and system: what bounds the systems in flight per SM).  y is streamed straight from global
// memory in both sweeps through a register ring filled kSplU knots ahead (the second pass re-reads it from L2), so no load
// sits on the serial recurrences; c0..c3 of a segment are written together in the backward sweep as four coalesced rows.
constexpr int kSplU = 8;

__device__ __forceinline__ void cp_async_8(void* smem_dst, const void* gmem_src)
{
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// kLatency (few blocks per SM, e.g. one source): nothing bounds shared memory, so the block also stages its whole y tile
// with cp.async (every row in flight at once) and factors the grid itself while the rows arrive -- no pre-kernel, no
// global load inside the sweeps.  Same arithmetic in both modes.
template <bool kLatency>
__global__ void __launch_bounds__(128)
few_spline_fit_kernel(const double* __restrict__ t_all, const double* __restrict__ fac_all, const double* __restrict__ y_all,
                      const int* __restrict__ n_t_src, int n_t, int n_sys, double* __restrict__ coef_all, int* status)
{
    extern __shared__ double4 smem4[];
    const int W = blockDim.x, tid = threadIdx.x, n = few_knots(n_t_src, blockIdx.y, n_t, status);
    double4* F = smem4;                                   // [n] {w_i, rA_i, rB_i, 1/h_i}
    double2* Bk = reinterpret_cast<double2*>(F + n);      // [n] {u_i, 1/d'_i}
    double* D = reinterpret_cast<double*>(Bk + n);        // [n][W]
    double* Y = D + (size_t)n * W;                        // kLatency: [n][W] knot values, then [6][n] raw factorisation
    const int src = blockIdx.y;
    const int q = blockIdx.x * W + tid;
    const double* y = y_all + (size_t)src * n_t * n_sys + q;
    if (kLatency) {
        if (q < n_sys)
            for (int i = 0; i < n; ++i) cp_async_8(&Y[i * W + tid], y + (size_t)i * n_sys);
        double* raw = Y + (size_t)n * W;
        factor_grid(t_all + (size_t)src * n_t, n, raw, raw + n, raw + 2 * n, raw + 3 * n, raw + 4 * n, raw + 5 * n, status);
        __syncthreads();
        for (int i = tid; i < n; i += W) {
            F[i] = make_double4(raw[n + i], raw[4 * n + i], raw[5 * n + i], raw[i]);
            Bk[i] = make_double2(raw[3 * n + i], raw[2 * n + i]);
        }
        cp_async_wait_all();
    } else {
        const double* fac = fac_all + (size_t)src * 6 * n_t; // inv_h, w, inv_d, u, rA, rB
        for (int i = tid; i < n; i += W) {
            F[i] = make_double4(fac[n + i], fac[4 * n + i], fac[5 * n + i], fac[i]);
            Bk[i] = make_double2(fac[3 * n + i], fac[2 * n + i]);
        }
    }
    __syncthreads();
    if (q >= n_sys) return;
    double* coef = coef_all + (size_t)src * (n_t - 1) * 4 * n_sys + q;
    auto ld = [&](int i) {
        if (!(i >= 0 && i < n)) return 0.0;
        return kLatency ? Y[i * W + tid] : __ldg(y + (size_t)i * n_sys);
    };

    // ---- forward substitution: D_i = rhs_i - w_i D_{i-1}, rhs_i = rA_i d_{i-1} + rB_i d_i  (one dependent FMA per knot)
    double ring[kSplU];
    const double y0 = ld(0), y1 = ld(1), y2 = ld(2);
#pragma unroll
    for (int u = 0; u < kSplU; ++u) ring[u] = ld(3 + u);
    double dl_prev = (y1 - y0) * F[0].w;                  // d_0
    double dl = (y2 - y1) * F[1].w;                       // d_1
    double d = F[0].y * dl_prev + F[0].z * dl;            // row 0
    D[tid] = d;
    double y_cur = y2;                                    // y_{i+1} at the top of iteration i
    for (int base = 1; base <= n - 2; base += kSplU) {
        double nxt[kSplU];
#pragma unroll
        for (int u = 0; u < kSplU; ++u) nxt[u] = ld(base + kSplU + 2 + u);
#pragma unroll
        for (int u = 0; u < kSplU; ++u) {
            const int i = base + u;
            if (i <= n - 2) {
                // here: dl_prev = d_{i-1}, dl = d_i, y_cur = y_{i+1}, ring[u] = y_{i+2}
                const double4 f = F[i];
                d = fma(-f.x, d, fma(f.y, dl_prev, f.z * dl));
                D[i * W + tid] = d;
                if (i < n - 2) {
                    const double y_nxt = ring[u];
                    dl_prev = dl; dl = (y_nxt - y_cur) * F[i + 1].w;
                    y_cur = y_nxt;
                }
            }
        }
#pragma unroll
        for (int u = 0; u < kSplU; ++u) ring[u] = nxt[u];
    }
    // now dl = d_{n-2}, dl_prev = d_{n-3} (n >= 4), y_cur = y_{n-1}
    {
        const double4 f = F[n - 1];
        d = fma(-f.x, d, fma(f.y, dl_prev, f.z * dl));
    }

    // ---- back substitution + coefficients, written segment by segment (coalesced rows of n_sys)
    double s_nxt = d * Bk[n - 1].y;
    double y_hi = y_cur;                                  // y_{i+1}
#pragma unroll
    for (int u = 0; u < kSplU; ++u) ring[u] = ld(n - 2 - u);
    for (int top = n - 2; top >= 0; top -= kSplU) {
        double nxt[kSplU];
#pragma unroll
        for (int u = 0; u < kSplU; ++u) nxt[u] = ld(top - kSplU - u);
#pragma unroll
        for (int u = 0; u < kSplU; ++u) {
            const int i = top - u;
            if (i >= 0) {
                const double2 b = Bk[i];
                const double ih = F[i].w;
                const double s = fma(-b.x, s_nxt, D[i * W + tid] * b.y);
                const double y_lo = ring[u];
                const double dli = (y_hi - y_lo) * ih;
                double* c = coef + (size_t)i * 4 * n_sys;
                c[0] = y_lo;
                c[n_sys] = s;
                c[(size_t)2 * n_sys] = (3.0 * dli - 2.0 * s - s_nxt) * ih;
                c[(size_t)3 * n_sys] = (s + s_nxt - 2.0 * dli) * (ih * ih);
                s_nxt = s; y_hi = y_lo;
            }
        }
#pragma unroll
        for (int u = 0; u < kSplU; ++u) ring[u] = nxt[u];
    }
}

// ------------------------------------------------------------------------------------------------------------------
// Double-double fit by iterative refinement.  One block per (source, chunk of <= kDdSys systems).
// ------------------------------------------------------------------------------------------------------------------
constexpr int kDdSys = 4;         // systems per block (each needs its own serial FP64 sweeps: lanes 0..3 of warp 0)
constexpr int kDdThreads = 128;
constexpr int kDdRefine = 2;

__global__ void __launch_bounds__(kDdThreads)
few_spline_fit_dd_kernel(const double* __restrict__ t_all, const double* __restrict__ y_all, const int* __restrict__ n_t_src,
                         int n_t, int n_sys, double* __restrict__ coef_all, int* status)
{
    extern __shared__ double smem[];
    const int n = few_knots(n_t_src, blockIdx.y, n_t, status), tid = threadIdx.x;
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
    const double* t = t_all + (size_t)src * n_t;
    const double* y = y_all + (size_t)src * n_t * n_sys + q0;
    dd* coef = reinterpret_cast<dd*>(coef_all) + (size_t)src * (n_t - 1) * 4 * n_sys + q0;

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

extern "C" size_t few_spline_fit_workspace(int n_src, int n_t)
{
    if (n_src <= 0 || n_t < 4) return 0;
    return few_align_up((size_t)n_src * 6 * n_t * sizeof(double));
}

extern "C" int few_spline_fit_ragged(few_ctx* ctx, const double* t, const double* y, const int* n_t_src, int n_src, int n_t, int n_sys,
                                     double* coef, void* workspace, size_t workspace_bytes, void* stream)
{
    int rc = few_spline_check(ctx, t, y, coef, n_src, n_t, n_sys);
    if (rc) return rc;
    FEW_REQUIRE(n_t <= FEW_MAX_NT_SPLINE, FEW_ERR_LIMIT, "n_t > FEW_MAX_NT_SPLINE");
    FEW_REQUIRE(workspace && ((uintptr_t)workspace % 256) == 0 && workspace_bytes >= few_spline_fit_workspace(n_src, n_t),
                FEW_ERR_WORKSPACE, "workspace NULL, misaligned or too small");
    cudaStream_t st = (cudaStream_t)stream;
    double* fac = static_cast<double*>(workspace);
    const size_t cap = (size_t)ctx->smem_optin, half = cap / 2;
    const long long total = (long long)n_sys * n_src;
    // Latency regime: so few systems that all 32-wide blocks, each with its two tiles, are resident at once (one wave).
    auto bytes_lat = [&](int w) { return (size_t)n_t * (48 + 48 + 16 * (size_t)w); };
    if (bytes_lat(32) <= cap && (total + 31) / 32 <= (long long)ctx->sm_count * (long long)(cap / bytes_lat(32))) {
        const int W = 32;
        dim3 grid((n_sys + W - 1) / W, n_src);
        FEW_CUDA_CHECK(cudaFuncSetAttribute(few_spline_fit_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes_lat(W)));
        few_spline_fit_kernel<true><<<grid, W, bytes_lat(W), st>>>(t, nullptr, y, n_t_src, n_t, n_sys, coef, ctx->d_status);
        FEW_LAUNCHED(ctx);
        return FEW_OK;
    }
    // Throughput regime.  Block width W (systems per block): as wide as possible (longer contiguous rows per store) while at
    // least two blocks fit an SM and the grid still covers every SM twice.
    few_spline_factor_kernel<<<n_src, 128, (size_t)6 * n_t * sizeof(double), st>>>(t, n_t_src, n_t, fac, ctx->d_status);
    FEW_LAUNCHED(ctx);
    auto bytes = [&](int w) { return (size_t)n_t * (48 + 8 * (size_t)w); };
    int W = 128;
    while (W > 32 && (bytes(W) > half || total / W < 2LL * ctx->sm_count)) W >>= 1;
    FEW_REQUIRE(bytes(W) <= cap, FEW_ERR_LIMIT, "n_t too large for shared memory");
    dim3 grid((n_sys + W - 1) / W, n_src);
    FEW_CUDA_CHECK(cudaFuncSetAttribute(few_spline_fit_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes(W)));
    few_spline_fit_kernel<false><<<grid, W, bytes(W), st>>>(t, fac, y, n_t_src, n_t, n_sys, coef, ctx->d_status);
    FEW_LAUNCHED(ctx);
    return FEW_OK;
}

extern "C" int few_spline_fit(few_ctx* ctx, const double* t, const double* y, int n_src, int n_t, int n_sys,
                              double* coef, void* workspace, size_t workspace_bytes, void* stream)
{
    return few_spline_fit_ragged(ctx, t, y, nullptr, n_src, n_t, n_sys, coef, workspace, workspace_bytes, stream);
}

extern "C" int few_spline_fit_dd_ragged(few_ctx* ctx, const double* t, const double* y, const int* n_t_src, int n_src, int n_t, int n_sys,
                                        double* coef_dd, void* stream)
{
    int rc = few_spline_check(ctx, t, y, coef_dd, n_src, n_t, n_sys);
    if (rc) return rc;
    const size_t bytes = ((size_t)8 + 2 * 2 + kDdSys * (2 + 2 + 1)) * n_t * sizeof(double);
    FEW_REQUIRE(bytes <= (size_t)ctx->smem_optin, FEW_ERR_LIMIT, "n_t too large for shared memory");
    FEW_CUDA_CHECK(cudaFuncSetAttribute(few_spline_fit_dd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    dim3 grid((n_sys + kDdSys - 1) / kDdSys, n_src);
    few_spline_fit_dd_kernel<<<grid, kDdThreads, bytes, (cudaStream_t)stream>>>(t, y, n_t_src, n_t, n_sys, coef_dd, ctx->d_status);
    FEW_LAUNCHED(ctx);
    return FEW_OK;
}

extern "C" int few_spline_fit_dd(few_ctx* ctx, const double* t, const double* y, int n_src, int n_t, int n_sys,
                                 double* coef_dd, void* stream)
{
    return few_spline_fit_dd_ragged(ctx, t, y, nullptr, n_src, n_t, n_sys, coef_dd, stream);
}
