// few_ylm.cu -- S0: spin-weight -2 spherical harmonics as per-source constants (Eq. (10):
// "the regular -2 spin-weighted spherical harmonics ... constant over the whole orbit").
//
// Computed from the Wigner small-d function,  sY_lm(theta, phi) = (-1)^s sqrt((2l+1)/4pi) d^l_{m,-s}(theta) e^{i m phi},
//   d^l_{a,b}(beta) = sqrt((l+a)!(l-a)!(l+b)!(l-b)!) sum_k (-1)^{a-b+k} cos(beta/2)^{2l+b-a-2k} sin(beta/2)^{a-b+2k}
//                     / ((l+b-k)! k! (a-b+k)! (l-a-k)!),
// which agrees with the Goldberg et al. convention (R11).  few_ylm_m2 backs the host helper few_ylm; the device
// kernel evaluates the same sum from shared tables.
#include <math.h>
#include "few_common.cuh"

__host__ __device__ static inline double few_fact(int k)
{
    double f = 1.0;
    for (int i = 2; i <= k; ++i) f *= (double)i;
    return f;
}

__host__ __device__ static inline double few_ipow(double x, int e)
{
    double r = 1.0;
    for (int i = 0; i < e; ++i) r *= x;
    return r;
}

// -2Y_lm(theta, phi); caller guarantees 2 <= l <= FEW_MAX_L, |m| <= l.
__host__ __device__ static inline void few_ylm_m2(int l, int m, double theta, double phi, double* re, double* im)
{
    const int a = m, b = 2;                    // d^l_{m, -s}, s = -2
    const double ch = cos(0.5 * theta), sh = sin(0.5 * theta);
    int k0 = (b - a) > 0 ? (b - a) : 0;        // a - b + k >= 0
    int k1 = (l + b) < (l - a) ? (l + b) : (l - a);
    double tot = 0.0;
    for (int k = k0; k <= k1; ++k) {
        double term = few_ipow(ch, 2 * l + b - a - 2 * k) * few_ipow(sh, a - b + 2 * k) /
                      (few_fact(l + b - k) * few_fact(k) * few_fact(a - b + k) * few_fact(l - a - k));
        tot += ((a - b + k) & 1) ? -term : term;
    }
    double d = sqrt(few_fact(l + a) * few_fact(l - a) * few_fact(l + b) * few_fact(l - b)) * tot;
    double v = sqrt((2.0 * l + 1.0) / (4.0 * 3.14159265358979323846)) * d;   // (-1)^s = +1
    *re = v * cos(m * phi);
    *im = v * sin(m * phi);
}

extern "C" int few_ylm(int l, int m, double theta, double phi, double* out_host)
{
    FEW_REQUIRE(out_host != nullptr, FEW_ERR_INVALID_ARG, "out is NULL");
    FEW_REQUIRE(l >= 2 && l <= FEW_MAX_L && m <= l && m >= -l, FEW_ERR_BAD_MODE, "need 2 <= l <= FEW_MAX_L and |m| <= l");
    few_ylm_m2(l, m, theta, phi, &out_host[0], &out_host[1]);
    return FEW_OK;
}

// One block per source.  The harmonics depend on (l, m) only -- 117 values for l <= 10 against 3843 modes -- so the block
// first tabulates -2Y_{l,m} for 2 <= l <= max l, |m| <= l in shared memory (one thread per entry, reading factorials and the
// powers of cos(theta/2), sin(theta/2) from small shared tables built in parallel) and every mode looks its two values up.
// Same sum, same operation order as few_ylm_m2.
constexpr int kYlmThreads = 1024;
constexpr int kYlmPow = 2 * FEW_MAX_L + 3;       // powers 0 .. 2l + 2
__host__ __device__ static inline int few_ylm_slot(int l, int m) { return l * l - 4 + m + l; }   // l >= 2, |m| <= l

__global__ void __launch_bounds__(kYlmThreads)
few_ylm_modes_kernel(const double* __restrict__ theta, const double* __restrict__ phi,
                     const int* __restrict__ l, const int* __restrict__ m, int n_src, int n_modes,
                     double2* __restrict__ ylm_plus, double2* __restrict__ ylm_minus, int* status)
{
    extern __shared__ double2 ylm_table[];
    __shared__ double fact_s[kYlmPow], chp[kYlmPow], shp[kYlmPow];
    __shared__ int lmax_s;
    const int s = blockIdx.x, tid = threadIdx.x;
    if (tid == 0) lmax_s = 2;
    const double th = theta[s], ph = phi[s];
    if (tid < kYlmPow) fact_s[tid] = few_fact(tid);
    else if (tid < 2 * kYlmPow) chp[tid - kYlmPow] = few_ipow(cos(0.5 * th), tid - kYlmPow);
    else if (tid < 3 * kYlmPow) shp[tid - 2 * kYlmPow] = few_ipow(sin(0.5 * th), tid - 2 * kYlmPow);
    __syncthreads();
    int lm = 2;
    bool bad = false;
    for (int j = tid; j < n_modes; j += kYlmThreads) {
        const int lj = l[j], mj = m[j];
        if (lj < 2 || lj > FEW_MAX_L || mj < 0 || mj > lj) bad = true; else lm = lj > lm ? lj : lm;
    }
    if (bad) atomicOr(status, FEW_DEV_BAD_MODE);
    lm = __reduce_max_sync(0xffffffffu, lm);
    if ((tid & 31) == 0 && lm > 2) atomicMax(&lmax_s, lm);
    __syncthreads();
    const int lmax = lmax_s, n_tab = (lmax + 1) * (lmax + 1) - 4;
    for (int idx = tid; idx < n_tab; idx += kYlmThreads) {
        int ll = (int)sqrt((double)(idx + 4));
        while (ll * ll > idx + 4) --ll;
        while ((ll + 1) * (ll + 1) <= idx + 4) ++ll;
        const int mm = idx - (ll * ll - 4) - ll;
        const int a = mm, b = 2;
        const int k0 = (b - a) > 0 ? (b - a) : 0, k1 = (ll + b) < (ll - a) ? (ll + b) : (ll - a);
        double tot = 0.0;
        for (int k = k0; k <= k1; ++k) {
            const double term = chp[2 * ll + b - a - 2 * k] * shp[a - b + 2 * k] /
                                (fact_s[ll + b - k] * fact_s[k] * fact_s[a - b + k] * fact_s[ll - a - k]);
            tot += ((a - b + k) & 1) ? -term : term;
        }
        const double d = sqrt(fact_s[ll + a] * fact_s[ll - a] * fact_s[ll + b] * fact_s[ll - b]) * tot;
        const double v = sqrt((2.0 * ll + 1.0) / (4.0 * 3.14159265358979323846)) * d;
        ylm_table[idx] = make_double2(v * cos(mm * ph), v * sin(mm * ph));
    }
    __syncthreads();
    for (int j = tid; j < n_modes; j += kYlmThreads) {
        const int lj = l[j], mj = m[j];
        double2 yp = make_double2(0.0, 0.0), ym = yp;
        if (!(lj < 2 || lj > FEW_MAX_L || mj < 0 || mj > lj)) { yp = ylm_table[few_ylm_slot(lj, mj)]; ym = ylm_table[few_ylm_slot(lj, -mj)]; }
        ylm_plus[(size_t)s * n_modes + j] = yp;
        ylm_minus[(size_t)s * n_modes + j] = ym;
    }
}

extern "C" int few_ylm_modes(few_ctx* ctx, const double* theta, const double* phi, const int* l, const int* m,
                             int n_src, int n_modes, double* ylm_plus, double* ylm_minus, void* stream)
{
    FEW_REQUIRE(ctx && theta && phi && l && m && ylm_plus && ylm_minus, FEW_ERR_INVALID_ARG, "NULL argument");
    FEW_REQUIRE(n_src > 0 && n_modes > 0, FEW_ERR_INVALID_ARG, "n_src and n_modes must be positive");
    const size_t smem = (size_t)((FEW_MAX_L + 1) * (FEW_MAX_L + 1) - 4) * sizeof(double2);
    FEW_CUDA_CHECK(cudaFuncSetAttribute(few_ylm_modes_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    few_ylm_modes_kernel<<<n_src, kYlmThreads, smem, (cudaStream_t)stream>>>(theta, phi, l, m, n_src, n_modes, (double2*)ylm_plus,
                                                                           (double2*)ylm_minus, ctx->d_status);
    FEW_LAUNCHED(ctx);
    return FEW_OK;
}
