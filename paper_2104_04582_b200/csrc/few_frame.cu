// few_frame.cu -- the two steps that follow the summation in the paper's pipeline:
//
//  * Detector (solar-system-barycentre) frame, sec. II A, Eq. (4)-(8), and the mu/d_L prefactor of Eq. (10):
//    "Following the summation, the frame transformation is performed".  The transformation is one complex
//    constant per source,  h_SSB = -(mu/d_L) e^{2 i psi} h(theta_src, phi_src = -pi/2)  (R22), so the product path
//    never runs it as a pass over h: few_frame_constants hands (theta_src, phi_src) to the harmonics and the factor to the
//    summation's plan kernel, which folds it into the per-mode harmonic constants.  few_frame_rotate is the separate
//    elementwise pass (what the paper's pipeline does), kept as an entry point for waveforms that already exist and as the
//    unfused baseline the fusion is measured against.
//
//  * Inner products with the PSD set to 1, Eq. (15)-(17): <a|b> = 2 dt Re sum_i conj(a_i) b_i (Parseval,
//    both polarisations, R23).  The product path reduces them inside the summation kernel (few_sum_waveform_ex);
//    few_inner_products is the separate two-pass reduction over stored series (data against data, or the unfused baseline).
#include <math.h>
#include <mutex>
#include "few_common.cuh"

namespace {

// One thread per source.  Eq. (4), (5): R, S from the sky and spin angles; cos(theta_src) = -R.S is taken
// together with sin(theta_src) = |R x S| through atan2, which is well conditioned at every angle (acos is not near the poles);
// Eq. (8) gives tan(psi) = N/D, and only cos(2 psi) = (D^2 - N^2)/(D^2 + N^2), sin(2 psi) = 2 N D/(D^2 + N^2) are needed, so
// no inverse trigonometric function enters the factor at all.  N = D = 0 (spin along the line of sight): psi = 0.
__global__ void few_frame_constants_kernel(const double* __restrict__ sky, const double* __restrict__ mu_over_dl, int n_src,
                                           double* __restrict__ theta, double* __restrict__ phi, double2* __restrict__ factor)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n_src) return;
    const double qS = sky[4 * s], pS = sky[4 * s + 1], qK = sky[4 * s + 2], pK = sky[4 * s + 3];
    double sqS, cqS, spS, cpS, sqK, cqK, spK, cpK, sd, cd;
    sincos(qS, &sqS, &cqS); sincos(pS, &spS, &cpS); sincos(qK, &sqK, &cqK); sincos(pK, &spK, &cpK);
    sincos(pS - pK, &sd, &cd);
    const double R[3] = {sqS * cpS, sqS * spS, cqS}, S[3] = {sqK * cpK, sqK * spK, cqK};
    const double dot = R[0] * S[0] + R[1] * S[1] + R[2] * S[2];
    const double cx = R[1] * S[2] - R[2] * S[1], cy = R[2] * S[0] - R[0] * S[2], cz = R[0] * S[1] - R[1] * S[0];
    theta[s] = atan2(sqrt(cx * cx + cy * cy + cz * cz), -dot);
    phi[s] = -1.57079632679489661923;
    const double N = cqS * sqK * cd - sqS * cqK, D = sqK * sd;
    const double n2 = N * N + D * D;
    double c2 = 1.0, s2 = 0.0;
    if (n2 > 0.0) { c2 = (D - N) * (D + N) / n2; s2 = 2.0 * N * D / n2; }
    const double a = mu_over_dl ? mu_over_dl[s] : 1.0;
    factor[s] = make_double2(-a * c2, -a * s2);
}

// h_out = factor[src] * h_in: 16 B read + 16 B written per sample, two samples in flight per thread.
__global__ void __launch_bounds__(256)
few_frame_rotate_kernel(const double2* __restrict__ h_in, const double2* __restrict__ factor, long long n_samples,
                        double2* __restrict__ h_out)
{
    const int src = blockIdx.y;
    const double2 f = factor[src];
    const double2* in = h_in + (size_t)src * n_samples;
    double2* out = h_out + (size_t)src * n_samples;
    const long long stride = (long long)gridDim.x * blockDim.x;
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    for (; i + stride < n_samples; i += 2 * stride) {
        const double2 a = __ldcs(&in[i]), b = __ldcs(&in[i + stride]);
        __stcs(&out[i], make_double2(f.x * a.x - f.y * a.y, f.x * a.y + f.y * a.x));
        __stcs(&out[i + stride], make_double2(f.x * b.x - f.y * b.y, f.x * b.y + f.y * b.x));
    }
    if (i < n_samples) {
        const double2 a = __ldcs(&in[i]);
        __stcs(&out[i], make_double2(f.x * a.x - f.y * a.y, f.x * a.y + f.y * a.x));
    }
}

// ---- standalone inner products: per-chunk partials (fixed chunk -> block mapping), then one block per source adds the chunks
// in a fixed order.  Same answer every run.
constexpr int kIpThreads = 256;
constexpr int kIpChunk = kIpThreads * 8;       // samples per block

__global__ void __launch_bounds__(kIpThreads)
few_inner_partial_kernel(const double2* __restrict__ d_all, const double2* __restrict__ h_all, long long n_samples, int n_chunks,
                         double* __restrict__ partial)
{
    __shared__ double red[3][kIpThreads / 32];
    const int src = blockIdx.y, chunk = blockIdx.x, tid = threadIdx.x;
    const double2* d = d_all + (size_t)src * n_samples;
    const double2* h = h_all + (size_t)src * n_samples;
    const long long base = (long long)chunk * kIpChunk;
    double a = 0.0, b = 0.0, c = 0.0;
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const long long i = base + r * kIpThreads + tid;
        if (i < n_samples) {
            const double2 dv = __ldcs(&d[i]), hv = __ldcs(&h[i]);
            a = fma(dv.x, hv.x, fma(dv.y, hv.y, a));
            b = fma(dv.x, hv.y, fma(-dv.y, hv.x, b));
            c = fma(hv.x, hv.x, fma(hv.y, hv.y, c));
        }
    }
    for (int o = 16; o; o >>= 1) {
        a += __shfl_xor_sync(0xffffffffu, a, o); b += __shfl_xor_sync(0xffffffffu, b, o); c += __shfl_xor_sync(0xffffffffu, c, o);
    }
    if ((tid & 31) == 0) { red[0][tid >> 5] = a; red[1][tid >> 5] = b; red[2][tid >> 5] = c; }
    __syncthreads();
    if (tid < 3) {
        double v = 0.0;
        for (int w = 0; w < kIpThreads / 32; ++w) v += red[tid][w];
        partial[((size_t)src * n_chunks + chunk) * 4 + tid] = v;
    }
}

__global__ void __launch_bounds__(kIpThreads)
few_inner_final_kernel(const double* __restrict__ partial, int n_chunks, double dt, double* __restrict__ inner)
{
    __shared__ double red[3][kIpThreads / 32];
    const int src = blockIdx.x, tid = threadIdx.x;
    const double* P = partial + (size_t)src * n_chunks * 4;
    double a = 0.0, b = 0.0, c = 0.0;
    for (int q = tid; q < n_chunks; q += kIpThreads) { a += P[4 * (size_t)q]; b += P[4 * (size_t)q + 1]; c += P[4 * (size_t)q + 2]; }
    for (int o = 16; o; o >>= 1) {
        a += __shfl_xor_sync(0xffffffffu, a, o); b += __shfl_xor_sync(0xffffffffu, b, o); c += __shfl_xor_sync(0xffffffffu, c, o);
    }
    if ((tid & 31) == 0) { red[0][tid >> 5] = a; red[1][tid >> 5] = b; red[2][tid >> 5] = c; }
    __syncthreads();
    if (tid < 3) {
        double v = 0.0;
        for (int w = 0; w < kIpThreads / 32; ++w) v += red[tid][w];
        inner[(size_t)src * 3 + tid] = 2.0 * dt * v;
    }
}

inline long long ip_chunks(long long n_samples) { return (n_samples + kIpChunk - 1) / kIpChunk; }

}  // namespace

extern "C" int few_frame_constants(few_ctx* ctx, const double* sky, const double* mu_over_dl, int n_src,
                                   double* theta, double* phi, double* factor, void* stream)
{
    FEW_REQUIRE(ctx && sky && theta && phi && factor, FEW_ERR_INVALID_ARG, "NULL argument");
    FEW_REQUIRE(n_src > 0, FEW_ERR_INVALID_ARG, "n_src must be positive");
    few_frame_constants_kernel<<<(n_src + 127) / 128, 128, 0, (cudaStream_t)stream>>>(sky, mu_over_dl, n_src, theta, phi, (double2*)factor);
    FEW_LAUNCHED(ctx);
    return FEW_OK;
}

extern "C" int few_frame_rotate(few_ctx* ctx, const double* h_in, const double* factor, int n_src, long long n_samples,
                                double* h_out, void* stream)
{
    FEW_REQUIRE(ctx && factor, FEW_ERR_INVALID_ARG, "NULL argument");
    FEW_REQUIRE(n_src > 0 && n_src <= 65535 && n_samples >= 0, FEW_ERR_INVALID_ARG, "bad sizes");
    if (n_samples == 0) return FEW_OK;
    FEW_REQUIRE(h_in && h_out, FEW_ERR_INVALID_ARG, "h_in or h_out is NULL");
    long long per_src = (n_samples + 2 * 256 - 1) / (2 * 256);
    const long long cap = (long long)ctx->sm_count * 8;             // 8 resident blocks per SM cover the machine; more only adds tails
    if ((long long)n_src * per_src > cap) per_src = cap / n_src > 1 ? cap / n_src : 1;
    few_frame_rotate_kernel<<<dim3((unsigned)per_src, n_src), 256, 0, (cudaStream_t)stream>>>((const double2*)h_in, (const double2*)factor,
                                                                                           n_samples, (double2*)h_out);
    FEW_LAUNCHED(ctx);
    return FEW_OK;
}

extern "C" size_t few_inner_products_workspace(int n_src, long long n_samples)
{
    if (n_src <= 0 || n_samples < 0) return 0;
    return few_align_up((size_t)n_src * (size_t)(ip_chunks(n_samples) > 0 ? ip_chunks(n_samples) : 1) * 4 * sizeof(double));
}

extern "C" int few_inner_products(few_ctx* ctx, const double* d, const double* h, int n_src, long long n_samples, double dt,
                                  double* inner, void* workspace, size_t workspace_bytes, void* stream)
{
    FEW_REQUIRE(ctx && inner, FEW_ERR_INVALID_ARG, "NULL argument");
    FEW_REQUIRE(n_src > 0 && n_src <= 65535 && n_samples >= 0, FEW_ERR_INVALID_ARG, "bad sizes");
    FEW_REQUIRE(dt > 0.0 && isfinite(dt), FEW_ERR_INVALID_ARG, "dt must be positive and finite");
    cudaStream_t st = (cudaStream_t)stream;
    if (n_samples == 0) { FEW_CUDA_CHECK(cudaMemsetAsync(inner, 0, (size_t)n_src * 3 * sizeof(double), st)); return FEW_OK; }
    FEW_REQUIRE(d && h, FEW_ERR_INVALID_ARG, "d or h is NULL");
    FEW_REQUIRE(workspace && ((uintptr_t)workspace % 256) == 0 && workspace_bytes >= few_inner_products_workspace(n_src, n_samples),
                FEW_ERR_WORKSPACE, "workspace NULL, misaligned or too small");
    const long long nc = ip_chunks(n_samples);
    FEW_REQUIRE(nc < 2147483647LL, FEW_ERR_LIMIT, "n_samples too large");
    few_inner_partial_kernel<<<dim3((unsigned)nc, n_src), kIpThreads, 0, st>>>((const double2*)d, (const double2*)h, n_samples, (int)nc,
                                                                             (double*)workspace);
    FEW_LAUNCHED(ctx);
    few_inner_final_kernel<<<n_src, kIpThreads, 0, st>>>((const double*)workspace, (int)nc, dt, inner);
    FEW_LAUNCHED(ctx);
    return FEW_OK;
}

// ---- few_inner_products_static: the same two kernels, with the per-chunk partial sums kept in memory that is part of the
// loaded library image instead of a workspace somebody had to allocate.
//
// Who this is for.  few_inner_products needs a workspace, and a workspace has to come from an allocator.  Some host programs
// are not allowed to run one at the point where they want <d|h> and <h|h>: code inside a region where the CUDA runtime refuses
// allocation calls, a sampler whose device memory was handed in full to a pool it may not grow, a plug-in that receives device
// pointers from its host application and owns no allocator of its own.  Such a caller passes d, h and inner (which it already
// has) and nothing else; this function calls no cudaMalloc / cudaFree and no library routine that allocates.
//
// The scratch array below lives in every GPU context that loads libfew_b200.so, from module load until the process exits,
// whether or not this entry point is ever called: kIpStaticMaxChunks x 4 doubles = 512 KB per GPU.  That is the price, and the
// reason the limit is modest.
//
// In HOST code the identifier few_ip_static_scratch is only a handle for the runtime (its host address means nothing to the
// GPU), so the address the kernels get is looked up with cudaGetSymbolAddress -- once per device, with that device current, on
// the first call made on that device -- and kept in g_ip_static_ptr.
constexpr int kIpStaticMaxChunks = FEW_INNER_STATIC_MAX_CHUNKS;
constexpr int kIpStaticMaxDevices = 64;

static __device__ __align__(256) double few_ip_static_scratch[(size_t)kIpStaticMaxChunks * 4];

namespace {
std::mutex g_ip_static_lock;
double* g_ip_static_ptr[kIpStaticMaxDevices];   // device address of few_ip_static_scratch on device i; NULL = not looked up yet
}  // namespace

extern "C" int few_inner_products_static(few_ctx* ctx, const double* d, const double* h, int n_src, long long n_samples, double dt,
                                         double* inner, void* stream)
{
    FEW_REQUIRE(inner, FEW_ERR_INVALID_ARG, "inner is NULL");
    FEW_REQUIRE(n_src > 0 && n_src <= 65535 && n_samples >= 0, FEW_ERR_INVALID_ARG, "bad sizes");
    FEW_REQUIRE(dt > 0.0 && isfinite(dt), FEW_ERR_INVALID_ARG, "dt must be positive and finite");
    const long long nc = ip_chunks(n_samples);
    FEW_REQUIRE(nc <= kIpStaticMaxChunks && (long long)n_src * nc <= kIpStaticMaxChunks, FEW_ERR_LIMIT,
                "n_src * ceil(n_samples / 2048) exceeds FEW_INNER_STATIC_MAX_CHUNKS: the built-in scratch array is too small for "
                "this call; use few_inner_products with a caller-owned workspace");
    cudaStream_t st = (cudaStream_t)stream;
    if (n_samples == 0) { FEW_CUDA_CHECK(cudaMemsetAsync(inner, 0, (size_t)n_src * 3 * sizeof(double), st)); return FEW_OK; }
    FEW_REQUIRE(d && h, FEW_ERR_INVALID_ARG, "d or h is NULL");

    int dev = -1;
    FEW_CUDA_CHECK(cudaGetDevice(&dev));
    FEW_REQUIRE(dev >= 0 && dev < kIpStaticMaxDevices, FEW_ERR_LIMIT, "device ordinal beyond the 64 this entry point keeps an address for");
    FEW_REQUIRE(!ctx || ctx->device == dev, FEW_ERR_INVALID_ARG, "ctx belongs to another device than the current one");
    double* scratch;
    {
        std::lock_guard<std::mutex> guard(g_ip_static_lock);
        if (!g_ip_static_ptr[dev]) {   // first call on this device: ask the runtime where this device's copy of the array is
            void* p = nullptr;
            FEW_CUDA_CHECK(cudaGetSymbolAddress(&p, few_ip_static_scratch));
            FEW_REQUIRE(p, FEW_ERR_CUDA, "cudaGetSymbolAddress returned a NULL address");
            g_ip_static_ptr[dev] = static_cast<double*>(p);
        }
        scratch = g_ip_static_ptr[dev];
    }
    // Nothing in the array has to start at zero: the first kernel stores (never accumulates into) the slots [src][chunk][0..2] for
    // every chunk of this call, and the second kernel reads exactly those slots, behind it on the same stream.  Whatever an
    // earlier call left in the array is either overwritten or never looked at.
    few_inner_partial_kernel<<<dim3((unsigned)nc, n_src), kIpThreads, 0, st>>>((const double2*)d, (const double2*)h, n_samples, (int)nc,
                                                                             scratch);
    if (ctx) ++ctx->launches;
    FEW_CUDA_CHECK(cudaGetLastError());
    few_inner_final_kernel<<<n_src, kIpThreads, 0, st>>>(scratch, (int)nc, dt, inner);
    if (ctx) ++ctx->launches;
    FEW_CUDA_CHECK(cudaGetLastError());
    return FEW_OK;
}
