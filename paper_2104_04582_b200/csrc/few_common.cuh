// few_common.cuh -- internal helpers of libfew_b200 (not part of the ABI, not shared with oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include "few.h"

constexpr int kHostGroups = 8;   // few_waveform_host: source groups whose input copies overlap earlier groups' kernels

struct few_ctx {
    int device;
    int sm_count;
    int smem_optin;      // max dynamic shared memory per block (bytes)
    int* d_status;       // device status word (FEW_DEV_* bits)
    int profile;         // few_profile_enable
    int profile_valid;   // a sum kernel was bracketed since profiling was switched on
    long long launches;  // kernels launched through this context so far (few_launch_count)
    int max_steps;       // few_set_max_steps: caller's bound on the summation's steps per source (0 = the default capacity)
    cudaEvent_t ev_sum[2];
    cudaStream_t side[2];  // few_waveform: the two spline fits run beside harmonics + mode selection
    cudaEvent_t ev_fork, ev_join[2];
    void* host_arena;      // few_waveform_host: grow-only device arena (inputs, h, workspace), freed by few_destroy
    size_t host_arena_bytes;
    void* host_stage;      // few_waveform_host: pinned staging block for the small inputs (one host->device copy instead of eight)
    size_t host_stage_bytes;
    cudaStream_t host_stream, copy_stream;   // few_waveform_host: kernels / host->device copies
    cudaEvent_t ev_group[8];                 // inputs of source group g have landed
};

void few_set_error(const char* fmt, ...);

// few_sum.cu: every size limit of the summation (tile count, shared memory of its kernels) in one place, so that the summation,
// few_waveform and few_waveform_host can all check them BEFORE they enqueue anything.  FEW_OK or FEW_ERR_LIMIT.
int few_sum_check_limits(const few_ctx* ctx, int n_src, int n_t, int n_modes, long long n_samples, int n_phase);

#define FEW_CUDA_CHECK(expr)                                                                     \
    do {                                                                                         \
        cudaError_t _e = (expr);                                                                 \
        if (_e != cudaSuccess) {                                                                 \
            few_set_error("%s failed at %s:%d: %s", #expr, __FILE__, __LINE__, cudaGetErrorString(_e)); \
            return FEW_ERR_CUDA;                                                                 \
        }                                                                                        \
    } while (0)

// after every kernel launch: count it (few_launch_count) and pick up a launch error
#define FEW_LAUNCHED(ctx)                                                                        \
    do {                                                                                         \
        ++(ctx)->launches;                                                                       \
        FEW_CUDA_CHECK(cudaGetLastError());                                                      \
    } while (0)

#define FEW_REQUIRE(cond, code, msg)                                                             \
    do {                                                                                         \
        if (!(cond)) { few_set_error("%s: %s", __func__, msg); return (code); }                  \
    } while (0)

static inline size_t few_align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

// Knot count of a source.  Uniform batches pass n_t_src == NULL: every source has n_t knots.  Ragged batches (the *_ragged
// entry points) keep the padded [n_src][n_t] layouts and give each source's own count; one outside [4, n_t] is reported
// (FEW_DEV_BAD_COUNT) and replaced by 4 (the first four rows exist for every source), so that no kernel reads the padding or
// anything outside the arrays.
__device__ __forceinline__ int few_knots(const int* __restrict__ n_t_src, int src, int n_t, int* status)
{
    if (!n_t_src) return n_t;
    int v = n_t_src[src];
    if (v < 4 || v > n_t) { atomicOr(status, FEW_DEV_BAD_COUNT); v = n_t < 4 ? n_t : 4; }
    return v;
}

// Carves consecutive 256-byte-aligned sub-buffers out of a caller-owned workspace.
struct few_carver {
    char* base; size_t off;
    explicit few_carver(void* p) : base(static_cast<char*>(p)), off(0) {}
    template <class T> T* take(size_t count) { T* r = reinterpret_cast<T*>(base + off); off += few_align_up(count * sizeof(T)); return r; }
};

// ------------------------------------------------------------------------------------------------
// double-double arithmetic (error-free transformations with FMA).  A value is hi + lo, |lo| <= ulp(hi)/2.
// ------------------------------------------------------------------------------------------------
struct dd { double hi, lo; };

__device__ __forceinline__ dd dd_make(double hi, double lo = 0.0) { dd r; r.hi = hi; r.lo = lo; return r; }
__device__ __forceinline__ dd two_sum(double a, double b)
{
    double s = __dadd_rn(a, b), bb = __dsub_rn(s, a);
    double e = __dadd_rn(__dsub_rn(a, __dsub_rn(s, bb)), __dsub_rn(b, bb));
    return dd_make(s, e);
}
__device__ __forceinline__ dd quick_two_sum(double a, double b)   // requires |a| >= |b|
{
    double s = __dadd_rn(a, b);
    return dd_make(s, __dsub_rn(b, __dsub_rn(s, a)));
}
__device__ __forceinline__ dd two_prod(double a, double b)
{
    double p = __dmul_rn(a, b);
    return dd_make(p, __fma_rn(a, b, -p));
}
__device__ __forceinline__ dd dd_add(dd a, dd b)
{
    dd s = two_sum(a.hi, b.hi), t = two_sum(a.lo, b.lo);
    s.lo = __dadd_rn(s.lo, t.hi);
    s = quick_two_sum(s.hi, s.lo);
    s.lo = __dadd_rn(s.lo, t.lo);
    return quick_two_sum(s.hi, s.lo);
}
__device__ __forceinline__ dd dd_neg(dd a) { return dd_make(-a.hi, -a.lo); }
__device__ __forceinline__ dd dd_sub(dd a, dd b) { return dd_add(a, dd_neg(b)); }
__device__ __forceinline__ dd dd_add_d(dd a, double b)
{
    dd s = two_sum(a.hi, b);
    s.lo = __dadd_rn(s.lo, a.lo);
    return quick_two_sum(s.hi, s.lo);
}
__device__ __forceinline__ dd dd_mul_d(dd a, double b)
{
    dd p = two_prod(a.hi, b);
    p.lo = __fma_rn(a.lo, b, p.lo);
    return quick_two_sum(p.hi, p.lo);
}
__device__ __forceinline__ dd dd_mul(dd a, dd b)
{
    dd p = two_prod(a.hi, b.hi);
    p.lo = __dadd_rn(p.lo, __fma_rn(a.hi, b.lo, __dmul_rn(a.lo, b.hi)));
    return quick_two_sum(p.hi, p.lo);
}
__device__ __forceinline__ dd dd_div(dd a, dd b)   // two Newton-style correction steps on the quotient
{
    double q1 = __ddiv_rn(a.hi, b.hi);
    dd r = dd_sub(a, dd_mul_d(b, q1));
    double q2 = __ddiv_rn(r.hi, b.hi);
    r = dd_sub(r, dd_mul_d(b, q2));
    double q3 = __ddiv_rn(r.hi, b.hi);
    dd q = quick_two_sum(q1, q2);
    return dd_add_d(q, q3);
}
__device__ __forceinline__ dd dd_from_diff(double a, double b) { return two_sum(a, -b); }  // a - b exactly
