// few_sum.cu -- S3: the interpolated summation (sec. III C, Eq. (9), Eq. (10)):
//   "the actual summation kernel evaluates the spline at the sampling rate of the output data stream.  Then, the output
//    phase and amplitude values are combined within each mode according to Eq. (1) ... A_{l,-m,-k,-n} = (-1)^{l+k} A*_{lmkn}
//    ... only compute modes for m >= 0 ... the modes in a single time step are combined."
//   h(t_i) = scale * sum_{j kept} [ Y+_j W_j + (m_j>0) (-1)^{l_j} Y-_j conj(W_j) ],  W_j = A_j(t_i) exp(-i(m_j Phi_phi + n_j Phi_r)).
//
// Algebra used (exact): with E = exp(-i theta) = e_r + i e_i and Ybar = (-1)^l Y- (0 for m = 0),
//   Y+ A E + Ybar conj(A) conj(E) = e_r U + e_i V,   U = Y+ A + Ybar conj(A),   V = i (Y+ A - Ybar conj(A)).
// U and V are linear in A's spline coefficients, and E depends on (m, n) only, so all kept l of one (m, n) PAIR are summed
// into one pair of complex cubics (U_mn, V_mn) per sparse segment BEFORE the sample loop.  The hot loop then costs, per
// sample and pair, 12 DFMA (two complex cubic Horners) + 4 DFMA (h += e_r U + e_i V) + 4 (E *= Z_r), with no per-l state.
//
// Three launches per call, all on the caller's stream, nothing read back to the host:
//   1. few_sum_plan_kernel  (one block per source): clips the dense sample grid to the sparse segments and prefix-sums
//        the per-segment tile counts (every block of the sum kernel works inside ONE segment, so its coefficients are
//        block-uniform); orders the kept modes by (m, sign n, |n|, l), finds the pairs and describes how E_mn = Z_phi^m Z_r^n
//        is reached from the previous pair (walking n upward from 0 with Z_r, then downward with conj Z_r).
//   2. few_sum_pack_kernel  (one block per source and segment): forms (U_mn, V_mn) from the kept modes' spline coefficients
//        and Y+, Ybar, scale, and writes them as a stream of 4 KB stages (30 pairs x 128 B + 30 descriptors).
//   3. few_sum_kernel       the hot loop.  Stages arrive in shared memory through a ring of TMA bulk copies
//        (cp.async.bulk + mbarrier) and are read with 128-bit broadcast loads.  Each thread owns R samples in registers;
//        per sample the two phases are evaluated ONCE in double-double (Horner, reduction by 2 pi, one sincos each).
//        Output: coalesced 16-byte streaming stores.
// FP64 pipe only: per-sample elementwise work with a reduction over modes, not a dense contraction.
#include "few_common.cuh"

namespace {

constexpr int kPlanThreads = 1024;
constexpr int kPlanSmemElems = 16384;         // 128 KB of (key, mode) words: the plan kernel's in-shared-memory sort capacity
constexpr int kSumThreads = 128;
#ifndef FEW_SUM_R
#define FEW_SUM_R 4
#define FEW_SUM_BPS 3
#endif
constexpr int kSumR = FEW_SUM_R;              // samples per thread
constexpr int kSumBlocksPerSm = FEW_SUM_BPS;  // resident blocks per SM (register budget 65536 / (128 * blocks))
constexpr int kTile = kSumThreads * kSumR;    // samples per block
constexpr int kStagePairs = 30;               // pairs per stage
constexpr int kStageBytes = 4096;             // 30 * 128 B of coefficients + 64 ints of header
constexpr int kStageD2 = kStageBytes / 16;    // stage size in double2
constexpr int kRing = 4;                      // stages in flight per block

// pair descriptor: bit 0 = special (anything but "advance E by one step"); then
constexpr int kAdvShift = 1, kAdvBits = 12;   // number of E steps before this pair
constexpr int kNewSub = 1 << 13;              // restart E from Z_phi^m (n changes sign or m changes)
constexpr int kDirNeg = 1 << 14;              // walk with conj(Z_r)
constexpr int kDmShift = 15, kDmBits = 7;     // m increment of a new run
constexpr int kNewRun = 1 << 22;               // new (m, k) run
constexpr int kKShift = 23, kKBits = 7;       // polar index of the run, offset by 64 (Kerr-shaped lists, |k| <= FEW_MAX_ABS_K)

struct sum_layout {
    long long* bounds;   // [n_src][n_t + 2]   pseudo-segment p covers samples [bounds[p], bounds[p+1])
    int* tile_start;     // [n_src][n_t + 2]   exclusive prefix of tiles per pseudo-segment; last = total
    int* n_groups;       // [n_src]            number of (m, n) pairs
    int* tile_counter;   // [1]                dynamic tile scheduler of the persistent sum kernel
    int* desc;           // [n_src][n_modes]   pair descriptors
    int* g_first;        // [n_src][n_modes+1] first sorted mode of each pair
    int* order_j;        // [n_src][n_modes]   mode index of sorted position r
    double* yfold;       // [n_src][n_modes][4] scale * (Y+ re, Y+ im, Ybar re, Ybar im) of sorted position r
    double* pack;        // [n_src][n_t - 1][max_stages][kStageBytes / 8]
    double* partial;     // [n_src][max_tiles][4]  per-tile sums of conj(d) h (re, im) and |h|^2 (fused inner products)
    unsigned long long* sortbuf;   // [n_src][sort_pow2] plan-kernel sort array when the mode list exceeds shared memory (else empty)
    int sort_pow2;
    int max_stages;
    int max_tiles;
};

__host__ __device__ inline int stages_for(int n_pairs) { return (n_pairs + kStagePairs - 1) / kStagePairs; }

__host__ inline long long sum_max_tiles(long long n_samples, int n_t) { return (n_samples + kTile - 1) / kTile + n_t + 1; }

sum_layout sum_carve(void* ws, int n_src, int n_t, int n_modes, long long n_samples, size_t* bytes = nullptr)
{
    few_carver c(ws);
    sum_layout L;
    L.max_stages = stages_for(n_modes);
    L.bounds = c.take<long long>((size_t)n_src * (n_t + 2));
    L.tile_start = c.take<int>((size_t)n_src * (n_t + 2));
    L.n_groups = c.take<int>(n_src);
    L.tile_counter = c.take<int>(1);
    L.desc = c.take<int>((size_t)n_src * n_modes);
    L.g_first = c.take<int>((size_t)n_src * (n_modes + 1));
    L.order_j = c.take<int>((size_t)n_src * n_modes);
    L.yfold = c.take<double>((size_t)n_src * n_modes * 4);
    L.pack = c.take<double>((size_t)n_src * (n_t - 1) * L.max_stages * (kStageBytes / 8));
    const long long mt = sum_max_tiles(n_samples, n_t);
    L.max_tiles = (int)(mt < 2147483647LL ? mt : 2147483647LL);
    L.partial = c.take<double>((size_t)n_src * (size_t)mt * 4);
    int p2 = 1;
    while (p2 < n_modes) p2 <<= 1;
    L.sort_pow2 = p2 > kPlanSmemElems ? p2 : 0;
    L.sortbuf = c.take<unsigned long long>((size_t)n_src * L.sort_pow2);
    if (bytes) *bytes = c.off;
    return L;
}

// t_i = t0 + i*dt with the product and the sum rounded separately (R14).
__device__ __forceinline__ double sample_time(double t0, double dt, long long i) { return __dadd_rn(t0, __dmul_rn((double)i, dt)); }

__device__ long long first_index(double tk, double t0, double dt, long long N, bool strict)
{
    // smallest i in [0, N] with t_i >= tk (strict: t_i > tk); t_i is non-decreasing in i for dt > 0
    double x = (tk - t0) / dt;
    long long i = !(x > 0.0) ? 0 : (x >= (double)N ? N : (long long)ceil(x));
    if (strict) {
        while (i > 0 && sample_time(t0, dt, i - 1) > tk) --i;
        while (i < N && !(sample_time(t0, dt, i) > tk)) ++i;
    } else {
        while (i > 0 && sample_time(t0, dt, i - 1) >= tk) --i;
        while (i < N && sample_time(t0, dt, i) < tk) ++i;
    }
    return i;
}

__device__ __forceinline__ int plan_block_scan(int v, int* warp_sums, int* total)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int o = 1; o < 32; o <<= 1) { int u = __shfl_up_sync(0xffffffffu, v, o); if (lane >= o) v += u; }
    if (lane == 31) warp_sums[wid] = v;
    __syncthreads();
    if (wid == 0) {
        int s = warp_sums[lane];
        for (int o = 1; o < 32; o <<= 1) { int u = __shfl_up_sync(0xffffffffu, s, o); if (lane >= o) s += u; }
        warp_sums[lane] = s;
    }
    __syncthreads();
    int res = v + (wid ? warp_sums[wid - 1] : 0);
    *total = warp_sums[kPlanThreads / 32 - 1];
    __syncthreads();
    return res;
}

// sort key: m | k + 64 | sign(n) | |n| | l  (ascending): runs of equal (m, k), inside them n = 0, 1, 2, ... then -1, -2, ...
__device__ __forceinline__ int key_m(unsigned k) { return (int)(k >> 25); }
__device__ __forceinline__ int key_k(unsigned k) { return (int)((k >> 18) & 0x7f) - 64; }
__device__ __forceinline__ unsigned key_run(unsigned k) { return k >> 18; }
__device__ __forceinline__ int key_dir(unsigned k) { return (int)(k >> 17) & 1; }
__device__ __forceinline__ int key_absn(unsigned k) { return (int)(k >> 5) & 0xfff; }
__device__ __forceinline__ int key_l(unsigned k) { return (int)(k & 0x1f); }

// Bitonic compare-exchange steps on buf[0, n) (n a power of two), which holds elements [c0, c0 + n) of the whole array: for
// size = size_first, 2 size_first, ..., size_last the strides min(size, n)/2 ... 1.  Direction from the GLOBAL index.
__device__ void plan_bitonic_steps(unsigned long long* buf, int c0, int n, int size_first, int size_last)
{
    for (int size = size_first; size <= size_last; size <<= 1) {
        for (int stride = (size < n ? size : n) >> 1; stride > 0; stride >>= 1) {
            for (int q = threadIdx.x; q < (n >> 1); q += kPlanThreads) {
                const int lo = ((q & ~(stride - 1)) << 1) | (q & (stride - 1)), hi = lo | stride;
                const unsigned long long a = buf[lo], b = buf[hi];
                const bool up = ((lo + c0) & size) == 0;
                if ((a > b) == up) { buf[lo] = b; buf[hi] = a; }
            }
            __syncthreads();
        }
    }
}

__global__ void __launch_bounds__(kPlanThreads, 1)
few_sum_plan_kernel(const double* __restrict__ t_all, const int* __restrict__ l, const int* __restrict__ m,
                    const int* __restrict__ kpol, const int* __restrict__ n, const int* __restrict__ keep_idx, const int* __restrict__ n_keep,
                    const double2* __restrict__ ylm_plus, const double2* __restrict__ ylm_minus,
                    const double* __restrict__ scale, const double2* __restrict__ factor, double t0, double dt, long long N,
                    int n_t, int n_modes, int smem_elems, sum_layout L, int* status)
{
    extern __shared__ unsigned long long plan_smem[];             // [smem_elems]
    unsigned long long* plan_sorted;                              // [n_pow2] (key << 32 | mode index), sorted ascending
    __shared__ int warp_sums[32];
    __shared__ int carry_s;

    const int src = blockIdx.x, tid = threadIdx.x;
    const double* t = t_all + (size_t)src * n_t;

    // ---- (a) sample ranges of the pseudo-segments and their tile prefix
    long long* B = L.bounds + (size_t)src * (n_t + 2);
    int* TS = L.tile_start + (size_t)src * (n_t + 2);
    for (int k = tid; k < n_t; k += kPlanThreads) {
        if (k + 1 < n_t && !(t[k + 1] > t[k])) atomicOr(status, FEW_DEV_NOT_INCREASING);
        if (k <= n_t - 2) B[k + 1] = first_index(t[k], t0, dt, N, false);
        else { B[n_t] = first_index(t[n_t - 1], t0, dt, N, true); B[n_t + 1] = N; B[0] = 0; }
    }
    __syncthreads();
    if (tid < 32) {           // warp 0: prefix over n_t + 1 pseudo-segments, 32 at a time
        int carry = 0;
        for (int base = 0; base <= n_t; base += 32) {
            int p = base + tid;
            int cnt = 0;
            if (p <= n_t) { long long c = B[p + 1] - B[p]; if (c < 0) c = 0; cnt = (int)((c + kTile - 1) / kTile); }
            int v = cnt;
            for (int o = 1; o < 32; o <<= 1) { int u = __shfl_up_sync(0xffffffffu, v, o); if (tid >= o) v += u; }
            if (p <= n_t) TS[p] = carry + v - cnt;
            carry += __shfl_sync(0xffffffffu, v, 31);
        }
        if (tid == 0) TS[n_t + 1] = carry;
    }

    // ---- (b) kept modes -> keys
    const int K = n_keep ? min(max(n_keep[src], 0), n_modes) : n_modes;
    int n_pow2 = 1;
    while (n_pow2 < K) n_pow2 <<= 1;
    // the sort runs in shared memory when the kept list fits (always for the Schwarzschild grid), else in the workspace with
    // the short-stride steps done chunk by chunk in shared memory (Kerr-shaped lists with > 16384 kept modes)
    const bool in_smem = n_pow2 <= smem_elems;
    plan_sorted = in_smem ? plan_smem : L.sortbuf + (size_t)src * L.sort_pow2;
    for (int q = tid; q < K; q += kPlanThreads) {
        int j = keep_idx ? keep_idx[(size_t)src * n_modes + q] : q;
        bool ok = j >= 0 && j < n_modes;
        int lj = ok ? l[j] : 2, mj = ok ? m[j] : 0, nj = ok ? n[j] : 0, kj = (ok && kpol) ? kpol[j] : 0;
        int an = nj < 0 ? -nj : nj;
        if (!ok || lj < 2 || lj > FEW_MAX_L || mj < 0 || mj > lj || an > FEW_MAX_ABS_N || kj < -FEW_MAX_ABS_K || kj > FEW_MAX_ABS_K) {
            atomicOr(status, FEW_DEV_BAD_MODE);
            lj = 2; mj = 0; an = 0; nj = 0; kj = 0; j = ok ? j : 0;
        }
        const unsigned key = ((unsigned)mj << 25) | ((unsigned)(kj + 64) << 18) | ((nj < 0 ? 1u : 0u) << 17) | ((unsigned)an << 5) |
                             (unsigned)lj;
        plan_sorted[q] = ((unsigned long long)key << 32) | (unsigned)j;
    }
    for (int q = K + tid; q < n_pow2; q += kPlanThreads) plan_sorted[q] = ~0ull;      // padding sorts to the end
    __syncthreads();
    // ---- (c) bitonic sort (keys are unique for a valid mode list; duplicates order by mode index)
    if (in_smem) {
        plan_bitonic_steps(plan_sorted, 0, n_pow2, 2, n_pow2);
    } else {
        const int CH = smem_elems;
        auto chunk_pass = [&](int size_first, int size_last) {
            for (int c0 = 0; c0 < n_pow2; c0 += CH) {
                for (int q = tid; q < CH; q += kPlanThreads) plan_smem[q] = plan_sorted[c0 + q];
                __syncthreads();
                plan_bitonic_steps(plan_smem, c0, CH, size_first, size_last);
                for (int q = tid; q < CH; q += kPlanThreads) plan_sorted[c0 + q] = plan_smem[q];
                __syncthreads();
            }
        };
        chunk_pass(2, CH);
        for (int size = 2 * CH; size <= n_pow2; size <<= 1) {
            for (int stride = size >> 1; stride >= CH; stride >>= 1) {             // long strides: straight through L2
                for (int q = tid; q < (n_pow2 >> 1); q += kPlanThreads) {
                    const int lo = ((q & ~(stride - 1)) << 1) | (q & (stride - 1)), hi = lo | stride;
                    const unsigned long long a = plan_sorted[lo], b = plan_sorted[hi];
                    const bool up = (lo & size) == 0;
                    if ((a > b) == up) { plan_sorted[lo] = b; plan_sorted[hi] = a; }
                }
                __syncthreads();
            }
            chunk_pass(size, size);
        }
    }
    // ---- (d) pairs: chunked scan of "new (m, n)" flags; descriptors; per-mode fold constants
    if (tid == 0) carry_s = 0;
    __syncthreads();
    int* desc = L.desc + (size_t)src * n_modes;
    int* gfirst = L.g_first + (size_t)src * (n_modes + 1);
    int* oj = L.order_j + (size_t)src * n_modes;
    double* yf = L.yfold + (size_t)src * n_modes * 4;
    // every harmonic constant carries the source's prefactor: the real mu/d_L `scale` of Eq. (10) and the complex detector-frame
    // `factor` of Eq. (4)-(8) (few_frame_constants); h is linear in (Y+, Ybar), so the frame rotation costs nothing per sample
    const double sc = scale ? scale[src] : 1.0;
    const double2 fc = factor ? make_double2(sc * factor[src].x, sc * factor[src].y) : make_double2(sc, 0.0);
    for (int base = 0; base < K; base += kPlanThreads) {
        int r = base + tid;
        bool new_run = false, new_sub = false, new_grp = false;
        unsigned key = 0, prev = 0;
        if (r < K) {
            key = (unsigned)(plan_sorted[r] >> 32); prev = r ? (unsigned)(plan_sorted[r - 1] >> 32) : 0u;
            new_run = r == 0 || key_run(key) != key_run(prev);
            new_sub = new_run || key_dir(key) != key_dir(prev);
            new_grp = new_sub || key_absn(key) != key_absn(prev);
        }
        int total, incl = plan_block_scan(new_grp ? 1 : 0, warp_sums, &total);
        int carry = carry_s;
        if (r < K) {
            int j = (int)(unsigned)(plan_sorted[r] & 0xffffffffull);
            oj[r] = j;
            if (new_grp) {
                int g = carry + incl - 1;
                int nadv = new_sub ? key_absn(key) : key_absn(key) - key_absn(prev);
                int dm = new_run ? key_m(key) - (r ? key_m(prev) : 0) : 0;
                int d = (nadv << kAdvShift) | (new_sub ? kNewSub : 0) | (key_dir(key) ? kDirNeg : 0) | (dm << kDmShift) |
                        (new_run ? kNewRun : 0) | ((key_k(key) + 64) << kKShift);
                if (new_sub || nadv != 1) d |= 1;
                desc[g] = d;
                gfirst[g] = r;
            }
            double2 yp = ylm_plus[(size_t)src * n_modes + j], yb = make_double2(0.0, 0.0);
            if (key_m(key) > 0) {                       // Eq. (9): the (l,-m,-k,-n) mirror, Ybar = (-1)^(l+k) Y_{l,-m}
                double2 ym = ylm_minus[(size_t)src * n_modes + j];
                double sg = ((key_l(key) + key_k(key)) & 1) ? -1.0 : 1.0;
                yb = make_double2(sg * ym.x, sg * ym.y);
            }
            yf[4 * r] = fc.x * yp.x - fc.y * yp.y; yf[4 * r + 1] = fc.x * yp.y + fc.y * yp.x;
            yf[4 * r + 2] = fc.x * yb.x - fc.y * yb.y; yf[4 * r + 3] = fc.x * yb.y + fc.y * yb.x;
        }
        __syncthreads();
        if (tid == 0) carry_s = carry + total;
        __syncthreads();
    }
    if (tid == 0) { L.n_groups[src] = carry_s; gfirst[carry_s] = K; if (src == 0) *L.tile_counter = 0; }
}

// (U_mn, V_mn) per pair and segment, written as the stage stream the sum kernel consumes.
__global__ void few_sum_pack_kernel(const double2* __restrict__ coef_amp, int n_t, int n_modes, sum_layout L)
{
    const int k = blockIdx.x, src = blockIdx.y, n_seg = n_t - 1;
    const int G = L.n_groups[src];
    const int* gfirst = L.g_first + (size_t)src * (n_modes + 1);
    const int* oj = L.order_j + (size_t)src * n_modes;
    const int* desc = L.desc + (size_t)src * n_modes;
    const double4* yf = reinterpret_cast<const double4*>(L.yfold) + (size_t)src * n_modes;
    const double2* in = coef_amp + ((size_t)src * n_seg + k) * 4 * n_modes;
    double2* out = reinterpret_cast<double2*>(L.pack) + ((size_t)src * n_seg + k) * L.max_stages * kStageD2;
    for (int idx = threadIdx.x; idx < 4 * G; idx += blockDim.x) {
        const int g = idx >> 2, p = idx & 3;
        double ur = 0.0, ui = 0.0, vr = 0.0, vi = 0.0;
        for (int r = gfirst[g]; r < gfirst[g + 1]; ++r) {
            const double2 c = in[(size_t)p * n_modes + oj[r]];
            const double4 y = yf[r];
            const double ar = y.x * c.x - y.y * c.y, ai = y.x * c.y + y.y * c.x;      // Y+ c
            const double br = y.z * c.x + y.w * c.y, bi = y.w * c.x - y.z * c.y;      // Ybar conj(c)
            ur += ar + br; ui += ai + bi;                                             // U  = a + b
            vr -= ai - bi; vi += ar - br;                                             // V  = i (a - b)
        }
        double2* slot = out + (size_t)(g / kStagePairs) * kStageD2 + (g % kStagePairs) * 8;
        slot[p] = make_double2(ur, ui);
        slot[4 + p] = make_double2(vr, vi);
    }
    const int n_stages = stages_for(G);
    for (int idx = threadIdx.x; idx < n_stages * 64; idx += blockDim.x) {     // header: [0] count, [1] special mask, [2+q] descriptor q
        const int s = idx >> 6, q = idx & 63;
        int v = 0;
        const int cnt = min(kStagePairs, G - s * kStagePairs);
        if (q == 0) v = cnt;
        else if (q == 1) { for (int i = 0; i < cnt; ++i) v |= (desc[s * kStagePairs + i] & 1) << i; }
        else if (q - 2 < cnt) v = desc[s * kStagePairs + q - 2];
        reinterpret_cast<int*>(out + (size_t)s * kStageD2 + kStagePairs * 8)[q] = v;
    }
}

// exp(-i Phi) for Phi = c0 + dx (c1 + dx (c2 + dx c3)) with double-double coefficients (R13, R15).
// c0, c1 dx and c2 dx^2 reach 1e3..1e6 rad and are carried as hi + lo pairs; c3 dx^3 stays below a few rad per segment
// and enters in FP64.  The sum is reduced by 2 pi with a three-part constant (k 2pi_1 and k 2pi_2 are exact products for
// k < 2^23) and the reduced argument goes through one sincos; the low word is applied as a first-order correction.
__device__ __forceinline__ dd dd_add_fast(dd a, dd b)            // error O(eps^2 (|a|+|b|)): enough for 1e-12 rad on 1e6 rad
{
    dd s = two_sum(a.hi, b.hi);
    s.lo = __dadd_rn(s.lo, __dadd_rn(a.lo, b.lo));
    return quick_two_sum(s.hi, s.lo);
}

__device__ __forceinline__ void phase_factor(const dd* __restrict__ c, int stride, double dx, double* zr, double* zi)
{
    dd r = dd_add_d(c[2 * stride], __dmul_rn(c[3 * stride].hi, dx));
    r = dd_add_fast(dd_mul_d(r, dx), c[stride]);
    r = dd_add_fast(dd_mul_d(r, dx), c[0]);
    const double p1 = 0x1.921fb54000000p+2, p2 = 0x1.10b4611800000p-28, p3 = 0x1.313198a2e0370p-59;   // 2 pi = p1 + p2 + p3
    const double kk = rint(r.hi * 1.591549430918953456e-01);
    double q = fma(-kk, p1, r.hi);            // exact
    q = fma(-kk, p2, q);
    const double ql = fma(-kk, p3, r.lo);
    double s, co;
    sincos(q, &s, &co);
    *zr = fma(-ql, s, co);                    // cos(q + ql)
    *zi = -fma(ql, co, s);                    // -sin(q + ql)
}

// ---- mbarrier / TMA bulk copy (1-D cp.async.bulk global -> shared, completion counted in bytes on an mbarrier)
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, unsigned long long* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity)
{
    unsigned ok;
    do {
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                     : "=r"(ok)
                     : "r"(smem_u32(bar)), "r"(parity)
                     : "memory");
    } while (!ok);
}

// E <- E * Z_r for the R samples of a thread (Z_r or conj Z_r, whichever zri currently holds)
template <int R>
__device__ __forceinline__ void advance_e(double (&er)[R], double (&ei)[R], const double (&zrr)[R], const double (&zri)[R])
{
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const double m1 = ei[r] * zri[r], m2 = ei[r] * zrr[r], e0 = er[r];
        er[r] = fma(e0, zrr[r], -m1);
        ei[r] = fma(e0, zri[r], m2);
    }
}

// acc_p += e_r U_p + e_i V_p for the four powers p of dx.  Every DFMA has one block-uniform operand (a coefficient, shared by
// the R samples of the thread) and two per-thread ones.  A DFMA that reads three registers none of which sits in the
// operand-reuse cache costs the FP64 pipe about one cycle more than the usual two, so the R samples are
// walked in alternating directions from one coefficient to the next: where the coefficient changes, e stays the same.
template <int R>
__device__ __forceinline__ void accumulate_pair(const double2* __restrict__ cp, const double (&er)[R], const double (&ei)[R],
                                                double (&are)[4][R], double (&aim)[4][R])
{
#pragma unroll
    for (int p = 0; p < 4; ++p) {
        const double2 u = cp[p];
#pragma unroll
        for (int r = 0; r < R; ++r) are[p][r] = fma(er[r], u.x, are[p][r]);
#pragma unroll
        for (int r = R - 1; r >= 0; --r) aim[p][r] = fma(er[r], u.y, aim[p][r]);
    }
#pragma unroll
    for (int p = 0; p < 4; ++p) {
        const double2 v = cp[4 + p];
#pragma unroll
        for (int r = 0; r < R; ++r) are[p][r] = fma(ei[r], v.x, are[p][r]);
#pragma unroll
        for (int r = R - 1; r >= 0; --r) aim[p][r] = fma(ei[r], v.y, aim[p][r]);
    }
}

// kKerr: Kerr-shaped mode lists (Eq. (1), Eq. (19)): a third phase factor Z_theta and runs of equal (m, k) with
// E restarting from Z_phi^m Z_theta^k; two more per-thread stashes live in dynamic shared memory.  The hot loop is the same.
template <int R, int kBlocksPerSm, bool kInner, bool kKerr>
__global__ void __launch_bounds__(kSumThreads, kBlocksPerSm)
few_sum_kernel(const double* __restrict__ t_all, const dd* __restrict__ coef_phase, double t0, double dt, long long N,
               int n_t, int n_src, int max_tiles, sum_layout L, double2* __restrict__ h_all, const double2* __restrict__ d_all)
{
    constexpr bool want_inner = kInner;      // the inner-product epilogue is compiled out of the plain waveform kernel
    __shared__ __align__(128) double2 ring[kRing][kStageD2];
    __shared__ __align__(8) unsigned long long full[kRing];
    __shared__ double2 stash_zp[R][kSumThreads], stash_pm[R][kSumThreads];   // per-thread Z_phi and Z_phi^m (touched ~20x per tile)
    __shared__ int tile_s;
    __shared__ double red_s[3][kSumThreads / 32];
    extern __shared__ double2 stash_dyn[];      // kKerr: [R][kSumThreads] Z_theta, then [R][kSumThreads] Z_phi^m Z_theta^k
    constexpr int n_ph = kKerr ? 3 : 2;

    const int tid = threadIdx.x, n_seg = n_t - 1;
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kRing; ++s) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    unsigned gst = 0;                       // stages consumed by this block so far: ring slot gst % kRing, parity (gst / kRing) & 1

    // Persistent block: tiles (R*128 samples of one sparse segment of one source) are handed out by an atomic counter, so
    // SMs never idle on wave boundaries and the blocks of an SM drift apart (one block's phase setup overlaps the others'
    // FP64 loops).
    for (;;) {
    __syncthreads();
    if (tid == 0) tile_s = atomicAdd(L.tile_counter, 1);
    __syncthreads();
    const int tg = tile_s;
    if (tg >= n_src * max_tiles) break;
    const int src = tg / max_tiles, tile = tg - src * max_tiles;
    const int* TS = L.tile_start + (size_t)src * (n_t + 2);
    if (tile >= TS[n_t + 1]) continue;
    // pseudo-segment of this tile: largest p with TS[p] <= tile
    int lo = 0, hi = n_t + 1;
    while (hi - lo > 1) { int mid = (lo + hi) >> 1; if (TS[mid] <= tile) lo = mid; else hi = mid; }
    const int p = lo;
    const long long* B = L.bounds + (size_t)src * (n_t + 2);
    const long long i_begin = B[p] + (long long)(tile - TS[p]) * (R * kSumThreads), i_end = B[p + 1];
    double2* h = h_all ? h_all + (size_t)src * N : nullptr;
    const double2* dat = d_all ? d_all + (size_t)src * N : nullptr;
    double* partial = L.partial + ((size_t)src * max_tiles + tile) * 4;

    if (p == 0 || p == n_t) {           // outside [t_0, t_last]: h = 0 (R12)
        if (h) {
#pragma unroll
            for (int r = 0; r < R; ++r) { long long i = i_begin + r * kSumThreads + tid; if (i < i_end) h[i] = make_double2(0.0, 0.0); }
        }
        if (want_inner && tid < 3) partial[tid] = 0.0;
        continue;
    }
    const int k = p - 1;
    const int n_stages = stages_for(L.n_groups[src]);
    const double2* gsrc = reinterpret_cast<const double2*>(L.pack) + ((size_t)src * n_seg + k) * L.max_stages * kStageD2;

    // ---- producer prologue: thread 0 arms the ring with the first kRing - 1 stages of this tile
    if (tid == 0) {
        for (int s = 0; s < kRing - 1 && s < n_stages; ++s) {
            const int b = (gst + s) % kRing;
            mbar_expect_tx(&full[b], kStageBytes);
            bulk_g2s(&ring[b][0], gsrc + (size_t)s * kStageD2, kStageBytes, &full[b]);
        }
    }

    // ---- per-sample setup (overlaps the first copies): dx and the two phase factors
    const double tk = t_all[(size_t)src * n_t + k];
    const dd* cph = coef_phase + ((size_t)src * n_seg + k) * 4 * n_ph;     // [4][n_ph] dd
    double zrr[R], zri[R], er[R], ei[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        long long i = i_begin + r * kSumThreads + tid;
        if (i >= i_end) i = i_end - 1;                              // tail lanes recompute the last sample, never store
        const double dx = __dsub_rn(sample_time(t0, dt, i), tk);
        double zpr, zpi;
        phase_factor(cph + 0, n_ph, dx, &zpr, &zpi);
        phase_factor(cph + n_ph - 1, n_ph, dx, &zrr[r], &zri[r]);
        if (kKerr) {
            double ztr, zti;
            phase_factor(cph + 1, n_ph, dx, &ztr, &zti);
            stash_dyn[r * kSumThreads + tid] = make_double2(ztr, zti);
            stash_dyn[(R + r) * kSumThreads + tid] = make_double2(1.0, 0.0);
        }
        // Z_phi and the run's Z_phi^m are needed only when m or the sign of n changes: parked in shared memory, not registers
        stash_zp[r][tid] = make_double2(zpr, zpi);
        stash_pm[r][tid] = make_double2(1.0, 0.0);
        er[r] = 1.0; ei[r] = 0.0;
    }
    double are[4][R], aim[4][R];                                    // sum over pairs of e_r U_p + e_i V_p, p = power of dx
#pragma unroll
    for (int q = 0; q < 4; ++q)
#pragma unroll
        for (int r = 0; r < R; ++r) are[q][r] = aim[q][r] = 0.0;
    bool neg = false;                                               // zri currently holds -Im Z_r (walking n downward)

    for (int st = 0; st < n_stages; ++st) {
        __syncthreads();                                            // stage st-1 fully consumed (and barriers initialised)
        if (tid == 0 && st + kRing - 1 < n_stages) {
            const int s = st + kRing - 1, b = (gst + kRing - 1) % kRing;
            mbar_expect_tx(&full[b], kStageBytes);
            bulk_g2s(&ring[b][0], gsrc + (size_t)s * kStageD2, kStageBytes, &full[b]);
        }
        const int b = gst % kRing;
        mbar_wait(&full[b], (gst / kRing) & 1u);
        ++gst;
        const double2* cp = &ring[b][0];
        const int* hdr = reinterpret_cast<const int*>(cp + kStagePairs * 8);
        const int ng = hdr[0];
        unsigned spec = (unsigned)hdr[1];
        int gi = 0;
        while (gi < ng) {
            if ((spec & 3u) == 0u && gi + 1 < ng) {                 // common: the next two n of the same run, E *= Z_r each
                advance_e<R>(er, ei, zrr, zri);
                accumulate_pair<R>(cp, er, ei, are, aim);
                advance_e<R>(er, ei, zrr, zri);
                accumulate_pair<R>(cp + 8, er, ei, are, aim);
                gi += 2; cp += 16; spec >>= 2;
                continue;
            }
            if (spec & 1u) {                                        // rare: new m, sign change of n, or a gap in n
                const int d = hdr[2 + gi];
                if (d & kNewRun) {
                    const int dm = (d >> kDmShift) & ((1 << kDmBits) - 1);
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        double2 pm = stash_pm[r][tid];
                        const double2 zp = stash_zp[r][tid];
                        for (int q = 0; q < dm; ++q) {
                            double a = pm.x * zp.x - pm.y * zp.y;
                            pm.y = pm.x * zp.y + pm.y * zp.x;
                            pm.x = a;
                        }
                        stash_pm[r][tid] = pm;
                        if (kKerr) {                                // base of the run: Z_phi^m Z_theta^k (k < 0: conjugate powers)
                            const int kk = ((d >> kKShift) & ((1 << kKBits) - 1)) - 64;
                            double2 zt = stash_dyn[r * kSumThreads + tid];
                            if (kk < 0) zt.y = -zt.y;
                            for (int q = 0; q < (kk < 0 ? -kk : kk); ++q) {
                                double a = pm.x * zt.x - pm.y * zt.y;
                                pm.y = pm.x * zt.y + pm.y * zt.x;
                                pm.x = a;
                            }
                            stash_dyn[(R + r) * kSumThreads + tid] = pm;
                        }
                    }
                }
                if (d & kNewSub) {
                    const bool want_neg = (d & kDirNeg) != 0;
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const double2 pm = kKerr ? stash_dyn[(R + r) * kSumThreads + tid] : stash_pm[r][tid];
                        er[r] = pm.x; ei[r] = pm.y;
                        if (want_neg != neg) zri[r] = -zri[r];
                    }
                    neg = want_neg;
                }
                const int nadv = (d >> kAdvShift) & ((1 << kAdvBits) - 1);
                for (int q = 0; q < nadv; ++q) advance_e<R>(er, ei, zrr, zri);
            } else {
                advance_e<R>(er, ei, zrr, zri);
            }
            accumulate_pair<R>(cp, er, ei, are, aim);
            ++gi; cp += 8; spec >>= 1;
        }
    }

    // ---- h = acc_0 + dx (acc_1 + dx (acc_2 + dx acc_3)), once per sample; optionally the tile's share of the PSD = 1 inner
    // products <d|h>, <h|h> so that a likelihood evaluation never writes h to HBM
    double s_re = 0.0, s_im = 0.0, s_hh = 0.0;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const long long i = i_begin + r * kSumThreads + tid;
        if (i < i_end) {
            const double dx = __dsub_rn(sample_time(t0, dt, i), tk);
            const double hr = fma(fma(fma(are[3][r], dx, are[2][r]), dx, are[1][r]), dx, are[0][r]);
            const double hi = fma(fma(fma(aim[3][r], dx, aim[2][r]), dx, aim[1][r]), dx, aim[0][r]);
            if (h) __stcs(&h[i], make_double2(hr, hi));
            if (want_inner) {
                if (dat) {
                    const double2 dv = __ldcs(&dat[i]);
                    s_re = fma(dv.x, hr, fma(dv.y, hi, s_re));      // Re conj(d) h
                    s_im = fma(dv.x, hi, fma(-dv.y, hr, s_im));     // Im conj(d) h
                }
                s_hh = fma(hr, hr, fma(hi, hi, s_hh));
            }
        }
    }
    if (want_inner) {                   // fixed tree: lanes by butterfly, then the warps in order -> the same bits every run
#pragma unroll
        for (int o = 16; o; o >>= 1) {
            s_re += __shfl_xor_sync(0xffffffffu, s_re, o);
            s_im += __shfl_xor_sync(0xffffffffu, s_im, o);
            s_hh += __shfl_xor_sync(0xffffffffu, s_hh, o);
        }
        if ((tid & 31) == 0) { red_s[0][tid >> 5] = s_re; red_s[1][tid >> 5] = s_im; red_s[2][tid >> 5] = s_hh; }
        __syncthreads();
        if (tid < 3) {
            double v = 0.0;
#pragma unroll
            for (int w = 0; w < kSumThreads / 32; ++w) v += red_s[tid][w];
            partial[tid] = v;
        }
    }
    }   // persistent tile loop
}

// inner[src] = 2 dt * (sum over the source's tiles of the per-tile partials): Eq. (16) with S_n = 1 by Parseval.  One block per
// source; thread q adds tiles q, q + 256, ... in order, then a fixed tree: deterministic.
constexpr int kInnerThreads = 256;
__global__ void __launch_bounds__(kInnerThreads)
few_sum_inner_kernel(sum_layout L, int n_t, int max_tiles, double dt, double* __restrict__ inner)
{
    __shared__ double red[3][kInnerThreads / 32];
    const int src = blockIdx.x, tid = threadIdx.x;
    const int n_tiles = L.tile_start[(size_t)src * (n_t + 2) + n_t + 1];
    const double* P = L.partial + (size_t)src * max_tiles * 4;
    double a = 0.0, b = 0.0, c = 0.0;
    for (int q = tid; q < n_tiles; q += kInnerThreads) { a += P[4 * (size_t)q]; b += P[4 * (size_t)q + 1]; c += P[4 * (size_t)q + 2]; }
    for (int o = 16; o; o >>= 1) {
        a += __shfl_xor_sync(0xffffffffu, a, o); b += __shfl_xor_sync(0xffffffffu, b, o); c += __shfl_xor_sync(0xffffffffu, c, o);
    }
    if ((tid & 31) == 0) { red[0][tid >> 5] = a; red[1][tid >> 5] = b; red[2][tid >> 5] = c; }
    __syncthreads();
    if (tid < 3) {
        double v = 0.0;
        for (int w = 0; w < kInnerThreads / 32; ++w) v += red[tid][w];
        inner[(size_t)src * 3 + tid] = 2.0 * dt * v;
    }
}

int plan_smem_elems(int n_modes)
{
    int p = 1;
    while (p < n_modes) p <<= 1;
    return p < kPlanSmemElems ? p : kPlanSmemElems;
}

}  // namespace

extern "C" size_t few_sum_waveform_workspace(int n_src, int n_t, int n_modes, long long n_samples)
{
    if (n_src <= 0 || n_t < 2 || n_modes <= 0 || n_samples < 0) return 0;
    size_t bytes = 0;
    sum_carve(nullptr, n_src, n_t, n_modes, n_samples, &bytes);
    return bytes;
}

extern "C" int few_sum_waveform_kerr(few_ctx* ctx, const double* t, const double* coef_amp, const double* coef_phase_dd, int n_phase,
                                     const int* l, const int* m, const int* k, const int* n, const int* keep_idx, const int* n_keep,
                                     const double* ylm_plus, const double* ylm_minus, const double* scale, const double* factor,
                                     double t0, double dt, long long n_samples, double* h, const double* d, double* inner,
                                     int n_src, int n_t, int n_modes, void* workspace, size_t workspace_bytes, void* stream)
{
    FEW_REQUIRE(n_phase == 2 || n_phase == 3, FEW_ERR_INVALID_ARG, "n_phase must be 2 (Phi_phi, Phi_r) or 3 (Phi_phi, Phi_theta, Phi_r)");
    FEW_REQUIRE(n_phase == 3 || k == nullptr, FEW_ERR_INVALID_ARG, "a polar index k needs the third phase (n_phase = 3)");
    FEW_REQUIRE(ctx && t && coef_amp && coef_phase_dd && l && m && n && ylm_plus && ylm_minus, FEW_ERR_INVALID_ARG, "NULL argument");
    FEW_REQUIRE((keep_idx == nullptr) == (n_keep == nullptr), FEW_ERR_INVALID_ARG, "keep_idx and n_keep must both be NULL or both be set");
    FEW_REQUIRE(n_src > 0 && n_modes > 0 && n_samples >= 0, FEW_ERR_INVALID_ARG, "sizes must be positive");
    FEW_REQUIRE(n_t >= 4, FEW_ERR_TOO_FEW_POINTS, "n_t < 4");
    FEW_REQUIRE(dt > 0.0 && isfinite(dt) && isfinite(t0), FEW_ERR_INVALID_ARG, "dt must be positive and finite");
    FEW_REQUIRE(n_src <= 65535 && n_t <= 65535, FEW_ERR_LIMIT, "n_src or n_t > 65535");
    FEW_REQUIRE(d == nullptr || inner != nullptr, FEW_ERR_INVALID_ARG, "d given but inner is NULL");
    cudaStream_t st = (cudaStream_t)stream;
    if (n_samples == 0) {
        if (inner) FEW_CUDA_CHECK(cudaMemsetAsync(inner, 0, (size_t)n_src * 3 * sizeof(double), st));
        return FEW_OK;
    }
    FEW_REQUIRE(h != nullptr || inner != nullptr, FEW_ERR_INVALID_ARG, "h and inner are both NULL");
    FEW_REQUIRE(workspace && ((uintptr_t)workspace % 256) == 0 &&
                    workspace_bytes >= few_sum_waveform_workspace(n_src, n_t, n_modes, n_samples),
                FEW_ERR_WORKSPACE, "workspace NULL, misaligned or too small");
    const int plan_elems = plan_smem_elems(n_modes);
    const size_t psm = (size_t)plan_elems * 8;
    FEW_REQUIRE(psm <= (size_t)ctx->smem_optin, FEW_ERR_LIMIT, "plan kernel's shared memory exceeds the device limit");
    long long max_tiles = sum_max_tiles(n_samples, n_t);
    FEW_REQUIRE(max_tiles < 2147483647LL, FEW_ERR_LIMIT, "n_samples too large");
    sum_layout L = sum_carve(workspace, n_src, n_t, n_modes, n_samples);

    FEW_CUDA_CHECK(cudaFuncSetAttribute(few_sum_plan_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)psm));
    few_sum_plan_kernel<<<n_src, kPlanThreads, psm, st>>>(t, l, m, k, n, keep_idx, n_keep, (const double2*)ylm_plus,
                                                          (const double2*)ylm_minus, scale, (const double2*)factor, t0, dt, n_samples,
                                                          n_t, n_modes, plan_elems, L, ctx->d_status);
    FEW_LAUNCHED(ctx);
    // few blocks (one waveform): 1024 threads finish a segment's 4 x pairs items in one sweep; a batch fills the SMs with
    // several 256-thread blocks each, which hides the dependent index -> coefficient loads better
    const int pack_threads = (long long)(n_t - 1) * n_src < 2LL * ctx->sm_count ? 1024 : 256;
    few_sum_pack_kernel<<<dim3(n_t - 1, n_src), pack_threads, 0, st>>>((const double2*)coef_amp, n_t, n_modes, L);
    FEW_LAUNCHED(ctx);
    if (ctx->profile) FEW_CUDA_CHECK(cudaEventRecord(ctx->ev_sum[0], st));
    FEW_REQUIRE(max_tiles * n_src < 2147483647LL - 65536, FEW_ERR_LIMIT, "n_src * n_samples too large");
    const long long want = max_tiles * n_src, resident = (long long)ctx->sm_count * kSumBlocksPerSm;
    const unsigned grid = (unsigned)(want < resident ? want : resident);
    const size_t kerr_smem = 2 * (size_t)kSumR * kSumThreads * sizeof(double2);      // Z_theta and run-base stashes
#define FEW_SUM_LAUNCH(INNER, KERR, SMEM, DPTR)                                                                                   \
    few_sum_kernel<kSumR, kSumBlocksPerSm, INNER, KERR><<<grid, kSumThreads, SMEM, st>>>(                                         \
        t, (const dd*)coef_phase_dd, t0, dt, n_samples, n_t, n_src, (int)max_tiles, L, (double2*)h, DPTR)
    if (n_phase == 3) {     // static + dynamic shared memory exceeds the 48 KB default: opt in
        FEW_CUDA_CHECK(cudaFuncSetAttribute(few_sum_kernel<kSumR, kSumBlocksPerSm, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kerr_smem));
        FEW_CUDA_CHECK(cudaFuncSetAttribute(few_sum_kernel<kSumR, kSumBlocksPerSm, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kerr_smem));
        if (inner) FEW_SUM_LAUNCH(true, true, kerr_smem, (const double2*)d);
        else FEW_SUM_LAUNCH(false, true, kerr_smem, nullptr);
    } else {
        if (inner) FEW_SUM_LAUNCH(true, false, 0, (const double2*)d);
        else FEW_SUM_LAUNCH(false, false, 0, nullptr);
    }
#undef FEW_SUM_LAUNCH
    FEW_LAUNCHED(ctx);
    if (ctx->profile) { FEW_CUDA_CHECK(cudaEventRecord(ctx->ev_sum[1], st)); ctx->profile_valid = 1; }
    if (inner) {
        few_sum_inner_kernel<<<n_src, kInnerThreads, 0, st>>>(L, n_t, (int)max_tiles, dt, inner);
        FEW_LAUNCHED(ctx);
    }
    return FEW_OK;
}

extern "C" int few_sum_waveform_ex(few_ctx* ctx, const double* t, const double* coef_amp, const double* coef_phase_dd,
                                   const int* l, const int* m, const int* n, const int* keep_idx, const int* n_keep,
                                   const double* ylm_plus, const double* ylm_minus, const double* scale, const double* factor,
                                   double t0, double dt, long long n_samples, double* h, const double* d, double* inner,
                                   int n_src, int n_t, int n_modes, void* workspace, size_t workspace_bytes, void* stream)
{
    return few_sum_waveform_kerr(ctx, t, coef_amp, coef_phase_dd, 2, l, m, nullptr, n, keep_idx, n_keep, ylm_plus, ylm_minus, scale,
                                 factor, t0, dt, n_samples, h, d, inner, n_src, n_t, n_modes, workspace, workspace_bytes, stream);
}

extern "C" int few_sum_waveform(few_ctx* ctx, const double* t, const double* coef_amp, const double* coef_phase_dd,
                                const int* l, const int* m, const int* n, const int* keep_idx, const int* n_keep,
                                const double* ylm_plus, const double* ylm_minus, const double* scale,
                                double t0, double dt, long long n_samples, double* h,
                                int n_src, int n_t, int n_modes, void* workspace, size_t workspace_bytes, void* stream)
{
    FEW_REQUIRE(n_samples == 0 || h != nullptr, FEW_ERR_INVALID_ARG, "h is NULL");
    return few_sum_waveform_ex(ctx, t, coef_amp, coef_phase_dd, l, m, n, keep_idx, n_keep, ylm_plus, ylm_minus, scale, nullptr,
                               t0, dt, n_samples, h, nullptr, nullptr, n_src, n_t, n_modes, workspace, workspace_bytes, stream);
}
