// few_sum.cu -- S3: the interpolated summation (sec. III C, Eq. (9), Eq. (10)):
//   "the actual summation kernel evaluates the spline at the sampling rate of the output data stream.  Then, the output
//    phase and amplitude values are combined within each mode according to Eq. (1) ... A_{l,-m,-k,-n} = (-1)^{l+k} A*_{lmkn}
//    ... only compute modes for m >= 0 ... the modes in a single time step are combined."
//   h(t_i) = scale * sum_{j kept} [ Y+_j W_j + (m_j>0) (-1)^{l_j} Y-_j conj(W_j) ],  W_j = A_j(t_i) exp(-i(m_j Phi_phi + n_j Phi_r)).
//
// Algebra used (exact).  With E = exp(-i theta), Ybar = (-1)^(l+k) Y- (0 for m = 0), a mode contributes
// alpha E + beta conj(E), alpha = Y+ A, beta = Ybar conj(A): complex cubics in dx (linear in A's spline coefficients).  E depends
// on (m, k, n) only, so all kept l of one (m, k, n) are summed into one (alpha, beta) per sparse segment BEFORE the sample loop.
// Further, E_{m,k,+-nu} = P rho^(+-nu) with P = exp(-i(m Phi_phi + k Phi_theta)) (one per RUN (m, k)) and
// rho^nu = exp(-i nu Phi_r) = c_nu + i s_nu, so the two signs of n share (c_nu, s_nu) -- a UNIT (m, k, nu):
//   sum over the run = P_r S + i P_i D,   S = sum_nu c_nu B1c_nu + s_nu B1s_nu,   D = sum_nu c_nu B2c_nu + s_nu B2s_nu,
//   B1c = (alpha+ + alpha-) + (beta+ + beta-),   B1s = i(alpha+ - alpha-) + i(beta- - beta+),
//   B2c = (alpha+ + alpha-) - (beta+ + beta-),   B2s = i(alpha+ - alpha-) - i(beta- - beta+).
// S and D are [samples] x [4 powers of dx x (re, im)] = sum over units of [samples x units] . [units x 8]: a small dense FP64
// contraction per sample tile, executed as DMMA.8x8x4 (mma.sync.m8n8k4.f64) on the FP64 pipe -- 8 samples x 4 consecutive nu
// per instruction; a lane carries (c_nu, s_nu) of ONE sample and ONE of the four nu and steps it by rho^4 (2 DMUL + 2 DFMA)
// between the 4 DMMAs of a step.  Per sample and unit: 32 FMA in DMMAs + 4 scalar FP64 operations (40 scalar operations in
// the per-(m,n)-pair DFMA form this replaces).  The same IEEE FMA arithmetic on the same pipe; what changes is that a DMMA
// reads 4 registers per 8 FMA where a DFMA reads 3 per FMA, which is what held the DFMA form at 0.75 of the pipe.
//
// Three launches per call, all on the caller's stream, nothing read back to the host:
//   1. few_sum_plan_kernel  (one block per source): clips the dense sample grid to the sparse segments and prefix-sums
//        the per-segment tile counts (every block of the sum kernel works inside ONE segment, so its coefficients are
//        block-uniform); orders the kept modes by (m, k, |n|, sign n, l) and cuts them into STEPS: the kept units of one run
//        whose nu fall into one aligned block of four (4b .. 4b+3), with a descriptor saying how (c, s) is reached.
//   2. few_sum_pack_kernel  (one block per source and segment): forms the four B matrices of every step from the kept modes'
//        spline coefficients and Y+, Ybar, scale, in DMMA fragment order, as a stream of stages (4 steps x 1 KB + header).
//   3. few_sum_kernel       the hot loop.  Stages arrive in shared memory through a ring of TMA bulk copies
//        (cp.async.bulk + mbarrier) and are read with conflict-free 128-bit loads.  Per sample the phases are evaluated ONCE in
//        double-double (Horner, reduction by 2 pi, one sincos each).  Output: coalesced 16-byte streaming stores.
#include "few_common.cuh"

namespace {

constexpr int kPlanThreads = 1024;
constexpr int kPlanSmemElems = 16384;         // 128 KB of (key, mode) words: the plan kernel's in-shared-memory sort capacity
constexpr int kSumThreads = 128;
#ifndef FEW_SUM_G
#define FEW_SUM_G 4
#define FEW_SUM_BPS 4
#endif
constexpr int kSumG = FEW_SUM_G;              // groups of 8 samples per warp
constexpr int kSumBlocksPerSm = FEW_SUM_BPS;  // resident blocks per SM (register budget 65536 / (128 * blocks))
constexpr int kTile = (kSumThreads / 32) * 8 * kSumG;   // samples per block
constexpr int kTileQ = kTile / kSumThreads;   // samples per thread in the per-sample prologue / epilogue
constexpr int kStageSteps = 4;                // steps per stage
constexpr int kStepD2 = 64;                   // a step's B fragments: [2][32 lanes] double2 = 1 KB
constexpr int kStageBytes = kStageSteps * kStepD2 * 16 + 128;   // + header: [0] steps in the stage, [1 + i] descriptor of step i
constexpr int kStageD2 = kStageBytes / 16;    // stage size in double2
constexpr int kRing = 4;                      // stages in flight per block

// step descriptor
constexpr int kNewRun = 1;                    // first step of a run (m, k): close the previous run, P <- Z_phi^m Z_theta^k, (c, s) <- rho^col
constexpr int kAdvShift = 1, kAdvBits = 12;   // multiplications by rho^4 before the step's DMMAs
constexpr int kDmShift = 13, kDmBits = 7;     // m increment of a new run
constexpr int kKShift = 20, kKBits = 7;       // polar index of the run, offset by 64 (Kerr-shaped lists, |k| <= FEW_MAX_ABS_K)

struct sum_layout {
    long long* bounds;   // [n_src][n_t + 2]   pseudo-segment p covers samples [bounds[p], bounds[p+1])
    int* tile_start;     // [n_src][n_t + 2]   exclusive prefix of tiles per pseudo-segment; last = total
    int* n_steps;        // [n_src]            number of steps
    int* tile_counter;   // [1]                dynamic tile scheduler of the persistent sum kernel
    int* desc;           // [n_src][cap]       step descriptors
    int* u_lo;           // [n_src][cap][8]    sorted range [u_lo, u_hi) of the modes of (step, nu & 3, sign of n)
    int* u_hi;           // [n_src][cap][8]
    int* order_j;        // [n_src][n_modes]   mode index of sorted position r
    double* yfold;       // [n_src][n_modes][4] scale * (Y+ re, Y+ im, Ybar re, Ybar im) of sorted position r
    double* pack;        // [n_src][n_t - 1][max_stages][kStageBytes / 8]
    double* partial;     // [n_src][max_tiles][4]  per-tile sums of conj(d) h (re, im) and |h|^2 (fused inner products)
    unsigned long long* sortbuf;   // [n_src][sort_pow2] plan-kernel sort array when the mode list exceeds shared memory (else empty)
    int sort_pow2;
    int cap;             // step capacity per source
    int max_stages;
    int max_tiles;
};

// Step capacity: a step holds up to 8 (m, k, n) triples of one run.  Any mode list on a grid (the paper's: 11 m x 8 blocks of
// nu = 88 steps for 3843 modes) needs far fewer than n_modes / 4 steps; a list with fewer than 4 modes per step on average AND
// more than 64 steps over that does not fit and is reported (FEW_DEV_SPARSE_LIST -> FEW_ERR_LIMIT).
__host__ __device__ inline int step_capacity(int n_modes) { int c = n_modes / 4 + 64; return c < n_modes ? c : n_modes; }
__host__ __device__ inline int stages_for(int n_steps) { return (n_steps + kStageSteps - 1) / kStageSteps; }

__host__ inline long long sum_max_tiles(long long n_samples, int n_t) { return (n_samples + kTile - 1) / kTile + n_t + 1; }

sum_layout sum_carve(void* ws, int n_src, int n_t, int n_modes, long long n_samples, size_t* bytes = nullptr)
{
    few_carver c(ws);
    sum_layout L;
    L.cap = step_capacity(n_modes);
    L.max_stages = stages_for(L.cap);
    L.bounds = c.take<long long>((size_t)n_src * (n_t + 2));
    L.tile_start = c.take<int>((size_t)n_src * (n_t + 2));
    L.n_steps = c.take<int>(n_src);
    L.tile_counter = c.take<int>(1);
    L.desc = c.take<int>((size_t)n_src * L.cap);
    L.u_lo = c.take<int>((size_t)n_src * L.cap * 8);
    L.u_hi = c.take<int>((size_t)n_src * L.cap * 8);
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

// sort key: m | k + 64 | |n| | sign(n) | l  (ascending): runs of equal (m, k); inside a run nu = |n| ascending, +nu before -nu
__device__ __forceinline__ int key_m(unsigned k) { return (int)(k >> 25); }
__device__ __forceinline__ int key_k(unsigned k) { return (int)((k >> 18) & 0x7f) - 64; }
__device__ __forceinline__ unsigned key_run(unsigned k) { return k >> 18; }
__device__ __forceinline__ int key_absn(unsigned k) { return (int)(k >> 6) & 0xfff; }
__device__ __forceinline__ int key_neg(unsigned k) { return (int)(k >> 5) & 1; }
__device__ __forceinline__ int key_l(unsigned k) { return (int)(k & 0x1f); }
__device__ __forceinline__ unsigned key_unit_sign(unsigned k) { return k >> 5; }      // (run, nu, sign): one (m, k, n) triple

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
    int* ulo = L.u_lo + (size_t)src * L.cap * 8;
    int* uhi = L.u_hi + (size_t)src * L.cap * 8;
    for (int q = tid; q < L.cap * 8; q += kPlanThreads) { ulo[q] = 0; uhi[q] = 0; }      // empty (step, nu & 3, sign) slots
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
        const unsigned key = ((unsigned)mj << 25) | ((unsigned)(kj + 64) << 18) | ((unsigned)an << 6) | ((nj < 0 ? 1u : 0u) << 5) |
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
    // ---- (d) steps: chunked scan of "new (run, nu >> 2)" flags; descriptors; (step, nu & 3, sign) ranges; fold constants
    if (tid == 0) carry_s = 0;
    __syncthreads();
    int* desc = L.desc + (size_t)src * L.cap;
    int* oj = L.order_j + (size_t)src * n_modes;
    double* yf = L.yfold + (size_t)src * n_modes * 4;
    // every harmonic constant carries the source's prefactor: the real mu/d_L `scale` of Eq. (10) and the complex detector-frame
    // `factor` of Eq. (4)-(8) (few_frame_constants); h is linear in (Y+, Ybar), so the frame rotation costs nothing per sample
    const double sc = scale ? scale[src] : 1.0;
    const double2 fc = factor ? make_double2(sc * factor[src].x, sc * factor[src].y) : make_double2(sc, 0.0);
    for (int base = 0; base < K; base += kPlanThreads) {
        int r = base + tid;
        bool new_run = false, new_step = false;
        unsigned key = 0, prev = 0;
        if (r < K) {
            key = (unsigned)(plan_sorted[r] >> 32); prev = r ? (unsigned)(plan_sorted[r - 1] >> 32) : 0u;
            new_run = r == 0 || key_run(key) != key_run(prev);
            new_step = new_run || (key_absn(key) >> 2) != (key_absn(prev) >> 2);
        }
        int total, incl = plan_block_scan(new_step ? 1 : 0, warp_sums, &total);
        int carry = carry_s;
        if (r < K) {
            const int j = (int)(unsigned)(plan_sorted[r] & 0xffffffffull);
            const int s = carry + incl - 1;                 // step of sorted position r
            oj[r] = j;
            if (s < L.cap) {
                if (new_step) {
                    const int blk = key_absn(key) >> 2;
                    const int adv = new_run ? blk : blk - (key_absn(prev) >> 2);
                    const int dm = new_run ? key_m(key) - (r ? key_m(prev) : 0) : 0;
                    desc[s] = (new_run ? kNewRun : 0) | (adv << kAdvShift) | (dm << kDmShift) | ((key_k(key) + 64) << kKShift);
                }
                const int slot = s * 8 + (key_absn(key) & 3) * 2 + key_neg(key);
                if (r == 0 || key_unit_sign(key) != key_unit_sign(prev)) ulo[slot] = r;
                const unsigned next = r + 1 < K ? (unsigned)(plan_sorted[r + 1] >> 32) : ~0u;
                if (r + 1 == K || key_unit_sign(key) != key_unit_sign(next)) uhi[slot] = r + 1;
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
    if (tid == 0) {
        int S = carry_s;
        if (S > L.cap) { atomicOr(status, FEW_DEV_SPARSE_LIST); S = L.cap; }
        L.n_steps[src] = S;
        if (src == 0) *L.tile_counter = 0;
    }
}

// The four B matrices of every step, in DMMA.8x8x4 fragment order, written as the stage stream the sum kernel consumes.
// Lane L of a warp supplies B[k = L & 3][o = L >> 2]: unit k of the step (nu = 4 blk + k), output o = 2 p + part (power p of
// dx, part 0 = re, 1 = im).  A step is 1 KB: [0][L] = (B1c, B2c), [1][L] = (B1s, B2s) as double2 (conflict-free LDS.128).
__global__ void few_sum_pack_kernel(const double2* __restrict__ coef_amp, int n_t, int n_modes, sum_layout L)
{
    const int seg = blockIdx.x, src = blockIdx.y, n_seg = n_t - 1;
    const int S = L.n_steps[src];
    const int* ulo = L.u_lo + (size_t)src * L.cap * 8;
    const int* uhi = L.u_hi + (size_t)src * L.cap * 8;
    const int* oj = L.order_j + (size_t)src * n_modes;
    const int* desc = L.desc + (size_t)src * L.cap;
    const double4* yf = reinterpret_cast<const double4*>(L.yfold) + (size_t)src * n_modes;
    const double2* in = coef_amp + ((size_t)src * n_seg + seg) * 4 * n_modes;
    double2* out = reinterpret_cast<double2*>(L.pack) + ((size_t)src * n_seg + seg) * L.max_stages * kStageD2;
    for (int idx = threadIdx.x; idx < 32 * S; idx += blockDim.x) {
        const int s = idx >> 5, lane = idx & 31, k = lane & 3, o = lane >> 2, p = o >> 1, part = o & 1;
        double ar[2] = {0.0, 0.0}, ai[2] = {0.0, 0.0}, br[2] = {0.0, 0.0}, bi[2] = {0.0, 0.0};   // alpha, beta of +nu [0] and -nu [1]
#pragma unroll
        for (int sg = 0; sg < 2; ++sg) {
            const int slot = s * 8 + k * 2 + sg;
            for (int r = ulo[slot]; r < uhi[slot]; ++r) {
                const double2 c = in[(size_t)p * n_modes + oj[r]];
                const double4 y = yf[r];
                ar[sg] += y.x * c.x - y.y * c.y; ai[sg] += y.x * c.y + y.y * c.x;      // Y+ c
                br[sg] += y.z * c.x + y.w * c.y; bi[sg] += y.w * c.x - y.z * c.y;      // Ybar conj(c)
            }
        }
        // a = alpha+ + alpha-, b = beta+ + beta-, da = alpha+ - alpha-, db = beta- - beta+ ;  i z = (-z.im, z.re)
        const double a_r = ar[0] + ar[1], a_i = ai[0] + ai[1], b_r = br[0] + br[1], b_i = bi[0] + bi[1];
        const double da_r = ar[0] - ar[1], da_i = ai[0] - ai[1], db_r = br[1] - br[0], db_i = bi[1] - bi[0];
        double b1c, b2c, b1s, b2s;
        if (part == 0) { b1c = a_r + b_r; b2c = a_r - b_r; b1s = -(da_i + db_i); b2s = -(da_i - db_i); }
        else           { b1c = a_i + b_i; b2c = a_i - b_i; b1s = da_r + db_r;    b2s = da_r - db_r; }
        double2* step = out + (size_t)(s / kStageSteps) * kStageD2 + (s % kStageSteps) * kStepD2;
        step[lane] = make_double2(b1c, b2c);
        step[32 + lane] = make_double2(b1s, b2s);
    }
    const int n_stages = stages_for(S);
    for (int idx = threadIdx.x; idx < n_stages * 32; idx += blockDim.x) {     // header: [0] steps in the stage, [1 + i] descriptor i
        const int st = idx >> 5, q = idx & 31;
        int v = 0;
        const int cnt = min(kStageSteps, S - st * kStageSteps);
        if (q == 0) v = cnt;
        else if (q - 1 < cnt) v = desc[st * kStageSteps + q - 1];
        reinterpret_cast<int*>(out + (size_t)st * kStageD2 + kStageSteps * kStepD2)[q] = v;
    }
    // steps of the last stage beyond S are never read (the header's count stops the consumer)
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

// D(8x8) += A(8x4) B(4x8) in FP64 on the FP64 pipe (SASS DMMA.8x8x4).  Lane L holds A[L >> 2][L & 3], B[L & 3][L >> 2],
// C[L >> 2][2 (L & 3)], C[L >> 2][2 (L & 3) + 1].
__device__ __forceinline__ void dmma884(double2& c, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c.x), "+d"(c.y) : "d"(a), "d"(b));
}

__device__ __forceinline__ double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }

// G: groups of 8 samples per warp (tile = 4 warps x 8 G samples).  kKerr: Kerr-shaped mode lists (Eq. (1),
// Eq. (19)): a third phase factor Z_theta, runs are (m, k) with P = Z_phi^m Z_theta^k.  The hot loop is the same.
template <int G, int kBlocksPerSm, bool kInner, bool kKerr>
__global__ void __launch_bounds__(kSumThreads, kBlocksPerSm)
few_sum_kernel(const double* __restrict__ t_all, const dd* __restrict__ coef_phase, double t0, double dt, long long N,
               int n_t, int n_src, int max_tiles, sum_layout L, double2* __restrict__ h_all, const double2* __restrict__ d_all)
{
    constexpr bool want_inner = kInner;      // the inner-product epilogue is compiled out of the plain waveform kernel
    constexpr int T = 32 * G, Q = T / kSumThreads;
    __shared__ __align__(128) double2 ring[kRing][kStageD2];
    __shared__ __align__(8) unsigned long long full[kRing];
    __shared__ __align__(16) double2 zphi_s[T];          // Z_phi = exp(-i Phi_phi) per sample of the tile
    __shared__ __align__(16) double2 rpow_s[T][4];       // rho, rho^2, rho^3, rho^4 per sample; after the loop: H_p, p = 0..3
    __shared__ __align__(16) double2 kerr_s[kKerr ? 2 * T : 1];   // kKerr: Z_theta, then the run's Z_phi^m, per sample
    __shared__ int tile_s;
    __shared__ double red_s[3][kSumThreads / 32];
    constexpr int n_ph = kKerr ? 3 : 2;

    const int tid = threadIdx.x, lane = tid & 31, n_seg = n_t - 1;
    const int row = lane >> 2, col = lane & 3;
    const int sbase = (tid >> 5) * (8 * G) + row;         // tile-relative sample of this lane's group 0 (group g: + 8 g)
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kRing; ++s) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    unsigned gst = 0;                       // stages consumed by this block so far: ring slot gst % kRing, parity (gst / kRing) & 1

    // Persistent block: tiles (T samples of one sparse segment of one source) are handed out by an atomic counter, so
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
    const long long i_begin = B[p] + (long long)(tile - TS[p]) * T, i_end = B[p + 1];
    double2* h = h_all ? h_all + (size_t)src * N : nullptr;
    const double2* dat = d_all ? d_all + (size_t)src * N : nullptr;
    double* partial = L.partial + ((size_t)src * max_tiles + tile) * 4;

    if (p == 0 || p == n_t) {           // outside [t_0, t_last]: h = 0 (R12)
        if (h) {
#pragma unroll
            for (int q = 0; q < Q; ++q) { long long i = i_begin + q * kSumThreads + tid; if (i < i_end) h[i] = make_double2(0.0, 0.0); }
        }
        if (want_inner && tid < 3) partial[tid] = 0.0;
        continue;
    }
    const int k = p - 1;
    const int n_steps = L.n_steps[src];
    const int n_stages = stages_for(n_steps);
    const double2* gsrc = reinterpret_cast<const double2*>(L.pack) + ((size_t)src * n_seg + k) * L.max_stages * kStageD2;

    // ---- producer prologue: thread 0 arms the ring with the first kRing - 1 stages of this tile
    if (tid == 0) {
        for (int s = 0; s < kRing - 1 && s < n_stages; ++s) {
            const int b = (gst + s) % kRing;
            mbar_expect_tx(&full[b], kStageBytes);
            bulk_g2s(&ring[b][0], gsrc + (size_t)s * kStageD2, kStageBytes, &full[b]);
        }
    }

    // ---- per-sample setup (overlaps the first copies), one thread per sample: dx, the phase factors, rho^1..4
    const double tk = t_all[(size_t)src * n_t + k];
    const dd* cph = coef_phase + ((size_t)src * n_seg + k) * 4 * n_ph;     // [4][n_ph] dd
#pragma unroll
    for (int q = 0; q < Q; ++q) {
        const int sx = q * kSumThreads + tid;
        long long i = i_begin + sx;
        if (i >= i_end) i = i_end - 1;                              // tail samples recompute the last one, never stored
        const double dx = __dsub_rn(sample_time(t0, dt, i), tk);
        double2 zp, r1;
        phase_factor(cph + 0, n_ph, dx, &zp.x, &zp.y);
        phase_factor(cph + n_ph - 1, n_ph, dx, &r1.x, &r1.y);
        zphi_s[sx] = zp;
        const double2 r2 = cmul(r1, r1);
        rpow_s[sx][0] = r1; rpow_s[sx][1] = r2; rpow_s[sx][2] = cmul(r2, r1); rpow_s[sx][3] = cmul(r2, r2);
        if (kKerr) {
            double2 zt;
            phase_factor(cph + 1, n_ph, dx, &zt.x, &zt.y);
            kerr_s[sx] = zt;
            kerr_s[T + sx] = make_double2(1.0, 0.0);
        }
    }
    __syncthreads();

    // lane state, per group g (sample sbase + 8 g, unit column col): (c, s) = rho^nu of the current step's nu = 4 blk + col;
    // z4 = rho^4; P of the current run; S, D accumulators of the run (C fragments: power col, (re, im)); H = sum over runs
    double cs_c[G], cs_s[G], z4r[G], z4i[G], pr[G], pi[G];
    double2 accS[G], accD[G], H[G];
#pragma unroll
    for (int g = 0; g < G; ++g) {
        const double2 z4 = rpow_s[sbase + 8 * g][3];
        z4r[g] = z4.x; z4i[g] = z4.y;
        cs_c[g] = 1.0; cs_s[g] = 0.0; pr[g] = 1.0; pi[g] = 0.0;
        accS[g] = accD[g] = H[g] = make_double2(0.0, 0.0);
    }

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
        const double2* bp = &ring[b][0] + lane;
        const int* hdr = reinterpret_cast<const int*>(&ring[b][0] + kStageSteps * kStepD2);
        const int ns = hdr[0];
        for (int si = 0; si < ns; ++si, bp += kStepD2) {
            const int d = hdr[1 + si];
            int adv = (d >> kAdvShift) & ((1 << kAdvBits) - 1);
            if (d & kNewRun) {      // rare (once per (m, k)): close the previous run, new P, (c, s) restart from rho^col
                const int dm = (d >> kDmShift) & ((1 << kDmBits) - 1);
#pragma unroll
                for (int g = 0; g < G; ++g) {
                    H[g].x = fma(pr[g], accS[g].x, fma(-pi[g], accD[g].y, H[g].x));      // H += P_r S + i P_i D
                    H[g].y = fma(pr[g], accS[g].y, fma(pi[g], accD[g].x, H[g].y));
                    accS[g] = accD[g] = make_double2(0.0, 0.0);
                    const int sx = sbase + 8 * g;
                    const double2 zp = zphi_s[sx];
                    double2 pm = kKerr ? kerr_s[T + sx] : make_double2(pr[g], pi[g]);
                    for (int q = 0; q < dm; ++q) pm = cmul(pm, zp);
                    if (kKerr) {                                    // P = Z_phi^m Z_theta^k (k < 0: conjugate powers)
                        if (col == 0) kerr_s[T + sx] = pm;          // the 4 lanes of a row hold the same value
                        const int kk = ((d >> kKShift) & ((1 << kKBits) - 1)) - 64;
                        double2 zt = kerr_s[sx];
                        if (kk < 0) zt.y = -zt.y;
                        for (int q = 0; q < (kk < 0 ? -kk : kk); ++q) pm = cmul(pm, zt);
                    }
                    pr[g] = pm.x; pi[g] = pm.y;
                    const double2 r0 = col ? rpow_s[sx][col - 1] : make_double2(1.0, 0.0);
                    cs_c[g] = r0.x; cs_s[g] = r0.y;
                }
                if (kKerr) __syncwarp();
            }
            for (; adv > 0; --adv) {                                // usually once: nu -> nu + 4
#pragma unroll
                for (int g = 0; g < G; ++g) {
                    const double m1 = cs_s[g] * z4i[g], m2 = cs_s[g] * z4r[g], e0 = cs_c[g];
                    cs_c[g] = fma(e0, z4r[g], -m1);
                    cs_s[g] = fma(e0, z4i[g], m2);
                }
            }
            const double2 b12c = bp[0], b12s = bp[32];
#pragma unroll
            for (int g = 0; g < G; ++g) dmma884(accS[g], cs_c[g], b12c.x);
#pragma unroll
            for (int g = 0; g < G; ++g) dmma884(accD[g], cs_c[g], b12c.y);
#pragma unroll
            for (int g = 0; g < G; ++g) dmma884(accS[g], cs_s[g], b12s.x);
#pragma unroll
            for (int g = 0; g < G; ++g) dmma884(accD[g], cs_s[g], b12s.y);
        }
    }
    __syncthreads();                                                // every warp is done with rpow_s: reuse it for H
#pragma unroll
    for (int g = 0; g < G; ++g) {                                   // close the last run; H_p of sample sx, power col -> shared
        H[g].x = fma(pr[g], accS[g].x, fma(-pi[g], accD[g].y, H[g].x));
        H[g].y = fma(pr[g], accS[g].y, fma(pi[g], accD[g].x, H[g].y));
        rpow_s[sbase + 8 * g][col] = H[g];
    }
    __syncthreads();

    // ---- h = H_0 + dx (H_1 + dx (H_2 + dx H_3)), one thread per sample; optionally the tile's share of the PSD = 1 inner
    // products <d|h>, <h|h> so that a likelihood evaluation never writes h to HBM
    double s_re = 0.0, s_im = 0.0, s_hh = 0.0;
#pragma unroll
    for (int q = 0; q < Q; ++q) {
        const int sx = q * kSumThreads + tid;
        const long long i = i_begin + sx;
        if (i < i_end) {
            const double dx = __dsub_rn(sample_time(t0, dt, i), tk);
            const double2 h0 = rpow_s[sx][0], h1 = rpow_s[sx][1], h2 = rpow_s[sx][2], h3 = rpow_s[sx][3];
            const double hr = fma(fma(fma(h3.x, dx, h2.x), dx, h1.x), dx, h0.x);
            const double hi = fma(fma(fma(h3.y, dx, h2.y), dx, h1.y), dx, h0.y);
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
#define FEW_SUM_LAUNCH(INNER, KERR, DPTR)                                                                                         \
    few_sum_kernel<kSumG, kSumBlocksPerSm, INNER, KERR><<<grid, kSumThreads, 0, st>>>(                                            \
        t, (const dd*)coef_phase_dd, t0, dt, n_samples, n_t, n_src, (int)max_tiles, L, (double2*)h, DPTR)
    if (n_phase == 3) {
        if (inner) FEW_SUM_LAUNCH(true, true, (const double2*)d);
        else FEW_SUM_LAUNCH(false, true, nullptr);
    } else {
        if (inner) FEW_SUM_LAUNCH(true, false, (const double2*)d);
        else FEW_SUM_LAUNCH(false, false, nullptr);
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
