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
// per instruction; a lane carries (c_nu, s_nu) of ONE sample and ONE of the four nu, read from a per-tile table of rho^nu in
// tensor memory (or, for lists with more than 8 nu-blocks, stepped by a three-term recurrence in registers).  Per sample and
// unit: 32 FMA in DMMAs (40 scalar operations in the per-(m,n)-pair DFMA form this replaces).  The same IEEE FMA arithmetic on
// the same pipe; what changes is that a DMMA reads 4 registers per 8 FMA where a DFMA reads 3 per FMA, which is what held the
// DFMA form at 0.75 of the pipe.
//
// Three launches per call, all on the caller's stream, nothing read back to the host:
//   1. few_sum_plan_kernel  (one block per source): clips the dense sample grid to the sparse segments and prefix-sums
//        the per-segment tile counts (every block of the sum kernel works inside ONE segment, so its coefficients are
//        block-uniform); orders the kept modes by (m, k, |n|, sign n, l) and cuts them into STEPS: the kept units of one run
//        whose nu fall into one aligned block of four (4b .. 4b+3), with a descriptor saying how (c, s) is reached.
//   2. few_sum_pack_kernel  (one block per source and segment): forms the four B matrices of every step from the kept modes'
//        spline coefficients and Y+, Ybar, scale, in DMMA fragment order, as a stream of stages (16 steps x 1 KB + header).
//   3. few_sum_kernel       the hot loop.  Stages arrive in shared memory through a ring of TMA bulk copies
//        (cp.async.bulk + mbarrier) and are read with conflict-free 128-bit loads.  Per sample the phases are evaluated ONCE in
//        double-double (Horner, reduction by 2 pi, one sincos each).  Output: coalesced 16-byte streaming stores.
#include <algorithm>
#include <vector>
#include "few_common.cuh"

namespace {

constexpr int kPlanThreads = 1024;
constexpr int kPlanSmemElems = 16384;         // 128 KB of (key, mode) words: the plan kernel's in-shared-memory sort capacity
// The block shape below (4 warps, 16-step stages, ring of 2) is the only one that is built and tested; the others that were
// measured (8 and 16 warps per block, 4- to 64-step stages, rings of 3 to 6) are in profiles/r02_variants.md.
constexpr int kSumWarps = 4;                  // warps per block (16 warps are resident per SM)
constexpr int kSumThreads = 32 * kSumWarps;
constexpr int kSumG = 4;                      // groups of 8 samples per warp
constexpr int kSumBlocksPerSm = 16 / kSumWarps;      // resident blocks per SM, recurrence instantiation (register budget 65536 / (32 * 16))
constexpr int kSumTabBlocksPerSm = 16 / kSumWarps;   // resident blocks per SM, table instantiation (16 x 32 lanes x 128 columns = all of tensor memory)
constexpr int kTile = (kSumThreads / 32) * 8 * kSumG;   // samples per block
constexpr int kStageSteps = 16;               // steps per stage: what a stage boundary costs (warp barrier, done counter, mbarrier wait) is
                                              // paid per stage, and the ring's depth does not matter
constexpr int kStepD2 = 64;                   // a step's B fragments: [2][32 lanes] double2 = 1 KB
constexpr int kHdrInts = kStageSteps < 32 ? 32 : 128;           // header: [i] descriptor of step i, [kStageSteps] steps in the stage
constexpr int kStageBytes = kStageSteps * kStepD2 * 16 + kHdrInts * 4;
constexpr int kStageD2 = kStageBytes / 16;    // stage size in double2
constexpr int kRing = 2;                      // stages in flight per block

// step descriptor
constexpr int kNewRun = 1;                    // first step of a run (m, k): close the previous run, P <- Z_phi^m Z_theta^k, (c, s) <- rho^col
constexpr int kAdvShift = 1, kAdvBits = 12;   // multiplications by rho^4 before the step's DMMAs
constexpr int kDmShift = 13, kDmBits = 7;     // m increment of a new run
constexpr int kKShift = 20, kKBits = 7;       // polar index of the run, offset by 64 (Kerr-shaped lists, |k| <= FEW_MAX_ABS_K)
constexpr int kSingle = 1 << 27;              // run with m = 0: no mirror, beta = 0, hence D = S: the c half is accumulated in S, the s half in D
constexpr int kSlotShift = 28, kSlotBits = 3; // table slot of the step's block nu >> 2 (sources in table mode)
constexpr int kTabSlots = 8;                  // distinct blocks nu >> 2 a source may use in table mode (the paper's grid: nu <= 31 -> 8)

// A tile of the sum kernel as the plan kernel hands it over (one 32-byte record, two 16-byte loads): first sample and sample
// count, pseudo-segment p (-1: no tile; 0: outside the trajectory, h = 0), the source, and the number of coefficient
// stages the tile consumes (0 for tiles without a summation), and the source's mode (1 table, 0 recurrence: which of the two
// instantiations of the sum kernel takes the tile).
struct __align__(16) tile_rec { long long i_begin; int count; int p; int n_stages; int src; int mode; int pad1; };   // n_stages, mode: filled by load_rec from src_info

struct sum_layout {
    long long* bounds;   // [n_src][n_t + 2]   pseudo-segment p covers samples [bounds[p], bounds[p+1])
    int* tile_start;     // [n_src][n_t + 2]   exclusive prefix of tiles per pseudo-segment; last = total
    int* n_steps;        // [n_src]            number of steps
    int2* src_info;      // [n_src]            (coefficient stages per tile, mode: 1 table / 0 recurrence) of the source
    int* blk_list;       // [n_src][8]         table mode: the distinct blocks nu >> 2 of the source, ascending (slot -> block), -1 = unused
    int* mode_count;     // [2]                sources in recurrence mode [0] / table mode [1] (zeroed before the plan kernel)
    tile_rec* tiles;     // [n_src][max_tiles] what the plan kernel hands every tile, so that a warp finds its work with one record
    int* desc;           // [n_src][cap]       step descriptors
    int* u_lo;           // [n_src][cap][8]    sorted range [u_lo, u_hi) of the modes of (step, nu & 3, sign of n)
    int* u_hi;           // [n_src][cap][8]
    int* order_j;        // [n_src][n_modes]   mode index of sorted position r
    double* yfold;       // [n_src][n_modes][4] scale * (Y+ re, Y+ im, Ybar re, Ybar im) of sorted position r
    double* pack;        // [n_src][n_t - 1][max_stages][kStageBytes / 8]
    double* partial;     // [n_src][max_tiles][4 warps][4]  per-warp sums of conj(d) h (re, im) and |h|^2 (fused inner products)
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

// Steps per source the workspace is laid out for: the default covers any kept list of the call (step_capacity), a caller's
// bound (few_set_max_steps) can only lower it.  A list that needs more sets FEW_DEV_SPARSE_LIST in the plan kernel either way.
__host__ inline int effective_cap(int n_modes, int max_steps)
{
    const int def = step_capacity(n_modes);
    return (max_steps > 0 && max_steps < def) ? max_steps : def;
}

sum_layout sum_carve(void* ws, int n_src, int n_t, int n_modes, long long n_samples, int max_steps, size_t* bytes = nullptr)
{
    few_carver c(ws);
    sum_layout L;
    L.cap = effective_cap(n_modes, max_steps);
    L.max_stages = stages_for(L.cap);
    L.bounds = c.take<long long>((size_t)n_src * (n_t + 2));
    L.tile_start = c.take<int>((size_t)n_src * (n_t + 2));
    L.n_steps = c.take<int>(n_src);
    L.src_info = c.take<int2>(n_src);
    L.blk_list = c.take<int>((size_t)n_src * kTabSlots);
    L.mode_count = c.take<int>(2);
    const long long mt = sum_max_tiles(n_samples, n_t);
    L.max_tiles = (int)(mt < 2147483647LL ? mt : 2147483647LL);
    L.tiles = c.take<tile_rec>((size_t)n_src * (size_t)mt);
    L.desc = c.take<int>((size_t)n_src * L.cap);
    L.u_lo = c.take<int>((size_t)n_src * L.cap * 8);
    L.u_hi = c.take<int>((size_t)n_src * L.cap * 8);
    L.order_j = c.take<int>((size_t)n_src * n_modes);
    L.yfold = c.take<double>((size_t)n_src * n_modes * 4);
    L.pack = c.take<double>((size_t)n_src * (n_t - 1) * L.max_stages * (kStageBytes / 8));
    L.partial = c.take<double>((size_t)n_src * (size_t)mt * (kSumThreads / 32) * 4);
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
    if (!(tk == tk)) return 0;       // NaN knot (reported elsewhere as not increasing): any in-range value, without the searches
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
                    const int* __restrict__ n_t_src, int n_t, int n_modes, int smem_elems, sum_layout L, int* status)
{
    extern __shared__ unsigned long long plan_smem[];             // [smem_elems]
    unsigned long long* plan_sorted;                              // [n_pow2] (key << 32 | mode index), sorted ascending
    __shared__ int warp_sums[32];
    __shared__ int carry_s;

    const int src = blockIdx.x, tid = threadIdx.x;
    const double* t = t_all + (size_t)src * n_t;
    // Blocks of a source work side by side: blockIdx.y >= 1 lay out the tiles (a), (e) -- that needs the time grids only --
    // and blockIdx.y == 0 orders the kept modes and cuts them into steps (b)-(d).
    if (blockIdx.y >= 1) {
    // ---- (a) sample ranges of the pseudo-segments and their tile prefix.  ns = the source's own knot count (ragged batches;
    // = n_t otherwise): pseudo-segments 0 .. ns, the arrays keep the stride n_t + 2 and the tile total also goes to TS[n_t + 1]
    const int ns = few_knots(n_t_src, src, n_t, status);
    long long* B = L.bounds + (size_t)src * (n_t + 2);
    int* TS = L.tile_start + (size_t)src * (n_t + 2);
    for (int k = tid; k < ns; k += kPlanThreads) {
        if (k + 1 < ns && !(t[k + 1] > t[k])) atomicOr(status, FEW_DEV_NOT_INCREASING);
        if (k <= ns - 2) B[k + 1] = first_index(t[k], t0, dt, N, false);
        else { B[ns] = first_index(t[ns - 1], t0, dt, N, true); B[ns + 1] = N; B[0] = 0; }
    }
    __syncthreads();
    if (tid < 32) {           // warp 0: prefix over ns + 1 pseudo-segments, 32 at a time
        int carry = 0;
        for (int base = 0; base <= ns; base += 32) {
            int p = base + tid;
            int cnt = 0;
            if (p <= ns) { long long c = B[p + 1] - B[p]; if (c < 0) c = 0; cnt = (int)((c + kTile - 1) / kTile); }
            int v = cnt;
            for (int o = 1; o < 32; o <<= 1) { int u = __shfl_up_sync(0xffffffffu, v, o); if (tid >= o) v += u; }
            if (p <= ns) TS[p] = carry + v - cnt;
            carry += __shfl_sync(0xffffffffu, v, 31);
        }
        if (tid == 0) { TS[ns + 1] = carry; TS[n_t + 1] = carry; }
    }
    __syncthreads();
    // ---- (e) tile records: tile q of pseudo-segment p covers samples [B[p] + (q - TS[p]) kTile, ...) inside [B[p], B[p+1]).
    // The gridDim.y - 1 tile blocks of a source each recompute (a) (cheap; they write the same B, TS) and share the records:
    // a thread takes tiles q, q + stride, ... and finds p by binary search (24.6 k records from one block took 36 us)
    {
        tile_rec* rec = L.tiles + (size_t)src * L.max_tiles;
        const int n_tiles = TS[ns + 1];
        const int tb = gridDim.y - 1, ry = blockIdx.y - 1;
        for (int q = ry * kPlanThreads + tid; q < L.max_tiles; q += tb * kPlanThreads) {
            tile_rec r;
            r.n_stages = 0; r.src = src; r.mode = 0; r.pad1 = 0;
            if (q < n_tiles) {
                int lo = 0, hi = ns + 1;                         // largest p with TS[p] <= q
                while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (TS[mid] <= q) lo = mid; else hi = mid; }
                const long long b0 = B[lo], b1 = B[lo + 1];
                r.i_begin = b0 + (long long)(q - TS[lo]) * kTile;
                const long long left = b1 - r.i_begin;
                r.count = (int)(left < kTile ? left : kTile);
                r.p = lo == ns ? 0 : lo;                         // after the last knot = before the first: outside, h = 0
            } else {
                r.i_begin = 0; r.count = 0; r.p = -1;
            }
            rec[q] = r;
        }
    }
    return;
    }   // blockIdx.y >= 1

    int* ulo = L.u_lo + (size_t)src * L.cap * 8;
    int* uhi = L.u_hi + (size_t)src * L.cap * 8;
    for (int q = tid; q < L.cap * 8; q += kPlanThreads) { ulo[q] = 0; uhi[q] = 0; }      // empty (step, nu & 3, sign) slots
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
    if (n_pow2 <= kPlanThreads && smem_elems >= 2 * kPlanThreads) {
        // up to 1024 keys (every list of the Schwarzschild grid after selection): one element per thread; compare-exchange
        // partners less than a warp apart are reached by shuffles, the others through shared memory, double-buffered: 15 block
        // barriers instead of 55
        unsigned long long v = tid < n_pow2 ? plan_sorted[tid] : ~0ull;
        __syncthreads();
        unsigned long long* xbuf = plan_smem;                      // [2][kPlanThreads]
        int pp = 0;
        for (int size = 2; size <= kPlanThreads; size <<= 1) {
            for (int stride = size >> 1; stride > 0; stride >>= 1) {
                unsigned long long o;
                if (stride >= 32) {
                    xbuf[pp * kPlanThreads + tid] = v;
                    __syncthreads();
                    o = xbuf[pp * kPlanThreads + (tid ^ stride)];
                    pp ^= 1;
                } else {
                    o = __shfl_xor_sync(0xffffffffu, v, stride);
                }
                const bool up = (tid & size) == 0, lower = (tid & stride) == 0;
                const bool take_min = lower == up;
                v = (take_min == (o < v)) ? o : v;
            }
        }
        __syncthreads();
        if (tid < n_pow2) plan_sorted[tid] = v;
        __syncthreads();
    } else if (in_smem) {
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
    // ---- (d0) the distinct blocks nu >> 2 of the list: at most kTabSlots of them -> table mode (the sum kernel keeps rho^nu of
    // every sample in shared memory), else recurrence mode
    __shared__ unsigned blk_mask[(FEW_MAX_ABS_N + 1) / 4 / 32];
    __shared__ int mode_s;
    if (tid < (FEW_MAX_ABS_N + 1) / 4 / 32) blk_mask[tid] = 0u;
    __syncthreads();
    for (int r = tid; r < K; r += kPlanThreads) {
        const int blk = key_absn((unsigned)(plan_sorted[r] >> 32)) >> 2;
        atomicOr(&blk_mask[blk >> 5], 1u << (blk & 31));
    }
    __syncthreads();
    if (tid == 0) {
        int cnt = 0;
        int* bl = L.blk_list + (size_t)src * kTabSlots;
        for (int q = 0; q < kTabSlots; ++q) bl[q] = -1;
        for (int wd = 0; wd < (FEW_MAX_ABS_N + 1) / 4 / 32; ++wd) {
            unsigned mk = blk_mask[wd];
            while (mk) { const int b = __ffs(mk) - 1; mk &= mk - 1; if (cnt < kTabSlots) bl[cnt] = wd * 32 + b; ++cnt; }
        }
        mode_s = cnt <= kTabSlots ? 1 : 0;
        atomicAdd(&L.mode_count[mode_s], 1);
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
                    int slot = 0;                               // rank of blk among the source's distinct blocks
                    for (int wd = 0; wd < (blk >> 5); ++wd) slot += __popc(blk_mask[wd]);
                    slot += __popc(blk_mask[blk >> 5] & ((1u << (blk & 31)) - 1u));
                    desc[s] = (new_run ? kNewRun : 0) | (adv << kAdvShift) | (dm << kDmShift) | ((key_k(key) + 64) << kKShift) |
                              (key_m(key) == 0 ? kSingle : 0) | ((slot & ((1 << kSlotBits) - 1)) << kSlotShift);
                }
                const int slot = s * 8 + (key_absn(key) & 3) * 2 + key_neg(key);      // (step, nu & 3, sign) range slot
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
        L.src_info[src] = make_int2(stages_for(S), mode_s);
    }
}

// The four B matrices of every step, in DMMA.8x8x4 fragment order, written as the stage stream the sum kernel consumes.
// Lane L of a warp supplies B[k = L & 3][o = L >> 2]: unit k of the step (nu = 4 blk + k), output o = 2 p + part (power p of
// dx, part 0 = re, 1 = im).  A step is 1 KB: [0][L] = (B1c, B2c), [1][L] = (B1s, B2s) as double2 (conflict-free LDS.128).
__global__ void __launch_bounds__(1024) few_sum_pack_kernel(const double2* __restrict__ coef_amp, const int* __restrict__ n_t_src, int n_t,
                                                            int n_modes, sum_layout L)
{
    const int seg = blockIdx.x, src = blockIdx.y, n_seg = n_t - 1;
    if (n_t_src) {      // ragged batch: segments beyond the source's own count do not exist (their coefficients were never written).
        int v = n_t_src[src];                              // A bad count is replaced by 4 exactly as few_knots() does in the plan, fit and
        if (v < 4 || v > n_t) v = n_t < 4 ? n_t : 4;       // selection kernels (which also report it), so that every stage the plan's tiles
        if (seg >= v - 1) return;                          // point at is written in this call and the sum kernel never reads stale memory
    }
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
    for (int idx = threadIdx.x; idx < n_stages * kHdrInts; idx += blockDim.x) {     // header: [i] descriptor i, [kStageSteps] steps in the stage
        const int st = idx / kHdrInts, q = idx % kHdrInts;
        int v = 0;
        const int cnt = min(kStageSteps, S - st * kStageSteps);
        if (q == kStageSteps) v = cnt;
        else if (q < cnt) v = desc[st * kStageSteps + q];
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

// All NP phase factors of a sample at once, z[p] = exp(-i Phi_p(dx)), c = [4][NP] dd coefficients: the NP evaluations are
// independent dependent-chains, written side by side so that they overlap (a lone chain of ~70 scalar FP64 instructions
// between other warps' DMMAs costs the pipe 4-9 cycles per instruction, profiles/r02_fp64_pipe_probes.md).  Not inlined: the
// sum kernel's code must stay small enough for the instruction caches (it ran a fifth slower with 28 KB of per-tile code).
template <int NP>
__device__ __noinline__ void phase_factors(const dd* __restrict__ c, double dx, double2* __restrict__ z)
{
    dd r[NP];
#pragma unroll
    for (int p = 0; p < NP; ++p) r[p] = dd_add_d(c[2 * NP + p], __dmul_rn(c[3 * NP + p].hi, dx));
#pragma unroll
    for (int p = 0; p < NP; ++p) r[p] = dd_add_fast(dd_mul_d(r[p], dx), c[NP + p]);
#pragma unroll
    for (int p = 0; p < NP; ++p) r[p] = dd_add_fast(dd_mul_d(r[p], dx), c[p]);
    const double p1 = 0x1.921fb54000000p+2, p2 = 0x1.10b4611800000p-28, p3 = 0x1.313198a2e0370p-59;   // 2 pi = p1 + p2 + p3
    double q[NP], ql[NP];
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        const double kk = rint(r[p].hi * 1.591549430918953456e-01);
        q[p] = fma(-kk, p2, fma(-kk, p1, r[p].hi));       // the inner fma is exact
        ql[p] = fma(-kk, p3, r[p].lo);
    }
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        double s, co;
        sincos(q[p], &s, &co);
        z[p] = make_double2(fma(-ql[p], s, co), -fma(ql[p], co, s));     // cos(q + ql), -sin(q + ql)
    }
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

// Tensor memory (TMEM, 256 KB per SM: 128 lanes x 512 columns x 32 bit) used as per-thread scratch: with the 32x32b shape,
// thread i of warp w reads and writes lane 32 (w % 4) + i, i.e. its own row of the block's allocation.  The table instantiation
// keeps rho^nu of its 8 G samples there: 16 bytes per (table slot, group) and thread = 128 columns for G = 4, four resident
// blocks per SM fill the 512 columns.  tcgen05.ld/st are warp-collective and asynchronous (wait::ld / wait::st).
__device__ __forceinline__ void tmem_alloc(unsigned* smem_dst, unsigned ncols)
{
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(smem_dst)), "r"(ncols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(unsigned taddr, unsigned ncols)
{
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tmem_st_x4(unsigned taddr, double2 v)
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(taddr), "r"(__double2loint(v.x)),
                 "r"(__double2hiint(v.x)), "r"(__double2loint(v.y)), "r"(__double2hiint(v.y))
                 : "memory");
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
// four (c, s) pairs = 16 columns of this thread's lane
__device__ __forceinline__ void tmem_ld_x16(unsigned taddr, double2 (&v)[4])
{
    unsigned r[16];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
                   "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                 : "r"(taddr)
                 : "memory");
    tmem_wait_ld();
#pragma unroll
    for (int g = 0; g < 4; ++g) v[g] = make_double2(__hiloint2double(r[4 * g + 1], r[4 * g]), __hiloint2double(r[4 * g + 3], r[4 * g + 2]));
}

__device__ __forceinline__ tile_rec load_rec(const tile_rec* p, const int2* __restrict__ src_info)
{
    const int4 a = __ldg(reinterpret_cast<const int4*>(p)), b = __ldg(reinterpret_cast<const int4*>(p) + 1);
    tile_rec r;
    r.i_begin = ((long long)(unsigned)a.y << 32) | (unsigned)a.x; r.count = a.z; r.p = a.w;
    r.src = b.y; r.pad1 = 0;
    const int2 info = __ldg(src_info + r.src);          // per source: stages per tile, mode (a cached load)
    r.n_stages = r.p <= 0 ? 0 : info.x;
    r.mode = info.y;
    return r;
}

// The sum kernel.  A block is 4 warps that share ONE thing: the ring of coefficient stages.  Everything else is per warp:
// a warp owns 8 G samples of every tile of its block (tile = 4 warps x 8 G samples inside one sparse segment of one source,
// so the coefficients are block-uniform), evaluates their phases, runs the step loop and stores their h, and never meets
// another warp at a barrier.  Tiles are assigned statically (block b takes tiles b, b + grid, ...; every tile of a source
// costs the same), each warp reads the tile records itself, two tiles ahead.  Ring protocol: full[slot] is an mbarrier the
// TMA bulk copy completes; when a warp is done with a slot it bumps done[slot], and the LAST of the 4 warps refills the slot
// with the stage kRing ahead in the block's stage stream (walking into the next tiles' records where the stream crosses a
// tile boundary).  So warps drift apart by at most the ring depth and wait only for data.  (Blocks of 8 or 16 warps measured
// 1-4 % slower on short kept lists, profiles/r02_variants.md; they are not built.)
// G: groups of 8 samples per warp.  kKerr: Kerr-shaped mode lists (Eq. (1), Eq. (19)): a third phase factor
// Z_theta, runs are (m, k) with P = Z_phi^m Z_theta^k.  The hot loop is the same.
// kTab: where the A operands (c, s) = rho^nu come from.  On the FP64 pipe a scalar instruction issued between the DMMAs of
// other warps costs far more than its two cycles, so the table instantiation computes rho^nu of every
// sample ONCE per tile -- rho^nu does not depend on the run (m, k) -- into the warp's rows of the block's tensor-memory
// allocation, in DMMA fragment order, and the step loop is loads and DMMAs only; it takes the sources whose lists use at most kTabSlots distinct blocks nu >> 2
// (the paper's grid: nu <= 31).  The recurrence instantiation steps x_b = rho^(4 b + col) in registers (2 DFMA per group and
// step) and takes every other source.  Both are launched; each works on the tiles whose record names its mode.
template <int G, bool kKerr, bool kTab>
struct sum_smem {
    static constexpr int W = 8 * G, kWarps = kSumThreads / 32;
    __align__(128) double2 ring[kRing][kStageD2];
    __align__(8) unsigned long long full[kRing];
    int done[kRing];                                            // warps finished with the slot's current stage
    __align__(16) double2 zphi[kWarps][W];                      // Z_phi = exp(-i Phi_phi) per sample
    __align__(16) double2 rpow[kWarps][W][4];                   // rho, rho^2, rho^3, rho^4 per sample; after the loop: H_p, p = 0..3
    __align__(16) double2 pcur[kWarps][W];                      // P = Z_phi^m Z_theta^k of the current run, per sample
    __align__(16) double2 hacc[kTab ? 1 : kWarps][G][32];       // per lane and group: H = sum over the closed runs (table mode: in rpow,
                                                                // whose rho^1..4 are dead once the table is built; same index map)
    __align__(16) double2 kerr[kKerr ? kWarps : 1][2][kKerr ? W : 1];   // kKerr: Z_theta, the run's Z_phi^m, per sample
    unsigned tmem_base;                                         // kTab: the block's tensor-memory allocation (rho^nu table)
};
template <int G, bool kKerr, bool kTab> constexpr size_t sum_smem_bytes() { return sizeof(sum_smem<G, kKerr, kTab>); }

template <int G, int kBlocksPerSm, bool kInner, bool kKerr, bool kTab>
__global__ void __launch_bounds__(kSumThreads, kBlocksPerSm)
few_sum_kernel(const double* __restrict__ t_all, const dd* __restrict__ coef_phase, double t0, double dt, long long N,
               int n_t, int n_src, int max_tiles, sum_layout L, double2* __restrict__ h_all, const double2* __restrict__ d_all)
{
    constexpr bool want_inner = kInner;      // the inner-product epilogue is compiled out of the plain waveform kernel
    constexpr int W = 8 * G, kWarps = kSumThreads / 32, QW = (W + 31) / 32;     // W: samples per warp and tile
    using smem_t = sum_smem<G, kKerr, kTab>;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    smem_t& sm = *reinterpret_cast<smem_t*>(smem_raw);
    auto& ring = sm.ring; auto& full = sm.full; auto& done_s = sm.done; auto& zphi_s = sm.zphi; auto& rpow_s = sm.rpow;
    auto& pcur_s = sm.pcur; auto& kerr_s = sm.kerr;
    constexpr int n_ph = kKerr ? 3 : 2;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, n_seg = n_t - 1;
    const int row = lane >> 2, col = lane & 3;
    const long long total_tiles = (long long)n_src * max_tiles;
    const long long stride = gridDim.x;
    const double2* pack = reinterpret_cast<const double2*>(L.pack);

    // issue the stage `s` stages after the start of tile sequence number `i` of this block (record ri; rn = record of i + 1)
    // into ring slot `slot`: walks forward through the block's tiles where s runs past a tile's stages
    auto issue = [&](long long i, int s, tile_rec ri, const tile_rec& rn, unsigned slot) {
        long long j = i;
        auto mine = [](const tile_rec& r) { return r.mode == (kTab ? 1 : 0) ? r.n_stages : 0; };
        while (s >= mine(ri)) {
            s -= mine(ri);
            ++j;
            const long long tg = blockIdx.x + j * stride;
            if (tg >= total_tiles) return;                          // the stream has ended
            ri = (j == i + 1) ? rn : load_rec(L.tiles + tg, L.src_info);
        }
        const double2* src = pack + ((size_t)ri.src * n_seg + (ri.p - 1)) * L.max_stages * kStageD2 + (size_t)s * kStageD2;
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");    // the warps' reads of the slot precede the copy's writes
        mbar_expect_tx(&full[slot], kStageBytes);
        bulk_g2s(&ring[slot][0], src, kStageBytes, &full[slot]);
    };

    if (L.mode_count[kTab ? 1 : 0] == 0) return;       // no source in this instantiation's mode
    constexpr unsigned kTmemCols = 16 * kTabSlots * ((kWarps + 3) / 4);     // 128 columns per warp: (c, s) x G = 4 groups x kTabSlots slots per thread
    if (kTab && warp == 0) tmem_alloc(&sm.tmem_base, kTmemCols);
    tile_rec cur, nxt;
    cur.p = -1; cur.n_stages = 0; cur.count = 0; cur.i_begin = 0; cur.src = 0; cur.mode = 0; cur.pad1 = 0;
    nxt = cur;
    if ((long long)blockIdx.x < total_tiles) cur = load_rec(L.tiles + blockIdx.x, L.src_info);
    if (blockIdx.x + stride < total_tiles) nxt = load_rec(L.tiles + blockIdx.x + stride, L.src_info);
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kRing; ++s) { mbar_init(&full[s], 1); done_s[s] = 0; }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        if ((long long)blockIdx.x < total_tiles) {
#pragma unroll 1
            for (int s = 0; s < kRing; ++s) issue(0, s, cur, nxt, s);
        }
    }
    if (kTab) asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();                        // the only block-wide barrier of the kernel (besides the one before the TMEM release)
    if (kTab) asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    // this warp's lanes (32 (warp % 4) ...) and columns of the allocation
    const unsigned tmem_row = kTab ? sm.tmem_base + ((unsigned)((warp & 3) * 32) << 16) + (unsigned)(warp >> 2) * (16 * kTabSlots) : 0u;
    // H of lane (row, col), group g: [g][lane] of the warp = [sample 8 g + row][col] of rpow (32 g + lane either way)
    double2* const hacc_w = kTab ? &rpow_s[warp][0][0] : &sm.hacc[kTab ? 0 : warp][0][0];
    unsigned gst = 0;                       // stages consumed by this warp so far: ring slot gst % kRing, use number gst / kRing

    for (long long i = 0;; ++i) {
    const long long tg = blockIdx.x + i * stride;
    if (tg >= total_tiles) break;
    tile_rec nn = cur;                      // record of tile i + 2: loaded now, needed at the end of this tile
    nn.p = -1; nn.n_stages = 0; nn.count = 0;
    if (tg + 2 * stride < total_tiles) nn = load_rec(L.tiles + tg + 2 * stride, L.src_info);
    if (cur.p >= 0 && cur.mode == (kTab ? 1 : 0)) {
    const int src = cur.src, p = cur.p;
    const long long w_begin = cur.i_begin + warp * W;               // this warp's samples: [w_begin, w_begin + w_count)
    const int w_count = min(max(cur.count - warp * W, 0), W);
    double2* h = h_all ? h_all + (size_t)src * N : nullptr;
    const double2* dat = d_all ? d_all + (size_t)src * N : nullptr;
    double* partial = L.partial + (((size_t)src * max_tiles + (size_t)(tg - (long long)src * max_tiles)) * kWarps + warp) * 4;

    if (cur.n_stages == 0) {                // outside [t_0, t_last] (R12), or nothing kept: h = 0
        if (h) {
#pragma unroll
            for (int q = 0; q < QW; ++q) { const int sx = q * 32 + lane; if (sx < w_count) h[w_begin + sx] = make_double2(0.0, 0.0); }
        }
        if (want_inner && lane < 3) partial[lane] = 0.0;
    } else {
    const int k = p - 1;
    const int n_stages = cur.n_stages;

    // ---- per-sample setup, one lane per sample of the warp: dx, the phase factors, rho^1..4 (and the rho^nu table)
    const double tk = t_all[(size_t)src * n_t + k];
    const dd* cph = coef_phase + ((size_t)src * n_seg + k) * 4 * n_ph;     // [4][n_ph] dd
#pragma unroll
    for (int q = 0; q < QW; ++q) {
        const int sx = q * 32 + lane;
        if (sx < W) {
            long long is = w_begin + sx;
            const long long i_last = cur.i_begin + cur.count - 1;
            if (is > i_last) is = i_last;                           // tail samples recompute the last one, never stored
            const double dx = __dsub_rn(sample_time(t0, dt, is), tk);
            double2 zf[n_ph];
            phase_factors<n_ph>(cph, dx, zf);
            const double2 zp = zf[0], r1 = zf[n_ph - 1];
            zphi_s[warp][sx] = zp;
            pcur_s[warp][sx] = make_double2(1.0, 0.0);
            const double2 r2 = cmul(r1, r1), r3 = cmul(r2, r1), r4 = cmul(r2, r2);
            if (kKerr) {
                const double2 zt = zf[n_ph > 2 ? 1 : 0];
                kerr_s[warp][0][sx] = zt;
                kerr_s[warp][1][sx] = make_double2(1.0, 0.0);
            }
            rpow_s[warp][sx][0] = r1; rpow_s[warp][sx][1] = r2; rpow_s[warp][sx][2] = r3; rpow_s[warp][sx][3] = r4;
        }
    }
    __syncwarp();
    if (kTab) {
        // table mode: x_b = rho^(4 b + col) of this lane's samples, for the blocks b the source uses (slot -> block, ascending,
        // in L.blk_list), by the three-term recurrence (below), into the lane's own tensor-memory row: column 16 slot + 4 g
        // holds (c, s) of group g.  (A rolled loop of four levels: the per-tile code must stay small for the instruction caches.)
        const int4* blp = reinterpret_cast<const int4*>(L.blk_list + (size_t)src * kTabSlots);
        const int4 bl0 = __ldg(blp), bl1 = __ldg(blp + 1);          // slot -> block, ascending, -1 = unused (blocks <= 255)
        static_assert(kTabSlots == 8 && FEW_MAX_ABS_N / 4 < 256, "the block list is packed into 8 bytes");
        unsigned long long bls = 0ull;                              // byte q = block of slot q, n_slots of them
        int n_slots = 0;
        {
            const int bl[8] = {bl0.x, bl0.y, bl0.z, bl0.w, bl1.x, bl1.y, bl1.z, bl1.w};
#pragma unroll
            for (int q = 0; q < 8; ++q) if (bl[q] >= 0) { bls |= (unsigned long long)(unsigned)bl[q] << (8 * q); n_slots = q + 1; }
        }
        double2 xa[G], xb[G];                                       // x_b, x_{b-1} of the G groups: G independent chains
        double twg[G];
#pragma unroll
        for (int g = 0; g < G; ++g) {
            const int sx = 8 * g + row;
            const double2 xm = rpow_s[warp][sx][3 - col];
            xa[g] = col ? rpow_s[warp][sx][col - 1] : make_double2(1.0, 0.0);
            xb[g] = make_double2(xm.x, -xm.y);
            twg[g] = 2.0 * rpow_s[warp][sx][3].x;
        }
        int slot = 0, target = n_slots ? (int)(bls & 0xffu) : -1;
        // four levels of the recurrence at a time, their 32 DFMA back to back, then the stores of those of the four blocks that
        // the list uses: a warp that leaves the FP64 pipe between two levels (the stores, a branch) waits for it again
#pragma unroll 1
        for (int b = 0; target >= 0; b += 4) {
            double2 l1[G], l2[G], l3[G], l4[G];
#pragma unroll
            for (int g = 0; g < G; ++g) { l1[g].x = fma(twg[g], xa[g].x, -xb[g].x); l1[g].y = fma(twg[g], xa[g].y, -xb[g].y); }
#pragma unroll
            for (int g = 0; g < G; ++g) { l2[g].x = fma(twg[g], l1[g].x, -xa[g].x); l2[g].y = fma(twg[g], l1[g].y, -xa[g].y); }
#pragma unroll
            for (int g = 0; g < G; ++g) { l3[g].x = fma(twg[g], l2[g].x, -l1[g].x); l3[g].y = fma(twg[g], l2[g].y, -l1[g].y); }
#pragma unroll
            for (int g = 0; g < G; ++g) { l4[g].x = fma(twg[g], l3[g].x, -l2[g].x); l4[g].y = fma(twg[g], l3[g].y, -l2[g].y); }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                if (b + q == target) {
#pragma unroll
                    for (int g = 0; g < G; ++g) tmem_st_x4(tmem_row + 16 * slot + 4 * g, q == 0 ? xa[g] : q == 1 ? l1[g] : q == 2 ? l2[g] : l3[g]);
                    ++slot; bls >>= 8;
                    target = slot < n_slots ? (int)(bls & 0xffu) : -1;
                }
            }
#pragma unroll
            for (int g = 0; g < G; ++g) { xb[g] = l3[g]; xa[g] = l4[g]; }
        }
        tmem_wait_st();
        __syncwarp();                       // rho^1..4 have been read: their storage becomes H (below)
    }

    // Lane state, per group g (sample 8 g + row of the warp, unit column col).  S, D: accumulators of the run (C fragments:
    // power col of dx, (re, im)).  P and H = sum over the closed runs of P_r S + i P_i D are touched once per run and live in
    // shared memory.  Recurrence mode only: x_b = rho^(4 b + col) = (c, s) of block b obeys the three-term recurrence
    // x_{b+1} = 2 cos(4 Phi_r) x_b - x_{b-1} (one DFMA per component; its error after b steps is at most b^2 u whatever the
    // angle: the Green's function sin(j theta) / sin(theta) is bounded by j), started from x_0 = rho^col and
    // x_{-1} = conj(rho^(4 - col)).  The two most recent blocks live in (xc, xs) and (yc, ys); `odd` says which is current,
    // so that a step overwrites the older one in place.
    constexpr int GR = kTab ? 1 : G;
    double xc[GR], xs[GR], yc[GR], ys[GR], tw[GR];
    double2 accS[G], accD[G];
#pragma unroll
    for (int g = 0; g < G; ++g) {
        if (!kTab) {
            tw[g % GR] = 2.0 * rpow_s[warp][8 * g + row][3].x;
            xc[g % GR] = 1.0; xs[g % GR] = 0.0; yc[g % GR] = 1.0; ys[g % GR] = 0.0;
        }
        accS[g] = accD[g] = make_double2(0.0, 0.0);
        hacc_w[32 * g + lane] = make_double2(0.0, 0.0);
    }
    bool single = false;                    // the current run has m = 0: D = S, and both accumulators gather S (c half, s half)
    bool odd = false;                       // (recurrence mode) the current block is in (yc, ys)

    for (int st = 0; st < n_stages; ++st) {
        const unsigned slot = gst % kRing;
        mbar_wait(&full[slot], (gst / kRing) & 1u);
        ++gst;
        const double2* bp = &ring[slot][0] + lane;
        const int* hdr = reinterpret_cast<const int*>(&ring[slot][0] + kStageSteps * kStepD2);
        int4 d4 = *reinterpret_cast<const int4*>(hdr), d8 = kStageSteps > 4 ? *(reinterpret_cast<const int4*>(hdr) + 1) : make_int4(0, 0, 0, 0);
        static_assert(kStageSteps == 4 || kStageSteps == 8 || (kStageSteps > 8 && kStageSteps < 128), "descriptors: 4 or 8 in registers, more from the header");
        const int ns = min(hdr[kStageSteps], kStageSteps);   // the clamp keeps the walk inside the ring slot whatever the header holds
        for (int si = 0; si < ns; ++si, bp += kStepD2) {
            int d;
            if (kStageSteps <= 8) {
                d = d4.x;
                d4.x = d4.y; d4.y = d4.z; d4.z = d4.w;
                if (kStageSteps > 4) { d4.w = d8.x; d8.x = d8.y; d8.y = d8.z; d8.z = d8.w; }
            } else {
                d = hdr[si];
            }
            double2 b12c, b12s;
            double2 av[G];                                          // table mode: (c, s) of this lane's unit, per group
            auto load_step = [&]() {
                b12c = bp[0]; b12s = bp[32];
                if constexpr (kTab) {
                    const int ts = (d >> kSlotShift) & ((1 << kSlotBits) - 1);
                    static_assert(!kTab || G == 4, "the table instantiation is written for G = 4 (16 columns per slot)");
                    tmem_ld_x16(tmem_row + 16 * ts, av);
                }
            };
            if (d & kNewRun) {      // rare (once per (m, k)): close the previous run, new P, (recurrence) x restarts from rho^col
                // One burst: every shared-memory operand first (P and H of the 4 groups; Z_phi and P of the lane's own sample),
                // then the scalar FP64 instructions in waves of independent ones (the new P's complex product, the 2 G inner
                // and the 2 G outer FMAs of H += P_r S + i P_i D), then the stores.  A warp that stalls between two FP64
                // instructions waits ~200 cycles behind the other warps' DMMAs before the pipe takes its next one
                // (profiles/r02_sum_kernel.md), so the close costs one such wait instead of one per group; and it runs BEFORE
                // this step's operand loads, while their 24 registers are free (with them live ptxas copied the 16 table
                // registers of every step: slower than no burst at all).
                {
                    double2 Pg[G], Hg[G];
#pragma unroll
                    for (int g = 0; g < G; ++g) { Pg[g] = pcur_s[warp][8 * g + row]; Hg[g] = hacc_w[32 * g + lane]; }
                    // the new run's P = P Z_phi^dm (Z_theta^k), one lane per sample, in the same burst: operands first
                    static_assert(W == 32, "one lane per sample");
                    const double2 zp1 = zphi_s[warp][lane];
                    double2 pm1 = kKerr ? kerr_s[warp][1][lane] : pcur_s[warp][lane];
                    double2 zt1 = kKerr ? kerr_s[warp][0][lane] : make_double2(1.0, 0.0);
                    __syncwarp();                                   // every lane has read the old P
                    {
                        const int dm = (d >> kDmShift) & ((1 << kDmBits) - 1);
                        for (int e = 0; e < dm; ++e) pm1 = cmul(pm1, zp1);
                        if (kKerr) {
                            kerr_s[warp][1][lane] = pm1;
                            const int kk = ((d >> kKShift) & ((1 << kKBits) - 1)) - 64;
                            if (kk < 0) zt1.y = -zt1.y;
                            for (int e = 0; e < (kk < 0 ? -kk : kk); ++e) pm1 = cmul(pm1, zt1);
                        }
                        pcur_s[warp][lane] = pm1;
                    }
                    if (single) {
#pragma unroll
                        for (int g = 0; g < G; ++g) { accS[g].x += accD[g].x; accS[g].y += accD[g].y; accD[g] = accS[g]; }
                    }
#pragma unroll
                    for (int g = 0; g < G; ++g) {
                        Hg[g].x = fma(-Pg[g].y, accD[g].y, Hg[g].x);
                        Hg[g].y = fma(Pg[g].y, accD[g].x, Hg[g].y);
                    }
#pragma unroll
                    for (int g = 0; g < G; ++g) {
                        Hg[g].x = fma(Pg[g].x, accS[g].x, Hg[g].x);
                        Hg[g].y = fma(Pg[g].x, accS[g].y, Hg[g].y);
                    }
#pragma unroll
                    for (int g = 0; g < G; ++g) {
                        hacc_w[32 * g + lane] = Hg[g]; accS[g] = accD[g] = make_double2(0.0, 0.0);
                        if (!kTab) {
                            const int sx = 8 * g + row;
                            const double2 x0 = col ? rpow_s[warp][sx][col - 1] : make_double2(1.0, 0.0), xm = rpow_s[warp][sx][3 - col];
                            xc[g % GR] = x0.x; xs[g % GR] = x0.y; yc[g % GR] = xm.x; ys[g % GR] = -xm.y;
                        }
                    }
                }
                __syncwarp();                                       // the new P is visible to the next close
                single = (d & kSingle) != 0;
                odd = false;
            }
            load_step();
            if (!kTab) {
                for (int adv = (d >> kAdvShift) & ((1 << kAdvBits) - 1); adv > 0; --adv) {   // usually once: block b -> b + 1, over block b - 1
                    if (!odd) {
#pragma unroll
                        for (int g = 0; g < GR; ++g) { yc[g] = fma(tw[g], xc[g], -yc[g]); ys[g] = fma(tw[g], xs[g], -ys[g]); }
                    } else {
#pragma unroll
                        for (int g = 0; g < GR; ++g) { xc[g] = fma(tw[g], yc[g], -xc[g]); xs[g] = fma(tw[g], ys[g], -xs[g]); }
                    }
                    odd = !odd;
                }
#pragma unroll
                for (int g = 0; g < G; ++g) av[g] = odd ? make_double2(yc[g % GR], ys[g % GR]) : make_double2(xc[g % GR], xs[g % GR]);
            }
#pragma unroll
            for (int g = 0; g < G; ++g) dmma884(accS[g], av[g].x, b12c.x);
            if (!single) {
#pragma unroll
                for (int g = 0; g < G; ++g) dmma884(accD[g], av[g].x, b12c.y);
            }
            // m = 0: the s half goes to the idle D accumulators (S = accS + accD at the close), so that two DMMAs on one
            // accumulator are 8 instructions apart, as in the other runs, instead of 4 (a dependent DMMA waits ~200 cycles)
            if (single) {
#pragma unroll
                for (int g = 0; g < G; ++g) dmma884(accD[g], av[g].y, b12s.x);
            } else {
#pragma unroll
                for (int g = 0; g < G; ++g) dmma884(accS[g], av[g].y, b12s.x);
#pragma unroll
                for (int g = 0; g < G; ++g) dmma884(accD[g], av[g].y, b12s.y);
            }
        }
        __syncwarp();                                               // every lane has read the slot
        if (lane == 0) {                                            // (the slot's data has been consumed: the loads fed DMMAs)
            if (atomicAdd(&done_s[slot], 1) == kWarps - 1) {        // the last of the 4 warps refills the slot
                done_s[slot] = 0;
                issue(i, st + kRing, cur, nxt, slot);
            }
        }
    }
#pragma unroll
    for (int g = 0; g < G; ++g) {                                   // close the last run; H_p of sample sx, power col -> shared
        const int sx = 8 * g + row;
        const double2 P = pcur_s[warp][sx];
        if (single) { accS[g].x += accD[g].x; accS[g].y += accD[g].y; accD[g] = accS[g]; }
        const double2 dd_ = accD[g];
        double2 Hg = hacc_w[32 * g + lane];
        Hg.x = fma(P.x, accS[g].x, fma(-P.y, dd_.y, Hg.x));
        Hg.y = fma(P.x, accS[g].y, fma(P.y, dd_.x, Hg.y));
        rpow_s[warp][sx][col] = Hg;                                 // (rho^1..4 of this sample are not needed any more)
    }
    __syncwarp();

    // ---- h = H_0 + dx (H_1 + dx (H_2 + dx H_3)), one lane per sample; optionally the warp's share of the PSD = 1 inner
    // products <d|h>, <h|h> so that a likelihood evaluation never writes h to HBM
    double s_re = 0.0, s_im = 0.0, s_hh = 0.0;
#pragma unroll
    for (int q = 0; q < QW; ++q) {
        const int sx = q * 32 + lane;
        if (sx < w_count) {
            const long long is = w_begin + sx;
            const double dx = __dsub_rn(sample_time(t0, dt, is), tk);
            const double2 h0 = rpow_s[warp][sx][0], h1 = rpow_s[warp][sx][1], h2 = rpow_s[warp][sx][2], h3 = rpow_s[warp][sx][3];
            const double hr = fma(fma(fma(h3.x, dx, h2.x), dx, h1.x), dx, h0.x);
            const double hi = fma(fma(fma(h3.y, dx, h2.y), dx, h1.y), dx, h0.y);
            if (h) __stcs(&h[is], make_double2(hr, hi));
            if (want_inner) {
                if (dat) {
                    const double2 dv = __ldcs(&dat[is]);
                    s_re = fma(dv.x, hr, fma(dv.y, hi, s_re));      // Re conj(d) h
                    s_im = fma(dv.x, hi, fma(-dv.y, hr, s_im));     // Im conj(d) h
                }
                s_hh = fma(hr, hr, fma(hi, hi, s_hh));
            }
        }
    }
    if (want_inner) {                   // fixed butterfly over the lanes -> the same bits every run
#pragma unroll
        for (int o = 16; o; o >>= 1) {
            s_re += __shfl_xor_sync(0xffffffffu, s_re, o);
            s_im += __shfl_xor_sync(0xffffffffu, s_im, o);
            s_hh += __shfl_xor_sync(0xffffffffu, s_hh, o);
        }
        if (lane == 0) { partial[0] = s_re; partial[1] = s_im; partial[2] = s_hh; }
    }
    __syncwarp();                       // the warp's shared arrays are rewritten by the next tile's setup
    }   // tile with a summation
    }   // tile exists
    cur = nxt; nxt = nn;
    }   // this block's tiles
    if (kTab) {
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        if (warp == 0) tmem_dealloc(sm.tmem_base, kTmemCols);
    }
}

// inner[src] = 2 dt * (sum over the source's tiles and their warps of the partials): Eq. (16) with S_n = 1 by Parseval.  One block per
// source; thread q adds tiles q, q + 256, ... in order, then a fixed tree: deterministic.
constexpr int kInnerThreads = 256;
__global__ void __launch_bounds__(kInnerThreads)
few_sum_inner_kernel(sum_layout L, int n_t, int max_tiles, double dt, double* __restrict__ inner)
{
    __shared__ double red[3][kInnerThreads / 32];
    const int src = blockIdx.x, tid = threadIdx.x;
    const int n_tiles = L.tile_start[(size_t)src * (n_t + 2) + n_t + 1];
    const double* P = L.partial + (size_t)src * max_tiles * (kSumThreads / 32) * 4;
    double a = 0.0, b = 0.0, c = 0.0;
    for (int q = tid; q < n_tiles * (kSumThreads / 32); q += kInnerThreads) { a += P[4 * (size_t)q]; b += P[4 * (size_t)q + 1]; c += P[4 * (size_t)q + 2]; }
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

int few_sum_check_limits(const few_ctx* ctx, int n_src, int n_t, int n_modes, long long n_samples, int n_phase)
{
    FEW_REQUIRE(n_src <= 65535 && n_t <= 65535, FEW_ERR_LIMIT, "n_src or n_t > 65535");
    FEW_REQUIRE((size_t)plan_smem_elems(n_modes) * 8 <= (size_t)ctx->smem_optin, FEW_ERR_LIMIT, "plan kernel's shared memory exceeds the device limit");
    const size_t smem_tab = n_phase == 3 ? sum_smem_bytes<kSumG, true, true>() : sum_smem_bytes<kSumG, false, true>();
    const size_t smem_rec = n_phase == 3 ? sum_smem_bytes<kSumG, true, false>() : sum_smem_bytes<kSumG, false, false>();
    FEW_REQUIRE(smem_tab <= (size_t)ctx->smem_optin && smem_rec <= (size_t)ctx->smem_optin, FEW_ERR_LIMIT,
                "sum kernel's shared memory exceeds the device limit");
    const long long max_tiles = sum_max_tiles(n_samples, n_t);
    FEW_REQUIRE(max_tiles < 2147483647LL, FEW_ERR_LIMIT, "n_samples too large");
    FEW_REQUIRE(max_tiles * n_src < 2147483647LL - 65536, FEW_ERR_LIMIT, "n_src * n_samples too large");
    return FEW_OK;
}

extern "C" size_t few_sum_waveform_workspace_ex(int n_src, int n_t, int n_modes, long long n_samples, int max_steps)
{
    if (n_src <= 0 || n_t < 2 || n_modes <= 0 || n_samples < 0) return 0;
    size_t bytes = 0;
    sum_carve(nullptr, n_src, n_t, n_modes, n_samples, max_steps, &bytes);
    return bytes;
}

extern "C" size_t few_sum_waveform_workspace(int n_src, int n_t, int n_modes, long long n_samples)
{
    return few_sum_waveform_workspace_ex(n_src, n_t, n_modes, n_samples, 0);
}

extern "C" int few_set_max_steps(few_ctx* ctx, int max_steps)
{
    FEW_REQUIRE(ctx != nullptr, FEW_ERR_INVALID_ARG, "ctx is NULL");
    FEW_REQUIRE(max_steps >= 0, FEW_ERR_INVALID_ARG, "max_steps must be >= 0 (0 = the default capacity)");
    ctx->max_steps = max_steps;
    return FEW_OK;
}

extern "C" int few_max_steps_for_modes(const int* m_host, const int* k_host, const int* n_host, int n_modes)
{
    FEW_REQUIRE(m_host && n_host && n_modes > 0, FEW_ERR_INVALID_ARG, "NULL argument or n_modes <= 0");
    // Valid lists (0 <= m <= FEW_MAX_L, |k| <= FEW_MAX_ABS_K, |n| <= FEW_MAX_ABS_N) are counted in a bitmap, a few microseconds for
    // the paper's grid (few_waveform_host does this on every call); anything else goes through a sort, so that the count is
    // right for any input and the kernels are the ones to report a bad mode.
    constexpr int kNuBlocks = FEW_MAX_ABS_N / 4 + 1, kKSpan = 2 * FEW_MAX_ABS_K + 1;
    const int k_span = k_host ? kKSpan : 1;
    std::vector<unsigned long long> bits(((size_t)(FEW_MAX_L + 1) * k_span * kNuBlocks + 63) / 64, 0ull);
    bool in_range = true;
    int count = 0;
    for (int j = 0; j < n_modes && in_range; ++j) {      // a step = one (m, k) run x one aligned block of four |n|: count the distinct (m, k, |n| >> 2)
        const int mm = m_host[j], kk = k_host ? k_host[j] : 0;
        const long long nu = n_host[j] < 0 ? -(long long)n_host[j] : (long long)n_host[j];
        if (mm < 0 || mm > FEW_MAX_L || kk < -FEW_MAX_ABS_K || kk > FEW_MAX_ABS_K || nu > FEW_MAX_ABS_N) { in_range = false; break; }
        const size_t bit = ((size_t)mm * k_span + (size_t)(k_host ? kk + FEW_MAX_ABS_K : 0)) * kNuBlocks + (size_t)(nu >> 2);
        const unsigned long long mask = 1ull << (bit & 63);
        if (!(bits[bit >> 6] & mask)) { bits[bit >> 6] |= mask; ++count; }
    }
    if (in_range) return count;
    std::vector<long long> keys((size_t)n_modes);
    for (int j = 0; j < n_modes; ++j) {
        const long long nu = n_host[j] < 0 ? -(long long)n_host[j] : (long long)n_host[j];
        keys[j] = ((long long)m_host[j] << 40) ^ (((long long)(k_host ? k_host[j] : 0) + 1024) << 24) ^ (nu >> 2);
    }
    std::sort(keys.begin(), keys.end());
    return (int)(std::unique(keys.begin(), keys.end()) - keys.begin());
}

extern "C" int few_sum_waveform_ragged(few_ctx* ctx, const double* t, const int* n_t_src, const double* coef_amp, const double* coef_phase_dd,
                                       int n_phase, const int* l, const int* m, const int* k, const int* n, const int* keep_idx,
                                       const int* n_keep, const double* ylm_plus, const double* ylm_minus, const double* scale,
                                       const double* factor, double t0, double dt, long long n_samples, double* h, const double* d,
                                       double* inner, int n_src, int n_t, int n_modes, void* workspace, size_t workspace_bytes, void* stream)
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
                    workspace_bytes >= few_sum_waveform_workspace_ex(n_src, n_t, n_modes, n_samples, ctx->max_steps),
                FEW_ERR_WORKSPACE, "workspace NULL, misaligned or too small");
    {   // every size limit, before the first launch
        const int lim = few_sum_check_limits(ctx, n_src, n_t, n_modes, n_samples, n_phase);
        if (lim != FEW_OK) return lim;
    }
    const int plan_elems = plan_smem_elems(n_modes);
    const size_t psm = (size_t)plan_elems * 8;
    const long long max_tiles = sum_max_tiles(n_samples, n_t);
    sum_layout L = sum_carve(workspace, n_src, n_t, n_modes, n_samples, ctx->max_steps);

    const int plan_tile_blocks = n_src >= 64 ? 1 : (64 / n_src < 8 ? 64 / n_src : 8);     // tile blocks per source: 8 for one waveform
    FEW_CUDA_CHECK(cudaMemsetAsync(L.mode_count, 0, 2 * sizeof(int), st));
    FEW_CUDA_CHECK(cudaFuncSetAttribute(few_sum_plan_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)psm));
    few_sum_plan_kernel<<<dim3(n_src, 1 + plan_tile_blocks), kPlanThreads, psm, st>>>(t, l, m, k, n, keep_idx, n_keep, (const double2*)ylm_plus,
                                                          (const double2*)ylm_minus, scale, (const double2*)factor, t0, dt, n_samples,
                                                          n_t_src, n_t, n_modes, plan_elems, L, ctx->d_status);
    FEW_LAUNCHED(ctx);
    // few blocks (one waveform): 1024 threads finish a segment's 4 x pairs items in one sweep; a batch fills the SMs with
    // several 256-thread blocks each, which hides the dependent index -> coefficient loads better
    const int pack_threads = (long long)(n_t - 1) * n_src < 2LL * ctx->sm_count ? 1024 : 256;
    few_sum_pack_kernel<<<dim3(n_t - 1, n_src), pack_threads, 0, st>>>((const double2*)coef_amp, n_t_src, n_t, n_modes, L);
    FEW_LAUNCHED(ctx);
    if (ctx->profile) FEW_CUDA_CHECK(cudaEventRecord(ctx->ev_sum[0], st));
    // both instantiations are launched: the table one (rho^nu of the 8 nu-blocks in use kept in tensor memory) takes the sources
    // whose lists fit its table, the recurrence one the others; an instantiation with no source returns at once
    const long long want = max_tiles * n_src;
#define FEW_SUM_LAUNCH(INNER, KERR, DPTR)                                                                                         \
    do {                                                                                                                          \
        auto ktab = few_sum_kernel<kSumG, kSumTabBlocksPerSm, INNER, KERR, true>;                                                 \
        auto krec = few_sum_kernel<kSumG, kSumBlocksPerSm, INNER, KERR, false>;                                                   \
        const size_t smem_tab = sum_smem_bytes<kSumG, KERR, true>(), smem_rec = sum_smem_bytes<kSumG, KERR, false>();             \
        FEW_CUDA_CHECK(cudaFuncSetAttribute(ktab, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_tab));                   \
        FEW_CUDA_CHECK(cudaFuncSetAttribute(krec, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_rec));                   \
        const long long res_tab = (long long)ctx->sm_count * kSumTabBlocksPerSm, res_rec = (long long)ctx->sm_count * kSumBlocksPerSm; \
        ktab<<<(unsigned)(want < res_tab ? want : res_tab), kSumThreads, smem_tab, st>>>(                                         \
            t, (const dd*)coef_phase_dd, t0, dt, n_samples, n_t, n_src, (int)max_tiles, L, (double2*)h, DPTR);                    \
        FEW_LAUNCHED(ctx);                                                                                                        \
        krec<<<(unsigned)(want < res_rec ? want : res_rec), kSumThreads, smem_rec, st>>>(                                         \
            t, (const dd*)coef_phase_dd, t0, dt, n_samples, n_t, n_src, (int)max_tiles, L, (double2*)h, DPTR);                    \
    } while (0)
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

extern "C" int few_sum_waveform_kerr(few_ctx* ctx, const double* t, const double* coef_amp, const double* coef_phase_dd, int n_phase,
                                     const int* l, const int* m, const int* k, const int* n, const int* keep_idx, const int* n_keep,
                                     const double* ylm_plus, const double* ylm_minus, const double* scale, const double* factor,
                                     double t0, double dt, long long n_samples, double* h, const double* d, double* inner,
                                     int n_src, int n_t, int n_modes, void* workspace, size_t workspace_bytes, void* stream)
{
    return few_sum_waveform_ragged(ctx, t, nullptr, coef_amp, coef_phase_dd, n_phase, l, m, k, n, keep_idx, n_keep, ylm_plus, ylm_minus,
                                   scale, factor, t0, dt, n_samples, h, d, inner, n_src, n_t, n_modes, workspace, workspace_bytes, stream);
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
