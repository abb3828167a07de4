// few_sum.cu -- S3: the interpolated summation (sec. III C, Eq. (9), Eq. (10)):
//   "the actual summation kernel evaluates the spline at the sampling rate of the output data stream.  Then, the output
//    phase and amplitude values are combined within each mode according to Eq. (1) ... A_{l,-m,-k,-n} = (-1)^{l+k} A*_{lmkn}
//    ... only compute modes for m >= 0 ... the modes in a single time step are combined."
//   h(t_i) = scale * sum_{j kept} [ Y+_j W_j + (m_j>0) (-1)^{l_j} Y-_j conj(W_j) ],  W_j = A_j(t_i) exp(-i(m_j Phi_phi + n_j Phi_r)).
//
// Three launches per call, all on the caller's stream, nothing read back to the host:
//   1. few_sum_plan_kernel  (one block per source)
//        - clips the dense sample grid to the sparse segments (first sample of every knot) and prefix-sums the
//          per-segment tile counts, so that every block of the sum kernel works inside ONE segment (uniform coefficients);
//        - orders the kept modes by (m, sign n, |n|, l) and describes them as "groups" (one (m, n) pair with a bit mask
//          of the l present) inside "runs" (one m): E_mn = Z_phi^m Z_r^n is then built by ONE complex multiply per
//          group (walking n upward from 0 with Z_r, downward with conj Z_r), shared by all l of the group;
//        - folds Y+, (-1)^l Y- and scale into 4 real constants per (m, l).
//   2. few_sum_pack_kernel  gathers the kept modes' spline coefficients into plan order, 64 contiguous bytes per mode
//        and segment (c0..c3 x re,im), so the hot loop streams them with 128-bit uniform loads.
//   3. few_sum_kernel       the hot loop.  Per thread R samples in registers; per sample the two phases are evaluated
//        ONCE in double-double (Horner on the dd coefficients, reduction by 2 pi in dd, one sincos each) giving
//        Z_phi = exp(-i Phi_phi), Z_r = exp(-i Phi_r); per mode 6 DFMA (complex cubic Horner) + 4 DFMA (S_l += A E);
//        per group 4 DFMA (E *= Z_r); per (m, l) 4 DFMA (fold into h).  Output: coalesced 16-byte stores.
// FP64 pipe only: the path is elementwise work with a reduction over modes, not a dense contraction.
#include "few_common.cuh"

namespace {

constexpr int kNSlot = FEW_MAX_L_PER_M;      // accumulators S_l per m-run
constexpr int kMaxRuns = FEW_MAX_L + 1;      // distinct m values
constexpr int kPlanThreads = 1024;
constexpr int kSumThreads = 128;
constexpr int kSumR = 2;                     // samples per thread
constexpr int kTile = kSumThreads * kSumR;   // samples per block

// group descriptor bits
constexpr int kMaskBits = 9, kAdvShift = 9, kAdvBits = 12;
constexpr int kNewSub = 1 << 21, kDirNeg = 1 << 22, kDmShift = 23, kNewRun = 1 << 30;

struct sum_layout {
    long long* bounds;   // [n_src][n_t + 2]   pseudo-segment p covers samples [bounds[p], bounds[p+1])
    int* tile_start;     // [n_src][n_t + 2]   exclusive prefix of tiles per pseudo-segment; last = total
    int* n_groups;       // [n_src]
    int* grp;            // [n_src][n_modes]
    int* order_j;        // [n_src][n_modes]   mode index of packed slot r
    int* run_mask;       // [n_src][kMaxRuns]  slot mask of each run
    double* yc;          // [n_src][kMaxRuns][kNSlot][4]
    double* pack;        // [n_src][n_t - 1][n_modes][8]
};

sum_layout sum_carve(void* ws, int n_src, int n_t, int n_modes, size_t* bytes = nullptr)
{
    few_carver c(ws);
    sum_layout L;
    L.bounds = c.take<long long>((size_t)n_src * (n_t + 2));
    L.tile_start = c.take<int>((size_t)n_src * (n_t + 2));
    L.n_groups = c.take<int>(n_src);
    L.grp = c.take<int>((size_t)n_src * n_modes);
    L.order_j = c.take<int>((size_t)n_src * n_modes);
    L.run_mask = c.take<int>((size_t)n_src * kMaxRuns);
    L.yc = c.take<double>((size_t)n_src * kMaxRuns * kNSlot * 4);
    L.pack = c.take<double>((size_t)n_src * (n_t - 1) * n_modes * 8);
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

__device__ __forceinline__ int key_m(unsigned k) { return (int)(k >> 21); }
__device__ __forceinline__ int key_dir(unsigned k) { return (int)(k >> 20) & 1; }
__device__ __forceinline__ int key_absn(unsigned k) { return (int)(k >> 8) & 0xfff; }
__device__ __forceinline__ int key_l(unsigned k) { return (int)(k & 0xff); }

__global__ void __launch_bounds__(kPlanThreads, 1)
few_sum_plan_kernel(const double* __restrict__ t_all, const int* __restrict__ l, const int* __restrict__ m,
                    const int* __restrict__ n, const int* __restrict__ keep_idx, const int* __restrict__ n_keep,
                    const double2* __restrict__ ylm_plus, const double2* __restrict__ ylm_minus,
                    const double* __restrict__ scale, double t0, double dt, long long N, int n_t, int n_modes,
                    sum_layout L, int* status)
{
    extern __shared__ unsigned plan_smem[];
    unsigned* ukey = plan_smem;                                   // [n_modes] unsorted keys
    unsigned* skey = ukey + n_modes;                              // [n_modes] sorted keys
    int* uj = reinterpret_cast<int*>(skey + n_modes);             // [n_modes]
    int* sj = uj + n_modes;                                       // [n_modes]
    unsigned short* gid = reinterpret_cast<unsigned short*>(sj + n_modes);   // [n_modes]
    unsigned short* rid = gid + n_modes;                          // [n_modes]
    int* gmask = reinterpret_cast<int*>(rid + n_modes);                      // [n_modes] (gid + rid = 4 n_modes bytes: aligned)
    __shared__ unsigned long long run_l[kMaxRuns];
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
    for (int r = tid; r < kMaxRuns; r += kPlanThreads) run_l[r] = 0ull;
    for (int q = tid; q < K; q += kPlanThreads) {
        int j = keep_idx ? keep_idx[(size_t)src * n_modes + q] : q;
        bool ok = j >= 0 && j < n_modes;
        int lj = ok ? l[j] : 2, mj = ok ? m[j] : 0, nj = ok ? n[j] : 0;
        int an = nj < 0 ? -nj : nj;
        if (!ok || lj < 2 || lj > FEW_MAX_L || mj < 0 || mj > lj || an > FEW_MAX_ABS_N) {
            atomicOr(status, FEW_DEV_BAD_MODE);
            lj = 2; mj = 0; an = 0; nj = 0; j = ok ? j : 0;
        }
        ukey[q] = ((unsigned)mj << 21) | ((nj < 0 ? 1u : 0u) << 20) | ((unsigned)an << 8) | (unsigned)lj;
        uj[q] = j;
    }
    __syncthreads();
    // ---- (c) rank sort (keys are unique for a valid mode list; ties fall back to list position)
    for (int q = tid; q < K; q += kPlanThreads) {
        unsigned key = ukey[q];
        int rank = 0;
        for (int p = 0; p < K; ++p) { unsigned kp = ukey[p]; rank += (kp < key || (kp == key && p < q)) ? 1 : 0; }
        skey[rank] = key; sj[rank] = uj[q];
    }
    __syncthreads();
    // ---- (d) group / run ids by a chunked scan of boundary flags (group count low 16 bits, run count high 16 bits)
    if (tid == 0) carry_s = 0;
    __syncthreads();
    for (int base = 0; base < K; base += kPlanThreads) {
        int r = base + tid, flag = 0;
        if (r < K) {
            unsigned key = skey[r], prev = r ? skey[r - 1] : 0u;
            bool new_run = r == 0 || key_m(key) != key_m(prev);
            bool new_grp = new_run || (key >> 8) != (prev >> 8);
            flag = (new_grp ? 1 : 0) | (new_run ? 1 << 16 : 0);
        }
        int total, incl = plan_block_scan(flag, warp_sums, &total);
        int carry = carry_s;
        if (r < K) {
            int v = carry + incl;
            gid[r] = (unsigned short)((v & 0xffff) - 1);
            int ru = (v >> 16) - 1;
            rid[r] = (unsigned short)ru;
            atomicOr(&run_l[ru], 1ull << key_l(skey[r]));
            gmask[r] = 0;
        }
        __syncthreads();
        if (tid == 0) carry_s = carry + total;
        __syncthreads();
    }
    const int G = carry_s & 0xffff, n_runs = carry_s >> 16;
    // ---- (e) slots, group masks
    for (int r = tid; r < K; r += kPlanThreads) {
        unsigned long long rl = run_l[rid[r]];
        int slot = __popcll(rl & ((1ull << key_l(skey[r])) - 1ull));
        if (__popcll(rl) > kNSlot) { atomicOr(status, FEW_DEV_TOO_MANY_L); slot = slot % kNSlot; }
        atomicOr(&gmask[gid[r]], 1 << slot);
    }
    __syncthreads();
    // ---- (f) emit descriptors, fold constants, packed order
    int* grp = L.grp + (size_t)src * n_modes;
    int* oj = L.order_j + (size_t)src * n_modes;
    double* yc = L.yc + (size_t)src * kMaxRuns * kNSlot * 4;
    const double sc = scale ? scale[src] : 1.0;
    for (int r = tid; r < K; r += kPlanThreads) {
        unsigned key = skey[r], prev = r ? skey[r - 1] : 0u;
        int j = sj[r];
        oj[r] = j;
        bool new_run = r == 0 || key_m(key) != key_m(prev);
        bool new_sub = new_run || key_dir(key) != key_dir(prev);
        bool new_grp = new_sub || key_absn(key) != key_absn(prev);
        if (new_grp) {
            int nadv = new_sub ? key_absn(key) : key_absn(key) - key_absn(prev);
            int dm = new_run ? key_m(key) - (r ? key_m(prev) : 0) : 0;
            grp[gid[r]] = gmask[gid[r]] | (nadv << kAdvShift) | (new_sub ? kNewSub : 0) | (key_dir(key) ? kDirNeg : 0) |
                          (dm << kDmShift) | (new_run ? kNewRun : 0);
        }
        // 4 real constants of the (m, l) fold:  h += Y+ S + Ybar conj(S),  Ybar = (-1)^l Y- for m > 0, else 0
        unsigned long long rl = run_l[rid[r]];
        int lj = key_l(key), slot = __popcll(rl & ((1ull << lj) - 1ull)) % kNSlot;
        double2 yp = ylm_plus[(size_t)src * n_modes + j], yb = make_double2(0.0, 0.0);
        if (key_m(key) > 0) {
            double2 ym = ylm_minus[(size_t)src * n_modes + j];
            double sg = (lj & 1) ? -1.0 : 1.0;
            yb = make_double2(sg * ym.x, sg * ym.y);
        }
        double* c = yc + ((size_t)rid[r] * kNSlot + slot) * 4;
        c[0] = sc * (yp.x + yb.x); c[1] = sc * (-yp.y + yb.y); c[2] = sc * (yp.y + yb.y); c[3] = sc * (yp.x - yb.x);
    }
    for (int r = tid; r < n_runs; r += kPlanThreads) {
        int cnt = __popcll(run_l[r]); if (cnt > kNSlot) cnt = kNSlot;
        L.run_mask[(size_t)src * kMaxRuns + r] = (1 << cnt) - 1;
    }
    if (tid == 0) L.n_groups[src] = G;
}

// coef_amp[src][k][p][2 n_modes] -> pack[src][k][r][p][re,im] for the kept modes in plan order.
__global__ void few_sum_pack_kernel(const double2* __restrict__ coef_amp, const int* __restrict__ n_keep, int n_t, int n_modes,
                                    sum_layout L)
{
    const int k = blockIdx.x, src = blockIdx.y, n_seg = n_t - 1;
    const int K = n_keep ? min(max(n_keep[src], 0), n_modes) : n_modes;
    const int* oj = L.order_j + (size_t)src * n_modes;
    const double2* in = coef_amp + ((size_t)src * n_seg + k) * 4 * n_modes;
    double2* out = reinterpret_cast<double2*>(L.pack) + ((size_t)src * n_seg + k) * n_modes * 4;
    for (int idx = threadIdx.x; idx < 4 * K; idx += blockDim.x) {
        int r = idx >> 2, p = idx & 3;
        out[idx] = in[(size_t)p * n_modes + oj[r]];
    }
}

// exp(-i Phi) for Phi = c0 + dx (c1 + dx (c2 + dx c3)) with double-double coefficients (R13, R15).
__device__ __forceinline__ void phase_factor(const dd* __restrict__ c, int stride, double dx, double* zr, double* zi)
{
    dd r = c[3 * stride];
    r = dd_add(dd_mul_d(r, dx), c[2 * stride]);
    r = dd_add(dd_mul_d(r, dx), c[stride]);
    r = dd_add(dd_mul_d(r, dx), c[0]);
    const double two_pi_hi = 6.283185307179586232e+00, two_pi_lo = 2.449293598294706414e-16;
    double kk = rint(r.hi * 1.591549430918953456e-01);
    dd q = dd_sub(r, two_prod(kk, two_pi_hi));
    q = dd_sub(q, two_prod(kk, two_pi_lo));
    double s, co;
    sincos(q.hi, &s, &co);
    *zr = fma(-q.lo, s, co);          // cos(hi + lo)
    *zi = -fma(q.lo, co, s);          // -sin(hi + lo)
}

template <int R>
__global__ void __launch_bounds__(kSumThreads)
few_sum_kernel(const double* __restrict__ t_all, const dd* __restrict__ coef_phase, double t0, double dt, long long N,
               int n_t, int n_modes, sum_layout L, double2* __restrict__ h_all)
{
    const int src = blockIdx.y, tid = threadIdx.x, n_seg = n_t - 1;
    const int* TS = L.tile_start + (size_t)src * (n_t + 2);
    const int tile = blockIdx.x;
    if (tile >= TS[n_t + 1]) return;
    // pseudo-segment of this tile: largest p with TS[p] <= tile
    int lo = 0, hi = n_t + 1;
    while (hi - lo > 1) { int mid = (lo + hi) >> 1; if (TS[mid] <= tile) lo = mid; else hi = mid; }
    const int p = lo;
    const long long* B = L.bounds + (size_t)src * (n_t + 2);
    const long long i_begin = B[p] + (long long)(tile - TS[p]) * (R * kSumThreads), i_end = B[p + 1];
    double2* h = h_all + (size_t)src * N;

    if (p == 0 || p == n_t) {           // outside [t_0, t_last]: h = 0 (R12)
#pragma unroll
        for (int r = 0; r < R; ++r) { long long i = i_begin + r * kSumThreads + tid; if (i < i_end) h[i] = make_double2(0.0, 0.0); }
        return;
    }
    const int k = p - 1;
    const double tk = t_all[(size_t)src * n_t + k];
    const dd* cph = coef_phase + ((size_t)src * n_seg + k) * 8;     // [4][2] dd

    double dx[R], zpr[R], zpi[R], zrr[R], zri[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        long long i = i_begin + r * kSumThreads + tid;
        if (i >= i_end) i = i_end - 1;                              // tail lanes recompute the last sample, never store
        dx[r] = __dsub_rn(sample_time(t0, dt, i), tk);
        phase_factor(cph + 0, 2, dx[r], &zpr[r], &zpi[r]);
        phase_factor(cph + 1, 2, dx[r], &zrr[r], &zri[r]);
    }

    double hre[R], him[R], pmr[R], pmi[R], er[R], ei[R], sti[R];
    double sre[kNSlot][R], sim[kNSlot][R];
#pragma unroll
    for (int r = 0; r < R; ++r) { hre[r] = him[r] = 0.0; pmr[r] = 1.0; pmi[r] = 0.0; er[r] = 1.0; ei[r] = 0.0; sti[r] = zri[r]; }
#pragma unroll
    for (int s = 0; s < kNSlot; ++s)
#pragma unroll
        for (int r = 0; r < R; ++r) sre[s][r] = sim[s][r] = 0.0;

    const int G = L.n_groups[src];
    const int* grp = L.grp + (size_t)src * n_modes;
    const int* run_mask = L.run_mask + (size_t)src * kMaxRuns;
    const double* yc = L.yc + (size_t)src * kMaxRuns * kNSlot * 4;
    const double2* cp = reinterpret_cast<const double2*>(L.pack) + ((size_t)src * n_seg + k) * n_modes * 4;

    auto fold = [&](int run) {
        const int rm = run_mask[run];
        const double* c = yc + (size_t)run * kNSlot * 4;
#pragma unroll
        for (int s = 0; s < kNSlot; ++s) {
            if (rm & (1 << s)) {
                const double a = c[4 * s], b = c[4 * s + 1], cc = c[4 * s + 2], d = c[4 * s + 3];
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    hre[r] = fma(a, sre[s][r], hre[r]); hre[r] = fma(b, sim[s][r], hre[r]);
                    him[r] = fma(cc, sre[s][r], him[r]); him[r] = fma(d, sim[s][r], him[r]);
                    sre[s][r] = 0.0; sim[s][r] = 0.0;
                }
            }
        }
    };

    int run = -1;
    for (int g = 0; g < G; ++g) {
        const int d = grp[g];
        if (d & kNewRun) {
            if (run >= 0) fold(run);
            ++run;
            const int dm = (d >> kDmShift) & 0x7f;
            for (int q = 0; q < dm; ++q) {
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    double a = pmr[r] * zpr[r] - pmi[r] * zpi[r];
                    pmi[r] = pmr[r] * zpi[r] + pmi[r] * zpr[r];
                    pmr[r] = a;
                }
            }
        }
        if (d & kNewSub) {
            const double sg = (d & kDirNeg) ? -1.0 : 1.0;
#pragma unroll
            for (int r = 0; r < R; ++r) { er[r] = pmr[r]; ei[r] = pmi[r]; sti[r] = sg * zri[r]; }
        }
        const int nadv = (d >> kAdvShift) & ((1 << kAdvBits) - 1);
        for (int q = 0; q < nadv; ++q) {
#pragma unroll
            for (int r = 0; r < R; ++r) {
                double a = er[r] * zrr[r] - ei[r] * sti[r];
                ei[r] = er[r] * sti[r] + ei[r] * zrr[r];
                er[r] = a;
            }
        }
#pragma unroll
        for (int s = 0; s < kNSlot; ++s) {
            if (d & (1 << s)) {
                const double2 c0 = __ldg(cp), c1 = __ldg(cp + 1), c2 = __ldg(cp + 2), c3 = __ldg(cp + 3);
                cp += 4;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    double ar = fma(fma(fma(c3.x, dx[r], c2.x), dx[r], c1.x), dx[r], c0.x);
                    double ai = fma(fma(fma(c3.y, dx[r], c2.y), dx[r], c1.y), dx[r], c0.y);
                    sre[s][r] = fma(ar, er[r], sre[s][r]); sre[s][r] = fma(-ai, ei[r], sre[s][r]);
                    sim[s][r] = fma(ar, ei[r], sim[s][r]); sim[s][r] = fma(ai, er[r], sim[s][r]);
                }
            }
        }
    }
    if (run >= 0) fold(run);

#pragma unroll
    for (int r = 0; r < R; ++r) {
        long long i = i_begin + r * kSumThreads + tid;
        if (i < i_end) __stcs(&h[i], make_double2(hre[r], him[r]));
    }
}

size_t plan_smem_bytes(int n_modes) { return (size_t)n_modes * (4 + 4 + 4 + 4 + 2 + 2 + 4) + 16; }

}  // namespace

extern "C" size_t few_sum_waveform_workspace(int n_src, int n_t, int n_modes, long long n_samples)
{
    (void)n_samples;
    if (n_src <= 0 || n_t < 2 || n_modes <= 0) return 0;
    size_t bytes = 0;
    sum_carve(nullptr, n_src, n_t, n_modes, &bytes);
    return bytes;
}

extern "C" int few_sum_waveform(few_ctx* ctx, const double* t, const double* coef_amp, const double* coef_phase_dd,
                                const int* l, const int* m, const int* n, const int* keep_idx, const int* n_keep,
                                const double* ylm_plus, const double* ylm_minus, const double* scale,
                                double t0, double dt, long long n_samples, double* h,
                                int n_src, int n_t, int n_modes, void* workspace, size_t workspace_bytes, void* stream)
{
    FEW_REQUIRE(ctx && t && coef_amp && coef_phase_dd && l && m && n && ylm_plus && ylm_minus, FEW_ERR_INVALID_ARG, "NULL argument");
    FEW_REQUIRE((keep_idx == nullptr) == (n_keep == nullptr), FEW_ERR_INVALID_ARG, "keep_idx and n_keep must both be NULL or both be set");
    FEW_REQUIRE(n_src > 0 && n_modes > 0 && n_samples >= 0, FEW_ERR_INVALID_ARG, "sizes must be positive");
    FEW_REQUIRE(n_t >= 4, FEW_ERR_TOO_FEW_POINTS, "n_t < 4");
    FEW_REQUIRE(dt > 0.0 && isfinite(dt) && isfinite(t0), FEW_ERR_INVALID_ARG, "dt must be positive and finite");
    FEW_REQUIRE(n_src <= 65535 && n_modes <= 65535, FEW_ERR_LIMIT, "n_src or n_modes > 65535");
    if (n_samples == 0) return FEW_OK;
    FEW_REQUIRE(h != nullptr, FEW_ERR_INVALID_ARG, "h is NULL");
    FEW_REQUIRE(workspace && ((uintptr_t)workspace % 256) == 0 &&
                    workspace_bytes >= few_sum_waveform_workspace(n_src, n_t, n_modes, n_samples),
                FEW_ERR_WORKSPACE, "workspace NULL, misaligned or too small");
    size_t psm = plan_smem_bytes(n_modes);
    FEW_REQUIRE(psm <= (size_t)ctx->smem_optin, FEW_ERR_LIMIT, "n_modes too large for the plan kernel's shared memory");
    long long max_tiles = (n_samples + kTile - 1) / kTile + n_t + 1;
    FEW_REQUIRE(max_tiles < 2147483647LL, FEW_ERR_LIMIT, "n_samples too large");
    cudaStream_t st = (cudaStream_t)stream;
    sum_layout L = sum_carve(workspace, n_src, n_t, n_modes);

    FEW_CUDA_CHECK(cudaFuncSetAttribute(few_sum_plan_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)psm));
    few_sum_plan_kernel<<<n_src, kPlanThreads, psm, st>>>(t, l, m, n, keep_idx, n_keep, (const double2*)ylm_plus,
                                                          (const double2*)ylm_minus, scale, t0, dt, n_samples, n_t, n_modes, L,
                                                          ctx->d_status);
    FEW_CUDA_CHECK(cudaGetLastError());
    few_sum_pack_kernel<<<dim3(n_t - 1, n_src), 256, 0, st>>>((const double2*)coef_amp, n_keep, n_t, n_modes, L);
    FEW_CUDA_CHECK(cudaGetLastError());
    if (ctx->profile) FEW_CUDA_CHECK(cudaEventRecord(ctx->ev_sum[0], st));
    few_sum_kernel<kSumR><<<dim3((unsigned)max_tiles, n_src), kSumThreads, 0, st>>>(t, (const dd*)coef_phase_dd, t0, dt, n_samples,
                                                                                   n_t, n_modes, L, (double2*)h);
    FEW_CUDA_CHECK(cudaGetLastError());
    if (ctx->profile) { FEW_CUDA_CHECK(cudaEventRecord(ctx->ev_sum[1], st)); ctx->profile_valid = 1; }
    return FEW_OK;
}
