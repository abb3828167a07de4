// few_select.cu -- S2: the Mode Selector (sec. III D): "taking arrays of the power within each mode at each
// sparse time step ... operates entirely within each time step.  It sorts the individual modes in descending order and
// computes a cumulative summation ... where the additional power contributed by an individual mode falls below a user
// provided threshold related to the total power emitted (eps) at that time step (the final entry in the cumulative sum)
// ... the union of all contributing modes across all time steps".
//
// Entries of a row (one source, one sparse step): every (l,m,n) plus the (l,-m,-n) mirror of each m>0 mode, each with its
// own power (R4).  With the row sorted by power descending (ties: lower entry index first, R7) and C the
// inclusive cumulative sum, the entry of rank r is kept iff r == 0 or C_{r-1} < (1-eps) C_last (R5).
//
// What the procedure defines is a SET, and the set is fixed by one number: C_{r-1} of an entry is G(key) = the summed power
// of all entries with a strictly larger key (plus earlier ties), G is monotone in the key, so the kept entries are exactly
// those with key >= kappa, kappa = min{k : G(k) < (1-eps) C_last}.  The kernels therefore SELECT instead of sorting the row
// (select_core, one block per row, nothing but the row's amplitudes read from HBM):
//   1. coarse: the key's top 14 bits are the binary exponent of the power and 3 mantissa bits.  A binary search over these buckets, each
//      step one masked block reduction, finds the bucket B in which the cumulative sum crosses the threshold.  Every entry
//      in a higher bucket is kept, every entry in a lower one dropped.
//   2. fine: the entries of bucket B are compacted into shared memory, rank-sorted by (power descending, entry index
//      ascending) and cumulatively summed in that order on top of the power above the bucket: this is the definition's
//      sort + cumsum, applied only where it can change the answer.  Ties need no special case.
//   3. fallback (more entries in the bucket than the shared arrays hold, e.g. a row of equal powers): a 63-step MSB-first
//      radix select on the full 64-bit pattern, ties at kappa resolved by entry index with an 18-step select.
// select_core sees the row through an `Entries` policy with one member, for_each(f): f(key, entry index, chain):
//   reg_entries     keys held in registers -- the fast kernel's candidates (few_select_row_fast_kernel: entries below
//                   eps*total/(4 n) are certainly dropped; the few hundred to ~1500 others are compacted and selected);
//   stream_entries  keys recomputed from the amplitudes on every pass (the row stays in L2) -- rows of any length: the
//                   Kerr-shaped grid's 78 507 entries, and the rows the fast kernel hands over (flat spectra, degenerate eps).
// The owners of the kept entries are OR-ed into a per-source bitmap; a last kernel compacts it into ascending keep_idx
// and n_keep.  (History: in-shared-memory LSD radix sort + scan 128 us per 7137-entry row; 63-step
// select alone 44 us; keys of the whole row in registers 26 us; this version ~11 us, profiles/r01d_kernels.md.)
#include "few_common.cuh"

namespace {

constexpr int kSelThreads = 256;
constexpr int kSelWarps = kSelThreads / 32;
constexpr int kPrepThreads = 1024;
constexpr int kBucketMax = 512;   // entries of the threshold's bucket that the fine step sorts in shared memory
constexpr int kBucketShift = 49;  // bucket of a key = its top 14 bits: the power's binary exponent and 3 mantissa bits (an eighth of a binade)

struct sel_layout {
    int* owner;       // [n_modes]   owner mode of mirror entry e - n_modes   (shared by sources)
    int* n_entries;   // [1]
    double* y2;       // [n_src][2 n_modes]  |Y|^2 per entry
    unsigned* bitmap; // [n_src][words]
    int* mirror_e;    // [n_modes]   entry index of the mirror of mode j, -1 if it has none   (shared by sources)
    double* y2m;      // [n_src][n_modes]    |Y_{l,-m}|^2 by mode (the mirror's weight beside the primary's)
    int* fb_list;     // [n_src * n_t]       rows left to the general kernel by the fast one
    int* fb_count;    // [1]
};

__host__ __device__ inline int sel_words(int n_modes) { return (n_modes + 31) / 32; }

sel_layout sel_carve(void* ws, int n_src, int n_t, int n_modes, size_t* bytes = nullptr)
{
    few_carver c(ws);
    sel_layout L;
    L.owner = c.take<int>(n_modes);
    L.n_entries = c.take<int>(1);
    L.y2 = c.take<double>((size_t)n_src * 2 * n_modes);
    L.bitmap = c.take<unsigned>((size_t)n_src * sel_words(n_modes));
    L.mirror_e = c.take<int>(n_modes);
    L.y2m = c.take<double>((size_t)n_src * n_modes);
    L.fb_list = c.take<int>((size_t)n_src * n_t);
    L.fb_count = c.take<int>(1);
    if (bytes) *bytes = c.off;
    return L;
}

// Inclusive block scan of one int per thread; returns the inclusive prefix, *total = block sum.
template <int kThreads>
__device__ __forceinline__ int block_scan_int(int v, int* warp_sums, int* total)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int o = 1; o < 32; o <<= 1) { int u = __shfl_up_sync(0xffffffffu, v, o); if (lane >= o) v += u; }
    if (lane == 31) warp_sums[wid] = v;
    __syncthreads();
    if (wid == 0) {
        int s = lane < kThreads / 32 ? warp_sums[lane] : 0;
        for (int o = 1; o < 32; o <<= 1) { int u = __shfl_up_sync(0xffffffffu, s, o); if (lane >= o) s += u; }
        if (lane < kThreads / 32) warp_sums[lane] = s;
    }
    __syncthreads();
    int res = v + (wid ? warp_sums[wid - 1] : 0);
    *total = warp_sums[kThreads / 32 - 1];
    __syncthreads();
    return res;
}

// Mirror list (modes with m > 0 in ascending j), |Y|^2 per entry, bitmap cleared.  One block per source.  The mirror index of a
// mode is the number of m > 0 modes before it: warp ballots per 1024-mode chunk, ONE scan of the (chunk, warp) counts, then
// popc of the lanes below -- two block barriers in all, whatever n_modes (the 42 273-mode grid took 42 block scans before).
constexpr int kPrepChunks = FEW_MAX_SELECT_MODES / kPrepThreads;
__global__ void __launch_bounds__(kPrepThreads)
few_select_prepare_kernel(const int* __restrict__ m, const double2* __restrict__ ylm_plus, const double2* __restrict__ ylm_minus,
                          int n_modes, sel_layout L, int* status)
{
    __shared__ int wcnt[kPrepChunks * 32];       // m > 0 modes per (chunk, warp), then their exclusive prefix
    __shared__ int total_s;
    const int src = blockIdx.x, tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const bool with_y = ylm_plus != nullptr;
    const int n_chunks = (n_modes + kPrepThreads - 1) / kPrepThreads;
#pragma unroll 4
    for (int c = 0; c < n_chunks; ++c) {                 // (unrolled: the loads of several chunks in flight)
        const int j = c * kPrepThreads + tid;
        const int mj = j < n_modes ? m[j] : 0;
        if (j < n_modes && mj < 0) atomicOr(status, FEW_DEV_BAD_MODE);
        const unsigned b = __ballot_sync(0xffffffffu, with_y && j < n_modes && mj > 0);
        if (lane == 0) wcnt[c * 32 + wid] = __popc(b);
    }
    __syncthreads();
    if (wid == 0) {                              // warp 0: exclusive scan of the n_chunks * 32 counts, 32 at a time
        int carry = 0;
        for (int base = 0; base < n_chunks * 32; base += 32) {
            const int v = wcnt[base + lane];
            int incl = v;
            for (int o = 1; o < 32; o <<= 1) { const int u = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += u; }
            wcnt[base + lane] = carry + incl - v;
            carry += __shfl_sync(0xffffffffu, incl, 31);
        }
        if (lane == 0) total_s = carry;
    }
    __syncthreads();
    double* y2 = L.y2 + (size_t)src * 2 * n_modes;
#pragma unroll 4
    for (int c = 0; c < n_chunks; ++c) {
        const int j = c * kPrepThreads + tid;
        const int mj = j < n_modes ? m[j] : 0;
        const bool flag = with_y && j < n_modes && mj > 0;
        const unsigned b = __ballot_sync(0xffffffffu, flag);
        if (j < n_modes) {
            const double2 yp = with_y ? ylm_plus[(size_t)src * n_modes + j] : make_double2(1.0, 0.0);
            y2[j] = __dadd_rn(__dmul_rn(yp.x, yp.x), __dmul_rn(yp.y, yp.y));
            double w_m = 0.0;
            int me = -1;
            if (flag) {
                const int e = wcnt[c * 32 + wid] + __popc(b & ((1u << lane) - 1u));
                me = n_modes + e;
                if (src == 0) L.owner[e] = j;
                const double2 ym = ylm_minus[(size_t)src * n_modes + j];
                w_m = __dadd_rn(__dmul_rn(ym.x, ym.x), __dmul_rn(ym.y, ym.y));
                y2[n_modes + e] = w_m;
            }
            if (src == 0) L.mirror_e[j] = me;
            L.y2m[(size_t)src * n_modes + j] = w_m;
        }
    }
    if (src == 0 && tid == 0) { *L.n_entries = n_modes + total_s; *L.fb_count = 0; }
    for (int w = tid; w < sel_words(n_modes); w += kPrepThreads) L.bitmap[(size_t)src * sel_words(n_modes) + w] = 0u;
}

// ---- block reductions over W warps; every thread gets the result.  `slot` alternates between calls so that one
// __syncthreads per reduction suffices.
template <int W> struct sel_red { double d[2][W]; long long i[2][W]; };

template <int W>
__device__ __forceinline__ double block_sum(double v, sel_red<W>& s, int& slot)
{
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) s.d[slot][threadIdx.x >> 5] = v;
    __syncthreads();
    double r = 0.0;
#pragma unroll
    for (int w = 0; w < W; ++w) r += s.d[slot][w];
    slot ^= 1;
    return r;
}
template <int W>
__device__ __forceinline__ long long block_sum_ll(long long v, sel_red<W>& s, int& slot)
{
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) s.i[slot][threadIdx.x >> 5] = v;
    __syncthreads();
    long long r = 0;
#pragma unroll
    for (int w = 0; w < W; ++w) r += s.i[slot][w];
    slot ^= 1;
    return r;
}
template <int W>
__device__ __forceinline__ long long block_max_ll(long long v, sel_red<W>& s, int& slot)
{
    for (int o = 16; o; o >>= 1) { long long u = __shfl_xor_sync(0xffffffffu, v, o); v = u > v ? u : v; }
    if ((threadIdx.x & 31) == 0) s.i[slot][threadIdx.x >> 5] = v;
    __syncthreads();
    long long r = s.i[slot][0];
#pragma unroll
    for (int w = 1; w < W; ++w) r = s.i[slot][w] > r ? s.i[slot][w] : r;
    slot ^= 1;
    return r;
}

// ---- shared state of one row's selection: T threads, BK = capacity of the fine step, NW = words of the owner bitmap
template <int T, int BK, int NW>
struct sel_shared {
    sel_red<T / 32> red;
    unsigned bitmap[NW];
    double bkt_p[BK], srt_p[BK];
    int bkt_e[BK], srt_e[BK];
    int bkt_count;
};

// Entries policy 1: keys (bit patterns of the powers, -1 = empty slot) and entry indices in registers.
template <int EPT>
struct reg_entries {
    const long long (&key)[EPT];
    const int (&ent)[EPT];
    __device__ __forceinline__ reg_entries(const long long (&k)[EPT], const int (&e)[EPT]) : key(k), ent(e) {}
    template <class F> __device__ __forceinline__ void for_each(F f) const
    {
#pragma unroll
        for (int i = 0; i < EPT; ++i) if (key[i] >= 0) f(key[i], ent[i], i & 3);
    }
};

// Entries policy 2: the row is re-read (L2) and the powers recomputed on every pass, with the same separately rounded
// operations as the definition: |A|^2 = re*re + im*im, P = |A|^2 |Y|^2.  Primary of mode j = entry j; its mirror (m > 0) =
// entry mirror_e[j], formed from the same |A_j|^2.  Thread tid owns modes tid, tid + T, ...: a fixed order per thread.
template <int T>
struct stream_entries {
    const double2* a; const double* y2p; const double* y2m; const int* mirror_e; int n_modes;
    template <class F> __device__ __forceinline__ void for_each(F f) const
    {
        for (int j = threadIdx.x; j < n_modes; j += T) {
            const double2 v = a[j];
            const double a2 = __dadd_rn(__dmul_rn(v.x, v.x), __dmul_rn(v.y, v.y));
            f(__double_as_longlong(__dmul_rn(a2, y2p[j])), j, 0);
            const int me = mirror_e[j];
            if (me >= 0) f(__double_as_longlong(__dmul_rn(a2, y2m[j])), me, 1);
        }
    }
};

// The selection proper.  thr = (1 - eps) * (total power of the row) > 0, or <= 0 for the degenerate case (eps >= 1, zero row).
// The entries E enumerates need not be the whole row: any superset of the kept entries whose total is >= thr gives the same
// set, because C_{r-1} of an entry is the summed power of the entries before it in the order and each of those is itself
// kept.  The threshold's exponent bucket is searched in [b_lo, b_hi]: the caller guarantees g(b_lo) >= thr and no key above
// bucket b_hi.  Marks the owners of the kept entries in S.bitmap (caller zeroes it and S.bkt_count, then __syncthreads).
template <int T, int BK, int NW, class Entries>
__device__ __forceinline__ void select_core(const Entries& E, double thr, int b_lo, int b_hi, int n_modes,
                                            const int* __restrict__ owner, sel_shared<T, BK, NW>& S, int& slot)
{
    const int tid = threadIdx.x;
    auto mark = [&](int e) { const int j = e < n_modes ? e : owner[e - n_modes]; atomicOr(&S.bitmap[j >> 5], 1u << (j & 31)); };
    long long kappa;            // kept  <=>  key > kappa  or  (key == kappa and entry index <= iota)
    int iota = 0x7fffffff;
    if (!(thr > 0.0)) {
        // only rank 0 survives, i.e. the largest power with the lowest entry index
        long long kmax_local = -1;
        E.for_each([&](long long k, int, int) { kmax_local = k > kmax_local ? k : kmax_local; });
        kappa = block_max_ll(kmax_local, S.red, slot);
        long long best = -0x7fffffff;       // max of -index
        E.for_each([&](long long k, int e, int) { if (k == kappa) { const long long c = -(long long)e; best = c > best ? c : best; } });
        iota = (int)(-block_max_ll(best, S.red, slot));
    } else {
        // ---- 1. coarse: g(x) = sum of powers with bucket >= x (bucket = key >> kBucketShift) is non-increasing in x;
        // B = the largest x in [b_lo, b_hi] with g(x) >= thr (the fixed reduction tree keeps monotonicity exactly).
        int s_lo = b_lo, s_hi = b_hi;
        while (s_lo < s_hi) {
            const int mid = (s_lo + s_hi + 1) >> 1;
            const int cand_hi = mid << (kBucketShift - 32);   // the bucket lives in the key's high word: one 32-bit compare
            double g4[4] = {0.0, 0.0, 0.0, 0.0};          // several chains: the DADD latency, not its rate, bounds this loop
            E.for_each([&](long long k, int, int c) { if ((int)(k >> 32) >= cand_hi) g4[c] += __longlong_as_double(k); });
            const double g = block_sum((g4[0] + g4[1]) + (g4[2] + g4[3]), S.red, slot);
            if (!(g < thr)) s_lo = mid; else s_hi = mid - 1;
        }
        const long long B = s_lo;
        const long long k_lo = B << kBucketShift;                   // bucket B = keys in [k_lo, k_hi)
        const long long k_hi = B >= (1ll << (63 - kBucketShift)) - 1 ? 0x7fffffffffffffffLL : (B + 1) << kBucketShift;
        double ga = 0.0; long long nb = 0;
        E.for_each([&](long long k, int, int) { ga += k >= k_hi ? __longlong_as_double(k) : 0.0; nb += (k >= k_lo && k < k_hi) ? 1 : 0; });
        const double g_above = block_sum(ga, S.red, slot);           // < thr by construction
        const long long n_bkt = block_sum_ll(nb, S.red, slot);
        if (n_bkt <= BK) {
            // ---- 2. fine: sort + cumulative sum of the bucket's entries, exactly as the definition orders them
            E.for_each([&](long long k, int e, int) {
                if (k >= k_lo && k < k_hi) { const int pos = atomicAdd(&S.bkt_count, 1); S.bkt_p[pos] = __longlong_as_double(k); S.bkt_e[pos] = e; }
            });
            __syncthreads();
            const int M = (int)n_bkt;
            for (int q = tid; q < M; q += T) {
                const double pq = S.bkt_p[q]; const int eq = S.bkt_e[q];
                int rank = 0;
                for (int r = 0; r < M; ++r) { const double pr = S.bkt_p[r]; rank += (pr > pq || (pr == pq && S.bkt_e[r] < eq)) ? 1 : 0; }
                S.srt_p[rank] = pq; S.srt_e[rank] = eq;
            }
            __syncthreads();
            if (tid < 32) {
                // warp 0: C_{r-1} = g_above + (sum of the sorted entries before r), lane l owning positions [kPer l, kPer (l + 1))
                constexpr int kPer = BK / 32;
                double loc = 0.0;
                for (int u = 0; u < kPer; ++u) { const int r = tid * kPer + u; loc += r < M ? S.srt_p[r] : 0.0; }
                double incl = loc;
                for (int o = 1; o < 32; o <<= 1) { const double v = __shfl_up_sync(0xffffffffu, incl, o); if (tid >= o) incl += v; }
                double c = g_above + (incl - loc);
                for (int u = 0; u < kPer; ++u) {
                    const int r = tid * kPer + u;
                    if (r < M) {
                        if (c < thr) mark(S.srt_e[r]);
                        c += S.srt_p[r];
                    }
                }
            }
            kappa = k_hi - 1; iota = -1;                             // below: key > kappa keeps everything above the bucket
        } else {
            // ---- 3. fallback.  G(c) = sum of powers with key > c is monotone non-increasing in c (the fixed reduction tree keeps
            // that exactly); build the largest c with G(c) >= thr bit by bit, then kappa = c + 1.
            long long lo = 0;
            for (int b = 62; b >= 0; --b) {
                const long long cand = lo | (1ll << b);
                double g4[4] = {0.0, 0.0, 0.0, 0.0};
                E.for_each([&](long long k, int, int c) { g4[c] += k > cand ? __longlong_as_double(k) : 0.0; });
                const double g = block_sum((g4[0] + g4[1]) + (g4[2] + g4[3]), S.red, slot);
                if (!(g < thr)) lo = cand;
            }
            kappa = lo + 1;
            // ties at kappa: the j-th (by entry index) is kept iff G(kappa) + j P < thr, accumulated one by one like the cumsum
            double g = 0.0; long long nt = 0;
            E.for_each([&](long long k, int, int) { g += k > kappa ? __longlong_as_double(k) : 0.0; nt += k == kappa ? 1 : 0; });
            g = block_sum(g, S.red, slot);
            const long long n_tie = block_sum_ll(nt, S.red, slot);
            if (n_tie > 1) {
                const double p = __longlong_as_double(kappa);
                long long keep_t = 0; double c = g;
                while (keep_t < n_tie && c < thr) { ++keep_t; c += p; }      // every thread computes the same count
                if (keep_t < n_tie) {
                    // iota = the keep_t-th smallest entry index among the ties: 18-bit select on the index
                    int lo_i = -1;                                           // largest index with count(ties <= index) < keep_t
                    for (int b = 17; b >= 0; --b) {
                        const int cand = lo_i < 0 ? (1 << b) - 1 : lo_i + (1 << b);
                        long long cnt = 0;
                        E.for_each([&](long long k, int e, int) { cnt += (k == kappa && e <= cand) ? 1 : 0; });
                        cnt = block_sum_ll(cnt, S.red, slot);
                        if (cnt < keep_t) lo_i = cand;
                    }
                    iota = lo_i + 1;
                }
            }
        }
    }
    E.for_each([&](long long k, int e, int) { if (k > kappa || (k == kappa && e <= iota)) mark(e); });
}

// General kernel, one (source, step) row per block pass, rows of any length: every pass of select_core streams the row's
// amplitudes (HBM once, then L2) and recomputes the powers.  Serves the Kerr-shaped grid (42 273 modes, 78 507 entries per
// row: ~10 passes of 676 KB) and the rows the fast kernel leaves in fb_list (flat spectra, degenerate thresholds); with
// fb_list == NULL the grid is (n_t, n_src) and every row is done here.
constexpr int kStreamThreads = 1024;
constexpr int kStreamBucket = 1024;
constexpr int kStreamWords = FEW_MAX_SELECT_MODES / 32;
constexpr int kStreamCand = 14336;     // candidates (power >= tau) of a long row that the kernel keeps in shared memory (168 KB)
struct stream_shared : sel_shared<kStreamThreads, kStreamBucket, kStreamWords> {
    long long cand_k[kStreamCand];
    int cand_e[kStreamCand];
    int warp_sums[32];
};

// Entries policy 3: the candidates of a long row, compacted into shared memory (keys and entry indices).
template <int T>
struct smem_entries {
    const long long* k; const int* e; int n;
    template <class F> __device__ __forceinline__ void for_each(F f) const
    {
        for (int q = threadIdx.x; q < n; q += T) f(k[q], e[q], (q / T) & 3);
    }
};

__global__ void __launch_bounds__(kStreamThreads)
few_select_row_stream_kernel(const double2* __restrict__ amp, const int* __restrict__ n_t_src, int n_t, int n_modes, double eps, sel_layout L,
                             const int* __restrict__ fb_list, const int* __restrict__ fb_count, int* status)
{
    // ragged batch: the steps past the source's last knot are padding (block-uniform; listed rows were checked by the fast kernel)
    if (!fb_list && (int)blockIdx.x >= few_knots(n_t_src, blockIdx.y, n_t, status)) return;
    extern __shared__ __align__(16) unsigned char stream_smem[];
    stream_shared& S = *reinterpret_cast<stream_shared*>(stream_smem);
    const int tid = threadIdx.x;
    const int n_rows = fb_list ? *fb_count : 1;
    const int n_ent = *L.n_entries;
    const int words = sel_words(n_modes);
    for (int q = fb_list ? blockIdx.x : 0; q < n_rows; q += gridDim.x) {
        const int row = fb_list ? fb_list[q] : blockIdx.y * n_t + blockIdx.x;
        const int src = row / n_t, k = row - src * n_t;
        const double2* a = amp + ((size_t)src * n_t + k) * n_modes;
        const double* y2p = L.y2 + (size_t)src * 2 * n_modes;
        const double* y2m = L.y2m + (size_t)src * n_modes;
        stream_entries<kStreamThreads> E{a, y2p, y2m, L.mirror_e, n_modes};
        __syncthreads();                                 // the previous row's shared state is no longer read
        for (int w = tid; w < words; w += kStreamThreads) S.bitmap[w] = 0u;
        if (tid == 0) S.bkt_count = 0;
        int slot = 0;
        double t2[2] = {0.0, 0.0};
        E.for_each([&](long long key, int, int c) { t2[c] += __longlong_as_double(key); });
        const double total = block_sum((t2[0] + t2[1]) + (0.0 + 0.0), S.red, slot);      // the same tree as the core's g(0)
        const double thr = (1.0 - eps) * total;
        // buckets below that of tau = eps total / (4 n) hold less than eps total / 4 altogether: the search starts there
        const long long tau_key = __double_as_longlong(0.25 * eps * total / (double)n_ent);
        const int b_lo = (eps > 1e-10 && tau_key > 0) ? (int)(tau_key >> kBucketShift) : 0;
        const int b_hi = (int)(__double_as_longlong(total) >> kBucketShift);
        // Second (and normally last) pass over the row: the entries below tau are certainly dropped (the fast kernel's argument),
        // the others -- a few thousand of a Kerr-shaped row's 78 507 -- are compacted, in a fixed order, into shared memory and
        // selected there; before, every step of the search streamed the whole row from L2 again (~13 passes).
        bool done = false;
        if (thr > 0.0 && tau_key > 0 && eps > 1e-10) {
            int n_cand = 0;
            for (int base = 0; base < n_modes; base += kStreamThreads) {
                const int j = base + tid;
                long long kp = -1, km = -1;
                int me = -1;
                if (j < n_modes) {
                    const double2 v = a[j];
                    const double a2 = __dadd_rn(__dmul_rn(v.x, v.x), __dmul_rn(v.y, v.y));
                    kp = __double_as_longlong(__dmul_rn(a2, y2p[j]));
                    me = L.mirror_e[j];
                    if (me >= 0) km = __double_as_longlong(__dmul_rn(a2, y2m[j]));
                }
                const int cnt = (kp >= tau_key ? 1 : 0) + (km >= tau_key ? 1 : 0);
                int tot;
                const int incl = block_scan_int<kStreamThreads>(cnt, S.warp_sums, &tot);
                int pos = n_cand + incl - cnt;
                if (kp >= tau_key) { if (pos < kStreamCand) { S.cand_k[pos] = kp; S.cand_e[pos] = j; } ++pos; }
                if (km >= tau_key) { if (pos < kStreamCand) { S.cand_k[pos] = km; S.cand_e[pos] = me; } }
                n_cand += tot;                           // block-uniform
            }
            __syncthreads();
            if (n_cand <= kStreamCand) {
                smem_entries<kStreamThreads> C{S.cand_k, S.cand_e, n_cand};
                double tc = 0.0;
                C.for_each([&](long long key, int, int) { tc += __longlong_as_double(key); });
                const double total_cand = block_sum(tc, S.red, slot);
                if (total_cand < thr) {                  // every candidate has C_{r-1} < thr: all kept
                    C.for_each([&](long long, int e, int) { const int j = e < n_modes ? e : L.owner[e - n_modes]; atomicOr(&S.bitmap[j >> 5], 1u << (j & 31)); });
                } else {
                    select_core(C, thr, b_lo, b_hi, n_modes, L.owner, S, slot);
                }
                done = true;
            }
        }
        if (!done) select_core(E, thr, b_lo, b_hi, n_modes, L.owner, S, slot);
        __syncthreads();
        unsigned* gb = L.bitmap + (size_t)src * words;
        for (int w = tid; w < words; w += kStreamThreads)
            if (S.bitmap[w]) atomicOr(&gb[w], S.bitmap[w]);
    }
}

// Fast kernel, one (source, step) row per block.  An entry whose power is below tau = eps * total / (4 n_entries) is
// certainly dropped: all such entries together hold less than eps * total / 4, so for each of them C_{r-1} > (1 - eps/4) total,
// a margin far outside rounding.  Only the candidates (power >= tau: the kept entries and a margin, a few hundred of the
// 7137) are compacted -- in a fixed order, so that every run adds the same numbers in the same order -- and go through
// select_core at 8 entries per thread instead of 32.  The mirror entry of mode j is formed beside the primary from the same
// |A_j|^2 (mirror_e[j] = its entry index, y2m[j] = |Y_{l,-m}|^2): no gather, no shared-memory copy of the row.
// A row with more than kCandMax candidates (a flat spectrum) or a degenerate threshold is appended to fb_list for the
// general kernel.
constexpr int kCandMax = 2048;
constexpr int kCandEpt = kCandMax / kSelThreads;
constexpr int kFastModes = 16 * kSelThreads;          // rows of up to 4096 modes: 16 primaries + 16 mirrors per thread
constexpr int kFastWords = kFastModes / 32;

template <int NPT>
__global__ void __launch_bounds__(kSelThreads, 3)
few_select_row_fast_kernel(const double2* __restrict__ amp, const int* __restrict__ n_t_src, int n_t, int n_modes, double eps, sel_layout L,
                           int* status)
{
    if ((int)blockIdx.x >= few_knots(n_t_src, blockIdx.y, n_t, status)) return;     // ragged batch: padding step (block-uniform)
    __shared__ sel_shared<kSelThreads, kBucketMax, kFastWords> S;
    __shared__ long long cand_k[kCandMax];
    __shared__ int cand_e[kCandMax];
    __shared__ int warp_sums[kSelWarps];
    const int tid = threadIdx.x;
    const int src = blockIdx.y, k = blockIdx.x;
    const int n_ent = *L.n_entries;
    const double2* a = amp + ((size_t)src * n_t + k) * n_modes;
    const double* y2p = L.y2 + (size_t)src * 2 * n_modes;
    const double* y2m = L.y2m + (size_t)src * n_modes;
    const int words = sel_words(n_modes);
    for (int w = tid; w < words; w += kSelThreads) S.bitmap[w] = 0u;
    if (tid == 0) S.bkt_count = 0;
    int slot = 0;

    long long kp[NPT], km[NPT];
    double t4[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
    for (int i = 0; i < NPT; ++i) {
        kp[i] = km[i] = -1;
        const int j = i * kSelThreads + tid;
        if (j < n_modes) {
            // branch-free, so that all of a thread's loads are in flight together (y2m is 0 where there is no mirror)
            const double2 v = a[j];
            const double wp = y2p[j], wm = y2m[j];
            const bool has_mirror = L.mirror_e[j] >= 0;
            const double a2 = __dadd_rn(__dmul_rn(v.x, v.x), __dmul_rn(v.y, v.y));
            const double p = __dmul_rn(a2, wp), pm = __dmul_rn(a2, wm);
            kp[i] = __double_as_longlong(p);
            km[i] = has_mirror ? __double_as_longlong(pm) : -1;
            t4[i & 1] += p;
            t4[2 + (i & 1)] += has_mirror ? pm : 0.0;
        }
    }
    const double total = block_sum((t4[0] + t4[1]) + (t4[2] + t4[3]), S.red, slot);
    const double thr = (1.0 - eps) * total;
    const long long tau_key = __double_as_longlong(0.25 * eps * total / (double)n_ent);
    int cnt = 0;
#pragma unroll
    for (int i = 0; i < NPT; ++i) cnt += (kp[i] >= tau_key ? 1 : 0) + (km[i] >= tau_key ? 1 : 0);
    int n_cand;
    const int incl = block_scan_int<kSelThreads>(cnt, warp_sums, &n_cand);
    if (!(thr > 0.0) || !(tau_key > 0) || !(eps > 1e-10) || n_cand > kCandMax) {   // block-uniform: hand the row to the general kernel
        if (tid == 0) L.fb_list[atomicAdd(L.fb_count, 1)] = src * n_t + k;
        return;
    }
    int pos = incl - cnt;
#pragma unroll
    for (int i = 0; i < NPT; ++i) {
        if (kp[i] >= tau_key) { cand_k[pos] = kp[i]; cand_e[pos] = i * kSelThreads + tid; ++pos; }
        if (km[i] >= tau_key) { cand_k[pos] = km[i]; cand_e[pos] = L.mirror_e[i * kSelThreads + tid]; ++pos; }
    }
    __syncthreads();
    long long ck[kCandEpt];
    int ce[kCandEpt];
    double tc = 0.0;
#pragma unroll
    for (int i = 0; i < kCandEpt; ++i) {
        const int q = i * kSelThreads + tid;
        ck[i] = q < n_cand ? cand_k[q] : -1;
        ce[i] = q < n_cand ? cand_e[q] : 0x7fffffff;
        tc += q < n_cand ? __longlong_as_double(ck[i]) : 0.0;
    }
    const double total_cand = block_sum(tc, S.red, slot);
    if (total_cand < thr) {
        // every candidate has C_{r-1} < thr: all kept
#pragma unroll
        for (int i = 0; i < kCandEpt; ++i)
            if (ck[i] >= 0) { const int e = ce[i]; const int j = e < n_modes ? e : L.owner[e - n_modes]; atomicOr(&S.bitmap[j >> 5], 1u << (j & 31)); }
    } else {
        // candidates lie in the exponent buckets of [tau, total]: ~log2(4 n_entries / eps) of them, 5-6 search steps instead of 11
        select_core(reg_entries<kCandEpt>(ck, ce), thr, (int)(tau_key >> kBucketShift), (int)(__double_as_longlong(total) >> kBucketShift), n_modes,
                    L.owner, S,
                    slot);
    }
    __syncthreads();
    unsigned* gb = L.bitmap + (size_t)src * words;
    for (int w = tid; w < words; w += kSelThreads)
        if (S.bitmap[w]) atomicOr(&gb[w], S.bitmap[w]);
}

// bitmap -> ascending keep_idx (padded with -1) and n_keep.  One block per source.  keep_all: identity list.  A thread takes
// whole bitmap words (popc), one block scan per 1024 words (32 768 modes), then writes its word's set bits in order.
__global__ void __launch_bounds__(kPrepThreads)
few_select_compact_kernel(sel_layout L, int n_modes, int keep_all, int* __restrict__ keep_idx, int* __restrict__ n_keep)
{
    __shared__ int warp_sums[32];
    const int src = blockIdx.x, tid = threadIdx.x;
    int* out = keep_idx + (size_t)src * n_modes;
    if (keep_all) {
        for (int j = tid; j < n_modes; j += kPrepThreads) out[j] = j;
        if (tid == 0) n_keep[src] = n_modes;
        return;
    }
    const int words = sel_words(n_modes);
    const unsigned* gb = L.bitmap + (size_t)src * words;
    int carry = 0;                               // block-uniform
    for (int base = 0; base < words; base += kPrepThreads) {
        const int w = base + tid;
        unsigned bits = w < words ? gb[w] : 0u;
        if (w == words - 1 && (n_modes & 31)) bits &= (1u << (n_modes & 31)) - 1u;
        int total;
        const int cnt = __popc(bits);
        int pos = carry + block_scan_int<kPrepThreads>(cnt, warp_sums, &total) - cnt;
        while (bits) { const int b = __ffs(bits) - 1; bits &= bits - 1; out[pos++] = w * 32 + b; }
        carry += total;
    }
    for (int j = carry + tid; j < n_modes; j += kPrepThreads) out[j] = -1;
    if (tid == 0) n_keep[src] = carry;
}

}  // namespace

extern "C" size_t few_select_modes_workspace(int n_src, int n_t, int n_modes)
{
    if (n_src <= 0 || n_t <= 0 || n_modes <= 0) return 0;
    size_t bytes = 0;
    sel_carve(nullptr, n_src, n_t, n_modes, &bytes);
    return bytes;
}

extern "C" int few_select_modes_ragged(few_ctx* ctx, const double* amp, const int* m, const double* ylm_plus, const double* ylm_minus,
                                       const int* n_t_src, double eps, int n_src, int n_t, int n_modes, int* keep_idx, int* n_keep,
                                       void* workspace, size_t workspace_bytes, void* stream)
{
    FEW_REQUIRE(ctx && amp && m && keep_idx && n_keep, FEW_ERR_INVALID_ARG, "NULL argument");
    FEW_REQUIRE(n_src > 0 && n_t > 0 && n_modes > 0, FEW_ERR_INVALID_ARG, "sizes must be positive");
    FEW_REQUIRE(ylm_plus == nullptr || ylm_minus != nullptr, FEW_ERR_INVALID_ARG, "ylm_minus is NULL but ylm_plus is not");
    FEW_REQUIRE(n_src <= 65535, FEW_ERR_LIMIT, "n_src > 65535");
    cudaStream_t st = (cudaStream_t)stream;
    sel_layout L{};
    if (!(eps > 0.0)) {       // R6: eps <= 0 keeps every mode, nothing is sorted
        few_select_compact_kernel<<<n_src, kPrepThreads, 0, st>>>(L, n_modes, 1, keep_idx, n_keep);
        FEW_LAUNCHED(ctx);
        return FEW_OK;
    }
    FEW_REQUIRE(n_modes <= FEW_MAX_SELECT_MODES, FEW_ERR_LIMIT, "n_modes > FEW_MAX_SELECT_MODES");
    FEW_REQUIRE(workspace && ((uintptr_t)workspace % 256) == 0 &&
                    workspace_bytes >= few_select_modes_workspace(n_src, n_t, n_modes),
                FEW_ERR_WORKSPACE, "workspace NULL, misaligned or too small");
    L = sel_carve(workspace, n_src, n_t, n_modes);
    few_select_prepare_kernel<<<n_src, kPrepThreads, 0, st>>>(m, (const double2*)ylm_plus, (const double2*)ylm_minus, n_modes, L,
                                                           ctx->d_status);
    FEW_LAUNCHED(ctx);
    const dim3 grid(n_t, n_src);
    FEW_REQUIRE(sizeof(stream_shared) <= (size_t)ctx->smem_optin, FEW_ERR_LIMIT, "stream kernel's shared memory exceeds the device limit");
    FEW_CUDA_CHECK(cudaFuncSetAttribute(few_select_row_stream_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(stream_shared)));
    if (n_modes <= kFastModes) {
        few_select_row_fast_kernel<16><<<grid, kSelThreads, 0, st>>>((const double2*)amp, n_t_src, n_t, n_modes, eps, L, ctx->d_status);
        FEW_LAUNCHED(ctx);
        // the rows the fast kernel left (usually none): a small persistent grid walks the list
        const long long n_rows = (long long)n_t * n_src;
        const unsigned fb_grid = (unsigned)(n_rows < ctx->sm_count ? n_rows : ctx->sm_count);
        few_select_row_stream_kernel<<<fb_grid, kStreamThreads, sizeof(stream_shared), st>>>((const double2*)amp, n_t_src, n_t, n_modes, eps, L,
                                                                                             L.fb_list, L.fb_count, ctx->d_status);
    } else {
        few_select_row_stream_kernel<<<grid, kStreamThreads, sizeof(stream_shared), st>>>((const double2*)amp, n_t_src, n_t, n_modes, eps, L, nullptr,
                                                                                          nullptr, ctx->d_status);
    }
    FEW_LAUNCHED(ctx);
    few_select_compact_kernel<<<n_src, kPrepThreads, 0, st>>>(L, n_modes, 0, keep_idx, n_keep);
    FEW_LAUNCHED(ctx);
    return FEW_OK;
}

extern "C" int few_select_modes(few_ctx* ctx, const double* amp, const int* m, const double* ylm_plus, const double* ylm_minus,
                                double eps, int n_src, int n_t, int n_modes, int* keep_idx, int* n_keep,
                                void* workspace, size_t workspace_bytes, void* stream)
{
    return few_select_modes_ragged(ctx, amp, m, ylm_plus, ylm_minus, nullptr, eps, n_src, n_t, n_modes, keep_idx, n_keep, workspace,
                                   workspace_bytes, stream);
}
