// few_select.cu -- S2: the Mode Selector (sec. III D): "taking arrays of the power within each mode at each
// sparse time step ... operates entirely within each time step.  It sorts the individual modes in descending order and
// computes a cumulative summation ... where the additional power contributed by an individual mode falls below a user
// provided threshold related to the total power emitted (eps) at that time step (the final entry in the cumulative sum)
// ... the union of all contributing modes across all time steps".
//
// One block per (source, sparse step).  The row of entry powers (every (l,m,n) plus the (l,-m,-n) mirror of each m>0
// mode, R4) is built in shared memory, sorted there by a stable LSD radix sort on the order-preserving bit
// pattern of the FP64 power (descending; ties keep ascending entry index, R7), scanned in FP64, thresholded
// (rank r kept iff r == 0 or C_{r-1} < (1-eps) C_last, R5), and the owners of the kept entries are OR-ed into a per-source
// bitmap.  A second kernel compacts the bitmap into ascending keep_idx and n_keep.  Nothing leaves the SM between the
// load of the amplitudes and the bitmap update; no library sort.
#include "few_common.cuh"

namespace {

constexpr int kSelThreads = 1024;
constexpr int kSelWarps = kSelThreads / 32;
constexpr int kRadixBits = 8;
constexpr int kRadix = 1 << kRadixBits;

struct sel_layout {
    int* owner;       // [n_modes]   owner mode of mirror entry e - n_modes   (shared by sources)
    int* n_entries;   // [1]
    double* y2;       // [n_src][2 n_modes]  |Y|^2 per entry
    unsigned* bitmap; // [n_src][words]
};

__host__ __device__ inline int sel_words(int n_modes) { return (n_modes + 31) / 32; }

sel_layout sel_carve(void* ws, int n_src, int n_modes, size_t* bytes = nullptr)
{
    few_carver c(ws);
    sel_layout L;
    L.owner = c.take<int>(n_modes);
    L.n_entries = c.take<int>(1);
    L.y2 = c.take<double>((size_t)n_src * 2 * n_modes);
    L.bitmap = c.take<unsigned>((size_t)n_src * sel_words(n_modes));
    if (bytes) *bytes = c.off;
    return L;
}

// Inclusive block scan of one int per thread (kSelThreads threads); returns the inclusive prefix, *total = block sum.
__device__ __forceinline__ int block_scan_int(int v, int* warp_sums, int* total)
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
    *total = warp_sums[kSelWarps - 1];
    __syncthreads();
    return res;
}

// Mirror list (modes with m > 0 in ascending j), |Y|^2 per entry, bitmap cleared.  One block per source.
__global__ void few_select_prepare_kernel(const int* __restrict__ m, const double2* __restrict__ ylm_plus,
                                          const double2* __restrict__ ylm_minus, int n_modes, sel_layout L, int* status)
{
    __shared__ int warp_sums[32];
    __shared__ int carry_s;
    const int src = blockIdx.x, tid = threadIdx.x;
    if (tid == 0) carry_s = 0;
    __syncthreads();
    const bool with_y = ylm_plus != nullptr;
    double* y2 = L.y2 + (size_t)src * 2 * n_modes;
    for (int base = 0; base < n_modes; base += kSelThreads) {
        int j = base + tid;
        int mj = j < n_modes ? m[j] : 0;
        if (j < n_modes && mj < 0) atomicOr(status, FEW_DEV_BAD_MODE);
        int flag = (with_y && j < n_modes && mj > 0) ? 1 : 0, total;
        int incl = block_scan_int(flag, warp_sums, &total);
        int carry = carry_s;
        if (j < n_modes) {
            double2 yp = with_y ? ylm_plus[(size_t)src * n_modes + j] : make_double2(1.0, 0.0);
            y2[j] = __dadd_rn(__dmul_rn(yp.x, yp.x), __dmul_rn(yp.y, yp.y));
            if (flag) {
                int e = carry + incl - 1;
                if (src == 0) L.owner[e] = j;
                double2 ym = ylm_minus[(size_t)src * n_modes + j];
                y2[n_modes + e] = __dadd_rn(__dmul_rn(ym.x, ym.x), __dmul_rn(ym.y, ym.y));
            }
        }
        __syncthreads();
        if (tid == 0) carry_s = carry + total;
        __syncthreads();
    }
    if (src == 0 && tid == 0) *L.n_entries = n_modes + carry_s;
    for (int w = tid; w < sel_words(n_modes); w += kSelThreads) L.bitmap[(size_t)src * sel_words(n_modes) + w] = 0u;
}

__device__ __forceinline__ unsigned digit_of(unsigned long long key, int shift) { return (unsigned)(key >> shift) & (kRadix - 1); }

// One (source, step) row.  Shared memory: keys[2][cap] u64, idx[2][cap] u16, hist[kSelWarps][kRadix] u32 (+ small).
__global__ void __launch_bounds__(kSelThreads, 1)
few_select_row_kernel(const double2* __restrict__ amp, int n_t, int n_modes, double eps, int cap, sel_layout L)
{
    extern __shared__ unsigned long long smem_u64[];
    unsigned long long* keys0 = smem_u64;
    unsigned long long* keys1 = keys0 + cap;
    unsigned* hist = reinterpret_cast<unsigned*>(keys1 + cap);          // [kSelWarps][kRadix]
    unsigned short* idx0 = reinterpret_cast<unsigned short*>(hist + kSelWarps * kRadix);
    unsigned short* idx1 = idx0 + cap;
    __shared__ double warp_d[32];
    __shared__ int warp_i[32];
    __shared__ unsigned bitmap_s[(FEW_MAX_SELECT_ENTRIES + 31) / 32];
    __shared__ int skip_s;

    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int src = blockIdx.y, k = blockIdx.x;
    const int n_ent = *L.n_entries;
    const double2* a = amp + ((size_t)src * n_t + k) * n_modes;
    const double* y2 = L.y2 + (size_t)src * 2 * n_modes;
    const int words = sel_words(n_modes);
    for (int w = tid; w < words; w += kSelThreads) bitmap_s[w] = 0u;

    // ---- entry powers -> descending-order keys.  P >= 0, so its bit pattern is monotone; ~bits sorts descending.
    for (int e = tid; e < n_ent; e += kSelThreads) {
        int j = e < n_modes ? e : L.owner[e - n_modes];
        double2 v = a[j];
        double a2 = __dadd_rn(__dmul_rn(v.x, v.x), __dmul_rn(v.y, v.y));
        double p = __dmul_rn(a2, y2[e]);
        keys0[e] = ~(unsigned long long)__double_as_longlong(p);
        idx0[e] = (unsigned short)e;
    }
    __syncthreads();

    // ---- stable LSD radix sort, 8 bits per pass; warp w owns the contiguous items [w*ipw, (w+1)*ipw)
    const int ipw = ((n_ent + kSelWarps - 1) / kSelWarps + 31) / 32 * 32;
    unsigned long long* kin = keys0; unsigned long long* kout = keys1;
    unsigned short* iin = idx0; unsigned short* iout = idx1;
    for (int shift = 0; shift < 64; shift += kRadixBits) {
        for (int b = tid; b < kSelWarps * kRadix; b += kSelThreads) hist[b] = 0u;
        if (tid == 0) skip_s = 0;
        __syncthreads();
        unsigned* myh = hist + wid * kRadix;
        for (int r = 0; r < ipw; r += 32) {
            int item = wid * ipw + r + lane;
            bool valid = item < n_ent;
            unsigned dgt = valid ? digit_of(kin[item], shift) : kRadix + lane;   // invalid lanes never match a digit
            unsigned peers = __match_any_sync(0xffffffffu, dgt);
            if (valid && lane == __ffs(peers) - 1) myh[dgt] += __popc(peers);
            __syncwarp();
        }
        __syncthreads();
        // exclusive scan over (digit major, warp minor): thread handles 8 consecutive (digit, warp) cells
        {
            const int cells = kSelWarps * kRadix / kSelThreads;   // 8
            int dgt = tid / (kSelWarps / cells), w0 = (tid % (kSelWarps / cells)) * cells;
            unsigned loc[cells]; int sum = 0;
#pragma unroll
            for (int c = 0; c < cells; ++c) { loc[c] = hist[(w0 + c) * kRadix + dgt]; sum += (int)loc[c]; }
            int total, incl = block_scan_int(sum, warp_i, &total);
            int run = incl - sum;
#pragma unroll
            for (int c = 0; c < cells; ++c) { hist[(w0 + c) * kRadix + dgt] = (unsigned)run; run += (int)loc[c]; }
            // a digit that holds every item: this pass is the identity permutation
            int dsum = sum;
            for (int o = 1; o < kSelWarps / cells; ++o) dsum += __shfl_down_sync(0xffffffffu, sum, o);
            if ((tid % (kSelWarps / cells)) == 0 && dsum == n_ent) skip_s = 1;
        }
        __syncthreads();
        if (skip_s) { __syncthreads(); continue; }
        for (int r = 0; r < ipw; r += 32) {
            int item = wid * ipw + r + lane;
            bool valid = item < n_ent;
            unsigned long long key = valid ? kin[item] : 0ull;
            unsigned dgt = valid ? digit_of(key, shift) : kRadix + lane;
            unsigned peers = __match_any_sync(0xffffffffu, dgt);
            unsigned below = peers & ((1u << lane) - 1u);
            if (valid) {
                unsigned dst = myh[dgt] + __popc(below);
                kout[dst] = key; iout[dst] = iin[item];
            }
            __syncwarp();
            if (valid && lane == __ffs(peers) - 1) myh[dgt] += __popc(peers);
            __syncwarp();
        }
        __syncthreads();
        { unsigned long long* tk = kin; kin = kout; kout = tk; unsigned short* ti = iin; iin = iout; iout = ti; }
    }

    // ---- inclusive FP64 cumulative sum in sorted order: blocked items per thread, then a block scan of the partials
    const int ipt = (n_ent + kSelThreads - 1) / kSelThreads;
    const int i0 = tid * ipt, i1 = min(i0 + ipt, n_ent);
    double part = 0.0;
    for (int i = i0; i < i1; ++i) part += __longlong_as_double((long long)~kin[i]);
    double v = part;
    for (int o = 1; o < 32; o <<= 1) { double u = __shfl_up_sync(0xffffffffu, v, o); if (lane >= o) v += u; }
    if (lane == 31) warp_d[wid] = v;
    __syncthreads();
    if (wid == 0) {
        double s = warp_d[lane];
        for (int o = 1; o < 32; o <<= 1) { double u = __shfl_up_sync(0xffffffffu, s, o); if (lane >= o) s += u; }
        warp_d[lane] = s;
    }
    __syncthreads();
    const double total = warp_d[kSelWarps - 1];
    const double thr = (1.0 - eps) * total;
    double c_prev = (v - part) + (wid ? warp_d[wid - 1] : 0.0);          // C_{i0 - 1}
    for (int i = i0; i < i1; ++i) {
        if (i == 0 || c_prev < thr) {
            int e = iin[i];
            int j = e < n_modes ? e : L.owner[e - n_modes];
            atomicOr(&bitmap_s[j >> 5], 1u << (j & 31));
        }
        c_prev += __longlong_as_double((long long)~kin[i]);
    }
    __syncthreads();
    unsigned* gb = L.bitmap + (size_t)src * words;
    for (int w = tid; w < words; w += kSelThreads)
        if (bitmap_s[w]) atomicOr(&gb[w], bitmap_s[w]);
}

// bitmap -> ascending keep_idx (padded with -1) and n_keep.  One block per source.  keep_all: identity list.
__global__ void few_select_compact_kernel(sel_layout L, int n_modes, int keep_all, int* __restrict__ keep_idx,
                                          int* __restrict__ n_keep)
{
    __shared__ int warp_sums[32];
    __shared__ int carry_s;
    const int src = blockIdx.x, tid = threadIdx.x;
    int* out = keep_idx + (size_t)src * n_modes;
    if (keep_all) {
        for (int j = tid; j < n_modes; j += kSelThreads) out[j] = j;
        if (tid == 0) n_keep[src] = n_modes;
        return;
    }
    const unsigned* gb = L.bitmap + (size_t)src * sel_words(n_modes);
    if (tid == 0) carry_s = 0;
    __syncthreads();
    for (int base = 0; base < n_modes; base += kSelThreads) {
        int j = base + tid;
        int flag = (j < n_modes && ((gb[j >> 5] >> (j & 31)) & 1u)) ? 1 : 0, total;
        int incl = block_scan_int(flag, warp_sums, &total);
        int carry = carry_s;
        if (flag) out[carry + incl - 1] = j;
        __syncthreads();
        if (tid == 0) carry_s = carry + total;
        __syncthreads();
    }
    const int cnt = carry_s;
    for (int j = cnt + tid; j < n_modes; j += kSelThreads) out[j] = -1;
    if (tid == 0) n_keep[src] = cnt;
}

size_t sel_row_smem(int cap) { return (size_t)cap * (2 * 8 + 2 * 2) + (size_t)kSelWarps * kRadix * 4; }

}  // namespace

extern "C" size_t few_select_modes_workspace(int n_src, int n_t, int n_modes)
{
    (void)n_t;
    if (n_src <= 0 || n_modes <= 0) return 0;
    size_t bytes = 0;
    sel_carve(nullptr, n_src, n_modes, &bytes);
    return bytes;
}

extern "C" int few_select_modes(few_ctx* ctx, const double* amp, const int* m, const double* ylm_plus, const double* ylm_minus,
                                double eps, int n_src, int n_t, int n_modes, int* keep_idx, int* n_keep,
                                void* workspace, size_t workspace_bytes, void* stream)
{
    FEW_REQUIRE(ctx && amp && m && keep_idx && n_keep, FEW_ERR_INVALID_ARG, "NULL argument");
    FEW_REQUIRE(n_src > 0 && n_t > 0 && n_modes > 0, FEW_ERR_INVALID_ARG, "sizes must be positive");
    FEW_REQUIRE(ylm_plus == nullptr || ylm_minus != nullptr, FEW_ERR_INVALID_ARG, "ylm_minus is NULL but ylm_plus is not");
    FEW_REQUIRE(n_src <= 65535, FEW_ERR_LIMIT, "n_src > 65535");
    cudaStream_t st = (cudaStream_t)stream;
    sel_layout L{};
    if (!(eps > 0.0)) {       // R6: eps <= 0 keeps every mode, nothing is sorted
        few_select_compact_kernel<<<n_src, kSelThreads, 0, st>>>(L, n_modes, 1, keep_idx, n_keep);
        FEW_CUDA_CHECK(cudaGetLastError());
        return FEW_OK;
    }
    FEW_REQUIRE(2 * (long long)n_modes <= FEW_MAX_SELECT_ENTRIES, FEW_ERR_LIMIT, "2*n_modes > FEW_MAX_SELECT_ENTRIES");
    FEW_REQUIRE(workspace && ((uintptr_t)workspace % 256) == 0 &&
                    workspace_bytes >= few_select_modes_workspace(n_src, n_t, n_modes),
                FEW_ERR_WORKSPACE, "workspace NULL, misaligned or too small");
    L = sel_carve(workspace, n_src, n_modes);
    few_select_prepare_kernel<<<n_src, kSelThreads, 0, st>>>(m, (const double2*)ylm_plus, (const double2*)ylm_minus, n_modes, L,
                                                          ctx->d_status);
    FEW_CUDA_CHECK(cudaGetLastError());
    const int cap = 2 * n_modes;
    size_t smem = sel_row_smem(cap);
    FEW_REQUIRE(smem <= (size_t)ctx->smem_optin, FEW_ERR_LIMIT, "row does not fit shared memory");
    FEW_CUDA_CHECK(cudaFuncSetAttribute(few_select_row_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    few_select_row_kernel<<<dim3(n_t, n_src), kSelThreads, smem, st>>>((const double2*)amp, n_t, n_modes, eps, cap, L);
    FEW_CUDA_CHECK(cudaGetLastError());
    few_select_compact_kernel<<<n_src, kSelThreads, 0, st>>>(L, n_modes, 0, keep_idx, n_keep);
    FEW_CUDA_CHECK(cudaGetLastError());
    return FEW_OK;
}
