// few_direct.cu -- direct (non-interpolated) summation, SURVEY.md section 8(f) NEXT-3.
// PAPER.md:151 (sec. III C): "The more basic option provided performs a direct summation with amplitude and trajectory
// information at the array density provided ... usually employed when densely stepping trajectories and amplitude
// calculations"; the slow comparison model "combin[es] the phase and amplitude information at each time point
// in the data stream without interpolating any of these quantities".
//   h_i = scale * factor * sum_j [ Y+_j W_ij + (m_j > 0) (-1)^{l_j} Y-_j conj(W_ij) ],  W_ij = A_ij exp(-i (m_j Phi_phi,i + n_j Phi_r,i))
// (Eq. (10) with the Eq. (9) fold).  amp[n_src][N][K][2] is the amplitude module's [n_t, n_modes] complex layout
// at dense n_t = N, phase[n_src][N][2] = (Phi_phi, Phi_r).
//
// Bound: HBM.  Every amplitude is read exactly once, 16 B per sample*mode evaluation, against ~12 FP64 instructions.
// Design: one thread per sample, a block owns kDirTile consecutive samples and walks the K modes in chunks of kDirChunk.  A
// chunk of the tile is kDirTile rows of 256 contiguous bytes in HBM; the block copies them with 16-byte cp.async (LDGSTS: a
// half-warp per row, so every request is a full 256-byte segment) into a shared-memory stage whose rows are padded by 16 B,
// so that thread i reading "its" row with 128-bit loads is bank-conflict free: the transposition from the mode-fastest HBM
// layout to the sample-per-thread register layout costs no instruction.  A ring of kDirStages stages (cp.async commit groups)
// keeps 2 stages = 70 KB per block in flight.  Mode constants travel with the chunk (48 more 16-byte pieces).
// (First version: one 1-D TMA bulk copy per 256-byte row.  ncu: 1.6 TB/s, warps parked at the barrier -- the TMA unit retires
// about one bulk request per 40 cycles per SM, so 256-byte requests cap at ~1.9 TB/s chip-wide; profiles/r01c_kernels.md, section few_direct_kernel.)
// exp(-i(m Phi_phi + n Phi_r)) = Z_phi^m Z_r^n with Z = exp(-i Phi) from ONE full-range sincos per phase and sample; along a
// mode list in the grid's natural order (n fastest) E advances by one complex multiplication per mode; jumps in (m, n) restart
// from Z_phi^m and a binary power of Z_r (block-uniform branch, once per (l, m) run of the full grid).
#include "few_common.cuh"

namespace {

constexpr int kDirTile = 128;                 // samples per block = threads per block
constexpr int kDirChunk = 16;                 // modes per stage
constexpr int kDirRowBytes = kDirChunk * 16 + 16;   // padded row: conflict-free 128-bit reads down a column of rows
constexpr int kDirStages = 3;
constexpr int kDirCstBytes = kDirChunk * 48;  // per-mode constants travelling with the chunk
constexpr int kDirStageBytes = kDirTile * kDirRowBytes + kDirCstBytes;
constexpr int kDirMaxStep = 8;                // |dn| up to which E is advanced step by step instead of restarted

struct dir_cst {          // 48 B per mode
    double k[4];          // Re h += k0 Wr + k1 Wi;  Im h += k2 Wr + k3 Wi
    int op;               // 0: E *= Z_r (dn = 1, same m);  1..kDirMaxStep: dn steps;  -1: restart E = Z_phi^m Z_r^n
    int m, n, pad;
};

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cp_async16(void* dst, const void* src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// z^e for e >= 0 by binary powering (e is block-uniform)
__device__ __forceinline__ void cpow(double zr, double zi, int e, double* pr, double* pi)
{
    double rr = 1.0, ri = 0.0;
    while (e) {
        if (e & 1) { const double a = rr * zr - ri * zi; ri = rr * zi + ri * zr; rr = a; }
        const double a = zr * zr - zi * zi; zi = 2.0 * zr * zi; zr = a;
        e >>= 1;
    }
    *pr = rr; *pi = ri;
}

// Per source: fold constants (with scale and the complex frame factor) and the E-walk opcodes.  One block per source.
__global__ void few_direct_prepare_kernel(const int* __restrict__ l, const int* __restrict__ m, const int* __restrict__ n,
                                          const double2* __restrict__ ylm_plus, const double2* __restrict__ ylm_minus,
                                          const double* __restrict__ scale, const double2* __restrict__ factor, int K, int K_pad,
                                          dir_cst* __restrict__ cst_all, int* status)
{
    const int src = blockIdx.x;
    dir_cst* cst = cst_all + (size_t)src * K_pad;
    const double sc = scale ? scale[src] : 1.0;
    const double2 fc = factor ? make_double2(sc * factor[src].x, sc * factor[src].y) : make_double2(sc, 0.0);
    for (int j = threadIdx.x; j < K_pad; j += blockDim.x) {
        dir_cst c;
        c.k[0] = c.k[1] = c.k[2] = c.k[3] = 0.0; c.op = 0; c.m = 0; c.n = 0; c.pad = 0;
        if (j < K) {
            int lj = l[j], mj = m[j], nj = n[j];
            const int an = nj < 0 ? -nj : nj;
            if (lj < 2 || lj > FEW_MAX_L || mj < 0 || mj > lj || an > FEW_MAX_ABS_N) { atomicOr(status, FEW_DEV_BAD_MODE); lj = 2; mj = 0; nj = 0; }
            const double2 yp = ylm_plus[(size_t)src * K + j];
            double2 yb = make_double2(0.0, 0.0);
            if (mj > 0) {                                   // Eq. (9): Ybar = (-1)^l Y_{l,-m}
                const double2 ym = ylm_minus[(size_t)src * K + j];
                const double sg = (lj & 1) ? -1.0 : 1.0;
                yb = make_double2(sg * ym.x, sg * ym.y);
            }
            const double ar = fc.x * yp.x - fc.y * yp.y, ai = fc.x * yp.y + fc.y * yp.x;     // a = f Y+
            const double br = fc.x * yb.x - fc.y * yb.y, bi = fc.x * yb.y + fc.y * yb.x;     // b = f Ybar
            c.k[0] = ar + br; c.k[1] = bi - ai; c.k[2] = ai + bi; c.k[3] = ar - br;          // a W + b conj(W)
            c.m = mj; c.n = nj;
            c.op = -1;
            if (j > 0) {
                const int mp = m[j - 1], dn = nj - n[j - 1];
                if (mp == mj && dn >= 1 && dn <= kDirMaxStep) c.op = dn == 1 ? 0 : dn;
            }
        }
        cst[j] = c;
    }
}

__global__ void __launch_bounds__(kDirTile, 2)
few_direct_kernel(const double2* __restrict__ amp_all, const double2* __restrict__ phase_all, const dir_cst* __restrict__ cst_all,
                  long long N, int K, int K_pad, double2* __restrict__ h_all)
{
    extern __shared__ __align__(128) unsigned char dsm[];
    const int tid = threadIdx.x, src = blockIdx.y;
    const long long i0 = (long long)blockIdx.x * kDirTile;
    const int rows = (int)((N - i0) < kDirTile ? (N - i0) : kDirTile);
    const double2* amp = amp_all + ((size_t)src * N + i0) * K;
    const unsigned char* cst_g = reinterpret_cast<const unsigned char*>(cst_all + (size_t)src * K_pad);
    const int n_chunks = K_pad / kDirChunk;

    // stage c: piece p = tid + kDirTile * u is the 16 bytes of mode c*16 + (p & 15) of row p >> 4
    auto issue = [&](int c) {
        unsigned char* st = dsm + (size_t)(c % kDirStages) * kDirStageBytes;
        const int cnt = (K - c * kDirChunk) < kDirChunk ? (K - c * kDirChunk) : kDirChunk;     // ragged last chunk
        const int q = tid & (kDirChunk - 1);
        const double2* g = amp + (size_t)c * kDirChunk + q;
        if (q < cnt) {
#pragma unroll
            for (int u = 0; u < kDirChunk; ++u) {
                const int r = (tid >> 4) + u * (kDirTile / kDirChunk);
                if (r < rows) cp_async16(st + r * kDirRowBytes + q * 16, g + (size_t)r * K);
            }
        }
        if (tid < kDirCstBytes / 16) cp_async16(st + kDirTile * kDirRowBytes + tid * 16, cst_g + (size_t)c * kDirCstBytes + tid * 16);
    };
    for (int c = 0; c < kDirStages - 1; ++c) { if (c < n_chunks) issue(c); cp_async_commit(); }

    // per-sample phase factors (overlaps the first copies)
    double zpr = 1.0, zpi = 0.0, zrr = 1.0, zri = 0.0;
    if (tid < rows) {
        const double2 ph = phase_all[(size_t)src * N + i0 + tid];
        double s, c;
        sincos(ph.x, &s, &c); zpr = c; zpi = -s;
        sincos(ph.y, &s, &c); zrr = c; zri = -s;
    }
    double pr = 1.0, pi = 0.0;          // Z_phi^m of the current run
    int m_cur = 0;
    double er = 1.0, ei = 0.0, hr = 0.0, hi = 0.0;

    for (int c = 0; c < n_chunks; ++c) {
        cp_async_wait<kDirStages - 2>();                            // this thread's pieces of stage c have landed
        __syncthreads();                                            // ... everyone's have; stage c-1 is fully consumed
        if (c + kDirStages - 1 < n_chunks) issue(c + kDirStages - 1);
        cp_async_commit();                                          // one group per iteration, empty or not
        const unsigned char* st = dsm + (size_t)(c % kDirStages) * kDirStageBytes;
        const double2* row = reinterpret_cast<const double2*>(st + tid * kDirRowBytes);
        const dir_cst* cs = reinterpret_cast<const dir_cst*>(st + kDirTile * kDirRowBytes);
        const int cnt = (K - c * kDirChunk) < kDirChunk ? (K - c * kDirChunk) : kDirChunk;
#pragma unroll 4
        for (int q = 0; q < cnt; ++q) {
            const int op = cs[q].op;
            if (op == 0) {
                const double a = er * zrr - ei * zri; ei = er * zri + ei * zrr; er = a;
            } else if (op > 0) {
                for (int u = 0; u < op; ++u) { const double a = er * zrr - ei * zri; ei = er * zri + ei * zrr; er = a; }
            } else {
                const int mj = cs[q].m, nj = cs[q].n;
                if (mj >= m_cur && mj - m_cur <= kDirMaxStep) {
                    for (int u = m_cur; u < mj; ++u) { const double a = pr * zpr - pi * zpi; pi = pr * zpi + pi * zpr; pr = a; }
                } else {
                    cpow(zpr, zpi, mj, &pr, &pi);
                }
                m_cur = mj;
                double qr, qi;
                cpow(zrr, nj < 0 ? -zri : zri, nj < 0 ? -nj : nj, &qr, &qi);
                er = pr * qr - pi * qi; ei = pr * qi + pi * qr;
            }
            const double2 a = row[q];
            const double wr = a.x * er - a.y * ei, wi = a.x * ei + a.y * er;
            const double4 k = *reinterpret_cast<const double4*>(cs[q].k);
            hr = fma(k.x, wr, fma(k.y, wi, hr));
            hi = fma(k.z, wr, fma(k.w, wi, hi));
        }
    }
    if (tid < rows) __stcs(&h_all[(size_t)src * N + i0 + tid], make_double2(hr, hi));
}

inline int dir_kpad(int K) { return (K + kDirChunk - 1) / kDirChunk * kDirChunk; }

}  // namespace

extern "C" size_t few_sum_direct_workspace(int n_src, int n_modes)
{
    if (n_src <= 0 || n_modes <= 0) return 0;
    return few_align_up((size_t)n_src * dir_kpad(n_modes) * sizeof(dir_cst));
}

extern "C" int few_sum_direct(few_ctx* ctx, const double* amp, const double* phase, const int* l, const int* m, const int* n,
                              const double* ylm_plus, const double* ylm_minus, const double* scale, const double* factor,
                              long long n_samples, int n_src, int n_modes, double* h,
                              void* workspace, size_t workspace_bytes, void* stream)
{
    FEW_REQUIRE(ctx && l && m && n && ylm_plus && ylm_minus, FEW_ERR_INVALID_ARG, "NULL argument");
    FEW_REQUIRE(n_src > 0 && n_src <= 65535 && n_modes > 0 && n_samples >= 0, FEW_ERR_INVALID_ARG, "bad sizes");
    if (n_samples == 0) return FEW_OK;
    FEW_REQUIRE(amp && phase && h, FEW_ERR_INVALID_ARG, "amp, phase or h is NULL");
    FEW_REQUIRE(workspace && ((uintptr_t)workspace % 256) == 0 && workspace_bytes >= few_sum_direct_workspace(n_src, n_modes),
                FEW_ERR_WORKSPACE, "workspace NULL, misaligned or too small");
    const long long tiles = (n_samples + kDirTile - 1) / kDirTile;
    FEW_REQUIRE(tiles < 2147483647LL, FEW_ERR_LIMIT, "n_samples too large");
    cudaStream_t st = (cudaStream_t)stream;
    const int K_pad = dir_kpad(n_modes);
    dir_cst* cst = static_cast<dir_cst*>(workspace);
    few_direct_prepare_kernel<<<n_src, 256, 0, st>>>(l, m, n, (const double2*)ylm_plus, (const double2*)ylm_minus, scale,
                                                     (const double2*)factor, n_modes, K_pad, cst, ctx->d_status);
    FEW_LAUNCHED(ctx);
    const size_t smem = (size_t)kDirStages * kDirStageBytes;
    FEW_CUDA_CHECK(cudaFuncSetAttribute(few_direct_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    few_direct_kernel<<<dim3((unsigned)tiles, n_src), kDirTile, smem, st>>>((const double2*)amp, (const double2*)phase, cst, n_samples,
                                                                           n_modes, K_pad, (double2*)h);
    FEW_LAUNCHED(ctx);
    return FEW_OK;
}
