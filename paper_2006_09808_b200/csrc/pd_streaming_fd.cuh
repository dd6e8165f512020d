// pd_streaming_fd.cuh -- the streaming variant: dual variable p kept in the FOURIER domain when W = identity (two
// launches per iteration, described first); the literal iteration for W != I on the same planes (four launches,
// sfd_dual_rows_kernel and sfd_cols_kernel<PLAIN> further down).
//
// Same algebra as pd_resident_tm.cuh (PAPER.md:49 line 1 commutes with the FFT when W = I):
//     p^_{n+1} = (p^_n + sigma (D X^_n - phi^)) / (1 + sigma),   X^_n = F chibar_n,   K p_{n+1} = F^-1 (D p^_{n+1}),
// so one iteration is ONE forward 2-D FFT and ONE inverse: two launches over the whole batch instead of four,
//   fd_cols : column FFT of Z (= X^_n), p^ update, column FFT of conj(D/(nx ny) p^_{n+1})      [PAPER.md:49 line 1]
//   fd_rows : row FFT (finishes K p_{n+1}), q-update, G^T M q_{n+1}, chi-update, over-relaxation,
//             row FFT of chibar_{n+1}                                                         [PAPER.md:49 lines 2-4]
// All state is pair-interleaved float2 [npairs][ny][nx] (lane x = slice 2j, lane y = slice 2j+1): every access of a
// group of T threads is one contiguous 8T-byte segment.  chibar and q are double-buffered by iteration parity, so
// that a row group can redo the q-update of the row ABOVE its own (it needs (M qy_{n+1})[y-1] for the divergence)
// from read-only data: no exchange between rows, no CTA-wide barrier; the duplicate loads hit L1/L2.
// chi and p^ are double-buffered too: then every load inside the update loops is from data that is read-only for
// the launch (ld.global.nc), which the scheduler may hoist above the stores of earlier elements -- with in-place
// updates every element would expose one full memory latency (load -> use -> store -> next load).
//
// chibar is never stored: chibar_n = chi_n + theta (chi_n - chi_{n-1}) is recomputed (bit-identically) from the two
// last iterates, which a third chi buffer keeps readable while chi_{n+1} is written.  Without a mask (M = 1) the
// mask plane is neither built nor read.
//
// HBM bytes per pixel PAIR and iteration: fd_cols Z r8 w8, phi^ r8, p^ r8 w8 = 40 ; fd_rows Z r8 w8, chi_n r8,
// chi_{n-1} r8, chi_{n+1} w8, qx r8 w8, qy r8 w8, M r8 = 80  ->  60 B per pixel of one slice and iteration, 56 without
// a mask.
//
// Gap (R9): data term by Parseval over mirror-paired columns (as in pd_resident_tm.cuh), q term in fd_rows;
// both as per-CTA partial sums.  Every CTA of fd_cols(n+1) reduces the partials of iteration n in the same fixed
// order and reaches the same stop decision; column block 0 records it.  No host round trip.
#pragma once
#include "pd_resident.cuh"    // packed fp32x2 helpers, FFT building blocks (fft_regs.cuh)

namespace pdk {

struct StreamFdArgs {
    int nx, ny, batch, npairs, max_iters, check_every, aniso;
    float alpha, sigma, tau, theta, inv_one_plus_sigma, tol;
    const float *field, *mask, *weight;
    long long mask_bstride;
    float *chi_out;
    float2 *Z, *phihat, *M2;                 // [npairs][ny][nx]
    float2 *W2;                              // literal path only: interleaved W; phihat then holds phi itself
    int literal;                             // 1: W != I or PD_OPT_FOURIER_DUAL = 0 (p kept in the image domain)
    int reg_l1;                              // 1: PD_REG_L1 (l1 on chi, shrinkage) instead of the paper's TV term
    int cols_contig;                         // general-length plan with a power-of-two ny: the PLAIN column kernel runs over
                                             // ceil(nx / 16) column blocks, the last one ragged
    float2 *phat[2], *qx2[2], *qy2[2];       // double-buffered by iteration parity: iteration n reads [n&1]
    float2 *chi3[3];                         // chi_n in [n%3], chi_{n-1} in [(n+2)%3], chi_{n+1} written to [(n+1)%3]
    const float *Dtab;                       // D/(nx*ny), [ny][nx]
    const float2 *tw_row, *tw_col;
    int *stop_iter;                          // slice b is active in iteration n (0-based) iff n < stop_iter[b]
    float *P0, *relgap, *relres;
    float *cscale;                           // [batch] power-of-two normalisation of every slice (pair_scale, pd_resident.cuh)
    int *iters_done;
    float *p0_part;                          // [npairs][nrowparts][2]
    float *gap_col[2];                       // [npairs][ncolparts][2], by iteration parity
    float *gap_row;                          // [npairs][nrowparts][2]
    float *res_part;                         // [npairs][nrowparts][4] (dn_a, cn_a, dn_b, cn_b)
    int ncolparts, nrowparts;
    int *iter;                               // device iteration counter of the graphed loop (kernels launched with n < 0 read it)
};

template <int N> struct SfdRowCfg {
    static constexpr int E = FftCfg<N>::E, T = FftCfg<N>::T;
    static constexpr int THREADS = 128;
    static constexpr int G = THREADS / T;
    static constexpr int LD = T + 1;
    static constexpr int SM_PER_GROUP = E * LD > FftCfg<N>::REGION ? E * LD : FftCfg<N>::REGION;
#ifndef PD_SFD_STAGE_MIN
#define PD_SFD_STAGE_MIN 256
#endif
    static constexpr bool STAGE = N >= PD_SFD_STAGE_MIN;   // park the spectrum in shared memory during the update loop
    // CTAs per SM the row kernel is compiled for (register cap 65536 / (128 MINB)).  4 (128 registers) measured 1.5-3 %
    // faster than 5 (96 registers) on both sizes, 6 and 7 slower (profiles/r02/README.md)
#ifndef PD_SFD_ROWS512_MINB
#define PD_SFD_ROWS512_MINB 4
#endif
#ifndef PD_SFD_ROWS256_MINB
#define PD_SFD_ROWS256_MINB 4
#endif
    static constexpr int MINB = N == 512 ? PD_SFD_ROWS512_MINB : (STAGE ? PD_SFD_ROWS256_MINB : 4);
#ifndef PD_SFD_UNROLL
#define PD_SFD_UNROLL 4
#endif
    static constexpr int UNROLL = PD_SFD_UNROLL;           // elements of the update loop per unrolled body (STAGE only)
};
template <int N, bool PLAIN = false> struct SfdColCfg {
    using Fft = FftCfg<N, true>;                       // column configuration of the line transform (fft_regs.cuh)
    static constexpr int E = Fft::E, T = Fft::T;
#ifndef PD_SFD_COLS512_HALF
#define PD_SFD_COLS512_HALF 16
#endif
    // HALF adjacent columns and their HALF mirror images per CTA: 64-byte segments at HALF = 8, whole 128-byte lines at 16.
    // 16 + 16 columns of 512 points are 512 threads and 131 KB, one CTA per SM: measured 7 % faster for the Fourier-domain
    // kernel at 512 (every C4 iteration takes the Parseval sums, i.e. the mirror-paired mapping: 33.1 -> 30.9 ms per step)
    // and 8 % slower for the PLAIN kernel, which always runs over contiguous blocks and keeps 16 columns, two CTAs per SM.
    static constexpr int HALF = (N == 512 && !PLAIN) ? PD_SFD_COLS512_HALF : 8, COLS = 2 * HALF;
    static constexpr int THREADS = COLS * T;
    static constexpr int CS = N + 1 > Fft::REGION ? N + 1 : Fft::REGION + 1;   // odd column stride
    static constexpr int SMEM_BYTES = (COLS * CS + Fft::TW) * (int)sizeof(float2) + 256;
#ifndef PD_SFD_COL_STAGE_MIN
#define PD_SFD_COL_STAGE_MIN 256
#endif
    static constexpr bool STAGE = N >= PD_SFD_COL_STAGE_MIN;   // park the spectrum in shared memory during the p^ update
};

// column kx of (column block cb, half h, slot cc): [8cb, 8cb+8) and its mirror images nx - kx; the self-mirrored
// columns 0 and nx/2 both sit in block 0, slot 0.
__host__ __device__ constexpr int sfd_column_of(int nx, int cb, int h, int cc, int half = 8) {
    const int lo = half * cb + cc;
    return h == 0 ? lo : (lo == 0 ? nx / 2 : nx - lo);
}

// L2 prefetch of one 128-byte line: no register is held while the line travels (used to start the operand rows of the
// update loops before the first FFT of a line)
__device__ __forceinline__ void prefetch_l2(const void *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// relgap of the pair's two lanes from the partial sums of iteration parity `par`, fixed order (same in every CTA)
__device__ __forceinline__ float2 sfd_gap_sum(const StreamFdArgs &a, int pair, int par) {
    float ga = 0.f, gb = 0.f;
    const float *gc = a.gap_col[par] + (long long)pair * a.ncolparts * 2;
    for (int k = 0; k < a.ncolparts; ++k) { ga += __ldcg(gc + 2 * k); gb += __ldcg(gc + 2 * k + 1); }
    const float *gr = a.gap_row + (long long)pair * a.nrowparts * 2;
    for (int k = 0; k < a.nrowparts; ++k) { ga += __ldcg(gr + 2 * k); gb += __ldcg(gr + 2 * k + 1); }
    return make_float2(ga, gb);
}

// The same sums by one whole warp: lane l takes the partials l, l + 32, ... of either array, then a butterfly over the
// lanes -- a fixed order again, so every CTA of a launch reaches the same value, at one L2 latency instead of
// ncolparts + nrowparts dependent additions by a single thread.  Result valid in every lane.
__device__ __forceinline__ float2 sfd_gap_sum_warp(const StreamFdArgs &a, const int pair, const int par, const int lane) {
    float ga = 0.f, gb = 0.f;
    const float *gc = a.gap_col[par] + (long long)pair * a.ncolparts * 2;
    for (int k = lane; k < a.ncolparts; k += 32) { ga += __ldcg(gc + 2 * k); gb += __ldcg(gc + 2 * k + 1); }
    const float *gr = a.gap_row + (long long)pair * a.nrowparts * 2;
    for (int k = lane; k < a.nrowparts; k += 32) { ga += __ldcg(gr + 2 * k); gb += __ldcg(gr + 2 * k + 1); }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        ga += __shfl_xor_sync(0xffffffffu, ga, o);
        gb += __shfl_xor_sync(0xffffffffu, gb, o);
    }
    return make_float2(ga, gb);
}

// ------------------------------------------------------------------------------------------------ normalisation
// c_b = 2^-floor(log2 rms(phi_b)) of every slice (pair_scale): one CTA per slice, fixed summation order.
__global__ void __launch_bounds__(256)
sfd_scale_kernel(const StreamFdArgs a) {
    __shared__ float red[8];
    const int b = blockIdx.x;
    const long long P = (long long)a.nx * a.ny;
    const float4 *f = reinterpret_cast<const float4 *>(a.field + (long long)b * P);
    float s = 0.f;
    for (int i = threadIdx.x; i < (int)(P / 4); i += 256) {
        const float4 v = __ldg(f + i);
        s = fmaf(v.x, v.x, fmaf(v.y, v.y, fmaf(v.z, v.z, fmaf(v.w, v.w, s))));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        float t = 0.f;
        for (int w = 0; w < 8; ++w) t += red[w];
        a.cscale[b] = pair_scale(t, (float)P);
    }
}

// ------------------------------------------------------------------------------------------------ init
// Load the pair's field rows (normalised, see sfd_scale_kernel), interleave the mask, zero the state that iteration 0 reads, partial sums of
// 1/2 ||phi||^2, row FFT of phi -> Z.  (chi_0 = chibar_0 = p_0 = q_0 = 0.)
template <int NX>
__global__ void __launch_bounds__(SfdRowCfg<NX>::THREADS)
sfd_init_rows_kernel(const StreamFdArgs a) {
    using Cfg = SfdRowCfg<NX>;
    constexpr int E = Cfg::E, T = Cfg::T, G = Cfg::G;
    __shared__ float2 sm[G * Cfg::SM_PER_GROUP];
    __shared__ float2 tws[FftCfg<NX>::TW];
    __shared__ float red[G][2];
    TwiddlesSmem<NX>::fill(tws, a.tw_row, threadIdx.x, Cfg::THREADS);
    __syncthreads();
    const int pair = blockIdx.y, s0 = 2 * pair, s1 = s0 + 1;
    const bool has_b = s1 < a.batch;
    const int g = threadIdx.x / T, j = threadIdx.x % T;
    const int y = blockIdx.x * G + g;
    const long long P = (long long)NX * a.ny, rowoff = (long long)y * NX, po = (long long)pair * P + rowoff;
    TwiddlesSmem<NX> tw;
    tw.w = tws + j;
    const float *fa = a.field + (long long)s0 * P + rowoff;
    const float *fb = a.field + (long long)s1 * P + rowoff;
    const float *ma = a.mask ? a.mask + s0 * a.mask_bstride + rowoff : nullptr;
    const float *mb = a.mask ? a.mask + s1 * a.mask_bstride + rowoff : nullptr;
    const float2 zero = make_float2(0.f, 0.f);
    const float ca = a.cscale[s0], cb = has_b ? a.cscale[s1] : 0.f;
    float2 v[E];
    float acc0 = 0.f, acc1 = 0.f;
#pragma unroll
    for (int m = 0; m < E; ++m) {
        const int x = j + T * m;
        const float va = ca * fa[x], vb = has_b ? cb * fb[x] : 0.f;
        v[m] = make_float2(va, vb);
        float wa = 1.f, wb = 1.f;
        if (a.literal) {   // phi and W interleaved, p_0 = 0; P0 = 1/2 ||W phi||^2
            if (a.weight) { wa = a.weight[(long long)s0 * P + rowoff + x]; wb = has_b ? a.weight[(long long)s1 * P + rowoff + x] : 0.f; }
            a.phihat[po + x] = v[m];
            a.W2[po + x] = make_float2(wa, wb);
            a.phat[0][po + x] = zero;
        }
        acc0 = fmaf(wa * va, wa * va, acc0);
        acc1 = fmaf(wb * vb, wb * vb, acc1);
        if (ma) a.M2[po + x] = make_float2(ma[x], has_b ? mb[x] : 0.f);
        a.chi3[0][po + x] = zero; a.chi3[2][po + x] = zero; a.qx2[0][po + x] = zero; a.qy2[0][po + x] = zero;
    }
    if (!a.literal) {   // phi^ needs the transform of the field; the literal path starts from chibar_0 = 0
        fft_line<NX, Cfg::LD>(v, sm + g * Cfg::SM_PER_GROUP, j, tw, WarpSync());
#pragma unroll
        for (int m = 0; m < E; ++m) a.Z[po + j + T * m] = v[m];
    }
    acc0 = group_sum<T>(acc0);
    acc1 = group_sum<T>(acc1);
    if (j == 0) { red[g][0] = acc0; red[g][1] = acc1; }
    __syncthreads();
    if (threadIdx.x < 2) {
        float t = 0.f;
        for (int k = 0; k < G; ++k) t += red[k][threadIdx.x];
        a.p0_part[((long long)pair * a.nrowparts + blockIdx.x) * 2 + threadIdx.x] = t;
    }
}

// phi^ = column FFT of the row-transformed field; p^_0 = 0; column block 0 finishes P0 and resets the per-slice state.
template <int NY>
__global__ void __launch_bounds__(SfdColCfg<NY>::THREADS)
sfd_init_cols_kernel(const StreamFdArgs a) {
    using Cfg = SfdColCfg<NY>;
    constexpr int E = Cfg::E, T = Cfg::T;
    extern __shared__ __align__(16) unsigned char sfd_smem[];
    float2 *smc = reinterpret_cast<float2 *>(sfd_smem);
    float2 *tws = smc + Cfg::COLS * Cfg::CS;
    TwiddlesSmem<NY, true>::fill(tws, a.tw_col, threadIdx.x, Cfg::THREADS);
    __syncthreads();
    const int pair = blockIdx.y, s0 = 2 * pair, s1 = s0 + 1;
    const int c = threadIdx.x & (Cfg::COLS - 1), j = threadIdx.x / Cfg::COLS;
    const int kx = sfd_column_of(a.nx, blockIdx.x, c / Cfg::HALF, c % Cfg::HALF, Cfg::HALF);
    const long long po = (long long)pair * a.nx * NY + kx;
    TwiddlesSmem<NY, true> tw;
    tw.w = tws + j;
    if (!a.literal) {
        float2 v[E];
#pragma unroll
        for (int m = 0; m < E; ++m) v[m] = a.Z[po + (long long)(j + T * m) * a.nx];
        fft_line<NY, T>(v, smc + c * Cfg::CS, j, tw, BlockSync());
        const float2 zero = make_float2(0.f, 0.f);
#pragma unroll
        for (int m = 0; m < E; ++m) {
            a.phihat[po + (long long)(j + T * m) * a.nx] = v[m];
            a.phat[0][po + (long long)(j + T * m) * a.nx] = zero;
        }
    }
    if (blockIdx.x == 0 && threadIdx.x < 2) {
        const int b = threadIdx.x ? s1 : s0;
        if (b < a.batch) {
            float t = 0.f;
            const float *pp = a.p0_part + (long long)pair * a.nrowparts * 2 + threadIdx.x;
            for (int k = 0; k < a.nrowparts; ++k) t += pp[2 * k];
            const float P0 = 0.5f * t;
            a.P0[b] = P0;
            a.relgap[b] = 0.f;
            a.relres[b] = 0.f;
            a.stop_iter[b] = (P0 == 0.f) ? 0 : a.max_iters;   // R13b: an all-zero slice is never scheduled
        }
    }
    if (blockIdx.x == 0)
        for (int k = threadIdx.x; k < a.nrowparts * 4; k += Cfg::THREADS) a.res_part[(long long)pair * a.nrowparts * 4 + k] = 0.f;
}

// ------------------------------------------------------------------------------------------------ column kernel
// Iteration n.  First the stop decision of iteration n-1 (if it was a checking iteration): every CTA of the pair
// reduces the same partial sums in the same order; block 0 records relgap and stop_iter.  Then
//   X^ = column FFT of Z (zero when n == 0) ; p^_{n+1} = (p^_n + sigma (D X^ - phi^))/(1 + sigma) ;
//   Z <- column FFT of conj(D/(nx ny) p^_{n+1})      (the row kernel's FFT finishes the inverse transform)
// want_gap: Sa = sum |dp(k) + conj dp(-k)|^2, Sb = sum |dp(k) - conj dp(-k)|^2, dp = p^_{n+1} - p^_n -- the two lanes'
// spectra accumulated directly (no difference of two large sums, so a weak slice does not lose digits to a strong
// partner); the mirror column is in this CTA.
// PLAIN (literal path): only Z <- column FFT of conj(D/(nx ny) X^), i.e. one application of K between two row passes;
// `decide` is set for the first of the two column launches of an iteration.
// NXC: the row length as a compile-time constant (square slices: NXC = NY) or 0 (taken from the arguments).  With a
// constant row pitch every access of a thread is base + immediate; with a run-time pitch the 64-bit address arithmetic
// of the five strided arrays was 28 % of the instructions of the 512-point kernel (profiles/r02/README.md).
template <int NY, bool PLAIN, int NXC>
__global__ void __launch_bounds__(SfdColCfg<NY, PLAIN>::THREADS, SfdColCfg<NY, PLAIN>::THREADS <= 128 ? 4 : (SfdColCfg<NY, PLAIN>::THREADS <= 256 ? 2 : 1))
sfd_cols_kernel(const StreamFdArgs a, const int n_arg, const int do_decide) {
    const int n = n_arg >= 0 ? n_arg : *a.iter;      // inside the graphed loop the iteration number lives on the device
    if (PLAIN && do_decide && n == 0) return;        // literal path: chibar_0 = 0, the first K application of iteration 0 is skipped
    using Cfg = SfdColCfg<NY, PLAIN>;
    constexpr int E = Cfg::E, T = Cfg::T, NT = Cfg::THREADS;
    extern __shared__ __align__(16) unsigned char sfd_smem[];
    float2 *smc = reinterpret_cast<float2 *>(sfd_smem);
    float2 *tws = smc + Cfg::COLS * Cfg::CS;
    float *dec = reinterpret_cast<float *>(tws + Cfg::Fft::TW);   // [0..1] stop flags of this launch ; [2..] reduction

    const int pair = blockIdx.y, s0 = 2 * pair, s1 = s0 + 1;
    const bool has_b = s1 < a.batch;
    int stop0 = a.stop_iter[s0], stop1 = has_b ? a.stop_iter[s1] : 0;
    if (n >= stop0 && n >= stop1) return;

    const bool decide = do_decide && n > 0 && a.tol > 0.f && (n % a.check_every) == 0;   // iteration n-1 was a checking one
    if (decide) {
        if (threadIdx.x < 32) {
            const float2 g = sfd_gap_sum_warp(a, pair, (n - 1) & 1, threadIdx.x);
            if (threadIdx.x == 0) {
                const float P0a = a.P0[s0], P0b = has_b ? a.P0[s1] : 0.f;
                const float ra = P0a > 0.f ? g.x / P0a : 0.f, rb = P0b > 0.f ? g.y / P0b : 0.f;
                int f0 = 0, f1 = 0;
                if (n < stop0 && ra < a.tol) f0 = 1;
                if (n < stop1 && rb < a.tol) f1 = 1;
                dec[0] = (float)f0; dec[1] = (float)f1;
                if (blockIdx.x == 0) {
                    if (n < stop0) { a.relgap[s0] = ra; if (f0) a.stop_iter[s0] = n; }
                    if (n < stop1) { a.relgap[s1] = rb; if (f1) a.stop_iter[s1] = n; }
                }
            }
        }
        __syncthreads();
        if (dec[0] != 0.f) stop0 = n;
        if (dec[1] != 0.f) stop1 = n;
        if (n >= stop0 && n >= stop1) return;
    }
    const bool last = (n + 1 == a.max_iters);
    const bool want_gap = !PLAIN && (last || (a.tol > 0.f && ((n + 1) % a.check_every) == 0));

    TwiddlesSmem<NY, true>::fill(tws, a.tw_col, threadIdx.x, NT);
    const int c = threadIdx.x & (Cfg::COLS - 1), j = threadIdx.x / Cfg::COLS;
    const int h = c / Cfg::HALF, cc = c % Cfg::HALF;
    const int nx = NXC ? NXC : a.nx;
    // Mirror-paired columns are needed only where the Parseval sums are taken (want_gap).  Everywhere else CTA cb owns the
    // CONTIGUOUS columns [16 cb, 16 cb + 16): a warp's access then touches two 128-byte lines (two rows) instead of four
    // (two rows x an adjacent and a mirrored 64-byte segment) -- the load/store path is what limits this kernel
    // (profiles/r02/ncu_sfd_cols_c4.md: MIO throttle first, L1TEX 70 %).  With a.cols_contig (general-length plans, nx not a
    // multiple of 16) the last block is ragged: its surplus threads redo column nx - 1 (they must reach the barriers) and do not store.
    const bool contig = PLAIN || !want_gap;
    const int kx_raw = contig ? Cfg::COLS * (int)blockIdx.x + c : sfd_column_of(nx, blockIdx.x, h, cc, Cfg::HALF);
    const bool kx_valid = kx_raw < nx;
    const int kx = kx_valid ? kx_raw : nx - 1;
    const bool self_mirror = (blockIdx.x == 0 && cc == 0);
    float2 *smg = smc + c * Cfg::CS;
    const float2 *smg_mir = self_mirror ? smg : smc + (c ^ Cfg::HALF) * Cfg::CS;
    const long long po = (long long)pair * nx * NY + kx;
    float2 *zc = a.Z + po, *phw = a.phat[(n & 1) ^ 1] + po;
    const float2 *phh = a.phihat + po, *phr = a.phat[n & 1] + po;
    const float *dcol = a.Dtab + kx;
    TwiddlesSmem<NY, true> tw;
    tw.w = tws + j;
    __syncthreads();

    float2 v[E];
    if (n > 0 || PLAIN) {
#pragma unroll
        for (int m = 0; m < E; ++m) v[m] = __ldcs(zc + (long long)(j + T * m) * nx);
        if (!PLAIN && cc == 1) {   // the 64-byte segments of phi^ and p^_n this half-block of 8 columns will read
#pragma unroll
            for (int m = 0; m < E; ++m) { prefetch_l2(phh + (long long)(j + T * m) * nx); prefetch_l2(phr + (long long)(j + T * m) * nx); }
        }
        fft_line<NY, T>(v, smg, j, tw, BlockSync());
    } else {
#pragma unroll
        for (int m = 0; m < E; ++m) v[m] = make_float2(0.f, 0.f);
    }
    const float2 sig2 = splat(a.sigma), inv2 = splat(a.inv_one_plus_sigma);
    const float NN = (float)nx * (float)NY;
    float Sa = 0.f, Sb = 0.f;
    if (PLAIN) {
#pragma unroll
        for (int m = 0; m < E; ++m) {
            const float d = __ldg(dcol + (long long)(j + T * m) * nx);
            v[m] = make_float2(d * v[m].x, -d * v[m].y);
        }
    } else if (Cfg::STAGE) {
        // Park X^ in the column's exchange region (slot ky), so that the registers hold the loads of the update in
        // flight instead of the spectrum; each slot then receives p^_{n+1}, from which both the Parseval sums and
        // the next transform's input are taken.
        __syncthreads();   // every thread's second FFT stage has read the region
#pragma unroll
        for (int m = 0; m < E; ++m) smg[j + T * m] = v[m];
#pragma unroll
        for (int m = 0; m < E; ++m) {
            const long long o = (long long)(j + T * m) * nx;
            const float d = __ldg(dcol + o);
            const float2 phat = __ldg(phh + o);
            const float2 pold = __ldg(phr + o);
            const float2 res = sub2(mul2(splat(d * NN), smg[j + T * m]), phat);
            const float2 pn = mul2(fma2(sig2, res, pold), inv2);
            __stcs(phw + o, pn);
            smg[j + T * m] = pn;
        }
        if (want_gap) {   // dp(k) dp(-k): p^_{n+1} of the mirror element from its slot, p^_n of both reloaded (L1/L2)
            __syncthreads();
            const float2 *phr_mir = a.phat[n & 1] + (long long)pair * nx * NY + (self_mirror ? kx : sfd_column_of(nx, blockIdx.x, h ^ 1, cc, Cfg::HALF));
#pragma unroll
            for (int m = 0; m < E; ++m) {
                const int ky = j + T * m, kym = (NY - ky) & (NY - 1);
                const float2 dp = sub2(smg[ky], __ldg(phr + (long long)ky * nx));
                const float2 dm = sub2(smg_mir[kym], __ldg(phr_mir + (long long)kym * nx));
                const float ax = dp.x + dm.x, ay = dp.y - dm.y, bx = dp.x - dm.x, by = dp.y + dm.y;
                Sa = fmaf(ax, ax, fmaf(ay, ay, Sa));
                Sb = fmaf(bx, bx, fmaf(by, by, Sb));
            }
        }
#pragma unroll
        for (int m = 0; m < E; ++m) {
            const float d = __ldg(dcol + (long long)(j + T * m) * nx);
            const float2 pn = smg[j + T * m];
            v[m] = make_float2(d * pn.x, -d * pn.y);
        }
    } else {
        if (want_gap) __syncthreads();   // the exchange region is free (readers of the FFT above are done)
#pragma unroll
        for (int m = 0; m < E; ++m) {
            const long long o = (long long)(j + T * m) * nx;
            const float d = __ldg(dcol + o);
            const float2 phat = __ldg(phh + o);
            const float2 pold = __ldg(phr + o);
            const float2 res = sub2(mul2(splat(d * NN), v[m]), phat);
            const float2 pn = mul2(fma2(sig2, res, pold), inv2);
            if (want_gap) smg[j + T * m] = sub2(pn, pold);
            __stcs(phw + o, pn);
            v[m] = make_float2(d * pn.x, -d * pn.y);
        }
        if (want_gap) {
            __syncthreads();
#pragma unroll
            for (int m = 0; m < E; ++m) {
                const int ky = j + T * m;
                const float2 dp = smg[ky];
                const float2 dm = smg_mir[(NY - ky) & (NY - 1)];
                const float ax = dp.x + dm.x, ay = dp.y - dm.y, bx = dp.x - dm.x, by = dp.y + dm.y;
                Sa = fmaf(ax, ax, fmaf(ay, ay, Sa));
                Sb = fmaf(bx, bx, fmaf(by, by, Sb));
            }
        }
    }
    fft_line<NY, T>(v, smg, j, tw, BlockSync());
    if (kx_valid) {
#pragma unroll
        for (int m = 0; m < E; ++m) __stcs(zc + (long long)(j + T * m) * nx, v[m]);
    }

    if (want_gap) {   // CTA sums in fixed order: warp shuffles, then warp 0 over the per-warp values
        __syncthreads();
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            Sa += __shfl_xor_sync(0xffffffffu, Sa, o);
            Sb += __shfl_xor_sync(0xffffffffu, Sb, o);
        }
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
        if (lane == 0) { dec[2 + 2 * warp] = Sa; dec[3 + 2 * warp] = Sb; }
        __syncthreads();
        if (threadIdx.x == 0) {
            float t1 = 0.f, t2 = 0.f;
            for (int w = 0; w < NT / 32; ++w) { t1 += dec[2 + 2 * w]; t2 += dec[3 + 2 * w]; }
            // 1/2 sum_x e^2 = sum_k |dp(k) +- conj dp(-k)|^2 / (8 nx ny sigma^2)   (Parseval; pd_resident_tm.cuh header)
            const float scale = 0.125f / (NN * a.sigma * a.sigma);
            float *gc = a.gap_col[n & 1] + ((long long)pair * a.ncolparts + blockIdx.x) * 2;
            gc[0] = scale * t1;
            gc[1] = scale * t2;
        }
    }
}

// ------------------------------------------------------------------------------------------------ row kernel
// isotropic / anisotropic projection of (tx, ty) onto the alpha-ball, both lanes (PAPER.md:49 line 2; R4, R13)
// alpha is per lane: every slice is iterated in its own normalisation (pair_scale)
__device__ __forceinline__ void sfd_project(float2 &tx, float2 &ty, const float2 alpha, const float2 alpha_sq, const bool aniso) {
    if (aniso) {
        tx.x = fminf(fmaxf(tx.x, -alpha.x), alpha.x); tx.y = fminf(fmaxf(tx.y, -alpha.y), alpha.y);
        ty.x = fminf(fmaxf(ty.x, -alpha.x), alpha.x); ty.y = fminf(fmaxf(ty.y, -alpha.y), alpha.y);
    } else {
        const float2 n2 = fma2(ty, ty, mul2(tx, tx));
        float2 sc;
        sc.x = proj_factor<kStreamingFastProj>(alpha.x, alpha_sq.x, n2.x);
        sc.y = proj_factor<kStreamingFastProj>(alpha.y, alpha_sq.y, n2.y);
        tx = mul2(tx, sc);
        ty = mul2(ty, sc);
    }
}

// Iteration n, one row y per group of T threads (same warp):
//   v = K p_{n+1}: row FFT of Z gives (v_a, -v_b)
//   q_{n+1} = proj_alpha(q_n + sigma M G chibar_n) for row y (stored) and, redundantly, its qy for row y-1
//   d = G^T (M q_{n+1}) ; chi_{n+1} = chi_n - tau (v + d) ; chibar_{n+1} = chi_{n+1} + theta (chi_{n+1} - chi_n)
//   Z <- row FFT of chibar_{n+1}
template <int NX, bool MASKED, bool ANISO>
__global__ void __launch_bounds__(SfdRowCfg<NX>::THREADS, SfdRowCfg<NX>::MINB)
sfd_rows_kernel(const StreamFdArgs a, const int n_arg) {
    const int n = n_arg >= 0 ? n_arg : *a.iter;
    using Cfg = SfdRowCfg<NX>;
    constexpr int E = Cfg::E, T = Cfg::T, G = Cfg::G;
    __shared__ float2 sm[G * Cfg::SM_PER_GROUP];
    __shared__ float2 tws[FftCfg<NX>::TW];
    __shared__ float red[G][6];

    const int pair = blockIdx.y, s0 = 2 * pair, s1 = s0 + 1;
    const bool act0 = n < a.stop_iter[s0];
    const bool act1 = (s1 < a.batch) && (n < a.stop_iter[s1]);
    if (!act0 && !act1) return;
    const bool last = (n + 1 == a.max_iters);
    const bool want_gap = last || (a.tol > 0.f && ((n + 1) % a.check_every) == 0);

    TwiddlesSmem<NX>::fill(tws, a.tw_row, threadIdx.x, Cfg::THREADS);
    const int g = threadIdx.x / T, j = threadIdx.x % T;
    const int y = blockIdx.x * G + g;
    const int ny = a.ny;
    float2 *smg = sm + g * Cfg::SM_PER_GROUP;
    TwiddlesSmem<NX> tw;
    tw.w = tws + j;
    const long long po = ((long long)pair * ny + y) * NX;
    const int rd = n & 1, wr = rd ^ 1;
    float2 *zr = a.Z + po;
    const float2 *qxr = a.qx2[rd] + po, *qyr = a.qy2[rd] + po, *M = a.M2 + po;
    float2 *qxw = a.qx2[wr] + po, *qyw = a.qy2[wr] + po, *chiw = a.chi3[(n + 1) % 3] + po;
    const float2 *chn = a.chi3[n % 3] + po, *chp = a.chi3[(n + 2) % 3] + po;   // chi_n, chi_{n-1}
    const bool has_up = y > 0, has_down = y < ny - 1;

    float2 v[E];
#pragma unroll
    for (int m = 0; m < E; ++m) v[m] = __ldcs(zr + j + T * m);
    {   // own row of chi_n, chi_{n-1}, qx, qy (and M): one 128-byte line per 16 elements; the rows above and below are
        // the neighbouring groups' own rows
        constexpr int LINES = NX / 16;
        for (int l = j; l < LINES; l += T) {
            prefetch_l2(chn + 16 * l); prefetch_l2(chp + 16 * l); prefetch_l2(qxr + 16 * l); prefetch_l2(qyr + 16 * l);
            if (MASKED) prefetch_l2(M + 16 * l);
        }
    }
    __syncthreads();   // twiddle table
    fft_line<NX, Cfg::LD>(v, smg, j, tw, WarpSync());
    // STAGE: park K p in the group's exchange region during the update loop, so that the registers hold loads in
    // flight instead of the spectrum (each thread reads back only what it wrote)
    constexpr bool STAGE = Cfg::STAGE;
    if (STAGE) {
        __syncwarp();   // the second FFT stage of the other threads has read the region
#pragma unroll
        for (int m = 0; m < E; ++m) smg[j + T * m] = v[m];
    }

    const float2 sig2 = splat(a.sigma), zero = make_float2(0.f, 0.f);
    const float2 alpha = make_float2(a.alpha * a.cscale[s0], (s1 < a.batch) ? a.alpha * a.cscale[s1] : 0.f);
    const float2 alpha_sq = mul2(alpha, alpha);
    constexpr bool aniso = ANISO;   // a template parameter: as a run-time flag both projections were computed and selected
    const float2 ntau2 = splat(-a.tau), ntau_v = make_float2(-a.tau, a.tau), theta2 = splat(a.theta);
    const float2 actm = make_float2(act0 ? 1.f : 0.f, act1 ? 1.f : 0.f);
    float2 gap = zero, dn = zero, cn = zero, mqx_prev = zero;
    // chibar_n = chi_n + theta (chi_n - chi_{n-1}), the same operations that produced it in iteration n-1 (PAPER.md:49 line 4)
    auto cbar_at = [&](const int off, float2 &chi_n) {
        chi_n = __ldg(chn + off);
        return fma2(theta2, sub2(chi_n, __ldg(chp + off)), chi_n);
    };
    float2 tmp, con;                                           // con: chi_n[y][x] of the next element
    float2 c0n = cbar_at(j, con), cun = has_up ? cbar_at(j - NX, tmp) : zero;
    // with the spectrum parked nothing in the loop is indexed by m at compile time: unroll by UNR only (the fully
    // unrolled 512-point kernel was 120 KB of straight-line code, far beyond the instruction cache)
    constexpr int UNR = STAGE ? Cfg::UNROLL : E;
#pragma unroll UNR
    for (int m = 0; m < E; ++m) {
        const int x = j + T * m;
        const float2 c0 = c0n, cu = cun, c_old = con;          // chibar_n[y][x], chibar_n[y-1][x], chi_n[y][x]
        if (m + 1 < E) { c0n = cbar_at(x + T, con); cun = has_up ? cbar_at(x + T - NX, tmp) : zero; }
        const float2 cd = has_down ? cbar_at(x + NX, tmp) : c0; // Neumann: no row below -> gy = 0
        // right neighbours [.][x+1]: lane j+1 (same m), or lane 0's element m+1 when j == T-1
        const float2 give0 = (j == 0 && m + 1 < E) ? c0n : c0;
        const float2 giveu = (j == 0 && m + 1 < E) ? cun : cu;
        float2 cr = shfl2(give0, (j + 1) & (T - 1), T);
        float2 cur = shfl2(giveu, (j + 1) & (T - 1), T);
        if (m == E - 1 && j == T - 1) { cr = c0; cur = cu; }   // Neumann: no column to the right -> gx = 0
        const float2 mm = MASKED ? __ldg(M + x) : make_float2(1.f, 1.f);
        // own row: q_{n+1}[y][x]
        const float2 gx = MASKED ? mul2(mm, sub2(cr, c0)) : sub2(cr, c0);
        const float2 gy = MASKED ? mul2(mm, sub2(cd, c0)) : sub2(cd, c0);
        float2 tx = fma2(sig2, gx, __ldg(qxr + x));
        float2 ty = fma2(sig2, gy, __ldg(qyr + x));
        sfd_project(tx, ty, alpha, alpha_sq, aniso);
        __stcs(qxw + x, tx);
        __stcs(qyw + x, ty);
        if (want_gap) {   // alpha |g| - <g, q_{n+1}>
            float2 gn;
            if (aniso) {
                gn = make_float2(fabsf(gx.x) + fabsf(gy.x), fabsf(gx.y) + fabsf(gy.y));
            } else {
                const float2 g2 = fma2(gy, gy, mul2(gx, gx));
                gn = make_float2(gap_sqrt<kStreamingFastProj>(g2.x), gap_sqrt<kStreamingFastProj>(g2.y));
            }
            gap = add2(gap, sub2(mul2(alpha, gn), fma2(gy, ty, mul2(gx, tx))));
        }
        // row above, redundantly: (M qy_{n+1})[y-1][x]
        float2 mqy_up = zero;
        if (has_up) {
            const float2 mu = MASKED ? __ldg(M - NX + x) : make_float2(1.f, 1.f);
            float2 ux = fma2(sig2, MASKED ? mul2(mu, sub2(cur, cu)) : sub2(cur, cu), __ldg(qxr - NX + x));
            float2 uy = fma2(sig2, MASKED ? mul2(mu, sub2(c0, cu)) : sub2(c0, cu), __ldg(qyr - NX + x));
            sfd_project(ux, uy, alpha, alpha_sq, aniso);
            mqy_up = MASKED ? mul2(mu, uy) : uy;
        }
        // d = G^T (M q) = -div(M q): qx is 0 in the last column and qy in the last row, so no predicate
        const float2 mqx = MASKED ? mul2(mm, tx) : tx;
        const float2 give = (j == T - 1 && m > 0) ? mqx_prev : mqx;
        float2 left = shfl2(give, (j + T - 1) & (T - 1), T);   // (M qx)[y][x-1]
        if (m == 0 && j == 0) left = zero;
        const float2 d = add2(sub2(left, mqx), sub2(mqy_up, MASKED ? mul2(mm, ty) : ty));
        mqx_prev = mqx;
        // chi_{n+1}, chibar_{n+1}; a lane whose slice has stopped keeps its chi
        const float2 step = fma2(ntau2, d, mul2(ntau_v, STAGE ? smg[x] : v[m]));
        const float2 c_new = fma2(actm, step, c_old);
        const float2 dc = sub2(c_new, c_old);
        dn = fma2(dc, dc, dn);
        cn = fma2(c_new, c_new, cn);
        const float2 cbar = fma2(theta2, dc, c_new);
        __stcs(chiw + x, c_new);
        if (STAGE) smg[x] = cbar; else v[m] = cbar;
    }
    if (!last) {   // the stop decision of this iteration is taken by the next column kernel
        if (STAGE) {
#pragma unroll
            for (int m = 0; m < E; ++m) v[m] = smg[j + T * m];
        }
        fft_line<NX, Cfg::LD>(v, smg, j, tw, WarpSync());
#pragma unroll
        for (int m = 0; m < E; ++m) __stcs(zr + j + T * m, v[m]);
    }

    // per-CTA partial sums, fixed order
    float s6[6] = {gap.x, gap.y, dn.x, cn.x, dn.y, cn.y};
#pragma unroll
    for (int k = 0; k < 6; ++k) s6[k] = group_sum<T>(s6[k]);
    if (j == 0) {
#pragma unroll
        for (int k = 0; k < 6; ++k) red[g][k] = s6[k];
    }
    __syncthreads();
    if (threadIdx.x < 6) {
        const int k = threadIdx.x;
        float t = 0.f;
        for (int q = 0; q < G; ++q) t += red[q][k];
        const long long part = (long long)pair * a.nrowparts + blockIdx.x;
        if (k < 2) { if (want_gap) a.gap_row[part * 2 + k] = t; }
        else if ((k < 4) ? act0 : act1) a.res_part[part * 4 + (k - 2)] = t;
    }
}

// ------------------------------------------------------------------------------------------------ row kernel, l1 on chi
// soft shrinkage of both lanes: sign(v) max(|v| - t, 0), the prox of t |.| (BASELINE.json north_star "or shrinkage")
__device__ __forceinline__ float2 shrink2(const float2 v, const float2 t) {
    return make_float2(copysignf(fmaxf(fabsf(v.x) - t.x, 0.f), v.x), copysignf(fmaxf(fabsf(v.y) - t.y, 0.f), v.y));
}

// PD_REG_L1: min 1/2||W(K chi - phi)||^2 + alpha ||M chi||_1 (north_star's alternative regulariser).
// No q: the row kernel of iteration n is
//   v = K p_{n+1}: row FFT of Z gives (v_a, -v_b) ; chi_{n+1} = shrink(chi_n - tau v, tau alpha M) ;
//   chibar_{n+1} = chi_{n+1} + theta (chi_{n+1} - chi_n) ; Z <- row FFT of chibar_{n+1}
// on the same planes and with the same column kernels / dual row kernel as the TV iteration (the q planes stay unused).
template <int NX, bool MASKED>
__global__ void __launch_bounds__(SfdRowCfg<NX>::THREADS, 4)
sfd_rows_l1_kernel(const StreamFdArgs a, const int n_arg) {
    const int n = n_arg >= 0 ? n_arg : *a.iter;
    using Cfg = SfdRowCfg<NX>;
    constexpr int E = Cfg::E, T = Cfg::T, G = Cfg::G;
    __shared__ float2 sm[G * Cfg::SM_PER_GROUP];
    __shared__ float2 tws[FftCfg<NX>::TW];
    __shared__ float red[G][4];

    const int pair = blockIdx.y, s0 = 2 * pair, s1 = s0 + 1;
    const bool act0 = n < a.stop_iter[s0];
    const bool act1 = (s1 < a.batch) && (n < a.stop_iter[s1]);
    if (!act0 && !act1) return;
    const bool last = (n + 1 == a.max_iters);
    const bool want_gap = last || (a.tol > 0.f && ((n + 1) % a.check_every) == 0);

    TwiddlesSmem<NX>::fill(tws, a.tw_row, threadIdx.x, Cfg::THREADS);
    const int g = threadIdx.x / T, j = threadIdx.x % T;
    const int y = blockIdx.x * G + g;
    float2 *smg = sm + g * Cfg::SM_PER_GROUP;
    TwiddlesSmem<NX> tw;
    tw.w = tws + j;
    const long long po = ((long long)pair * a.ny + y) * NX;
    float2 *zr = a.Z + po, *chiw = a.chi3[(n + 1) % 3] + po;
    const float2 *chn = a.chi3[n % 3] + po, *M = a.M2 + po;

    float2 v[E];
#pragma unroll
    for (int m = 0; m < E; ++m) v[m] = __ldcs(zr + j + T * m);
    __syncthreads();   // twiddle table
    fft_line<NX, Cfg::LD>(v, smg, j, tw, WarpSync());
    __syncwarp();      // the second FFT stage of the other threads has read the region
#pragma unroll
    for (int m = 0; m < E; ++m) smg[j + T * m] = v[m];

    const float2 ntau_v = make_float2(-a.tau, a.tau), theta2 = splat(a.theta);
    // threshold tau alpha per lane, in the lane's own normalisation (pair_scale)
    const float2 thr0 = make_float2(a.tau * a.alpha * a.cscale[s0], (s1 < a.batch) ? a.tau * a.alpha * a.cscale[s1] : 0.f);
    float2 dn = make_float2(0.f, 0.f), cn = dn;
#pragma unroll
    for (int m = 0; m < E; ++m) {
        const int x = j + T * m;
        const float2 c_old = __ldg(chn + x);
        const float2 thr = MASKED ? mul2(thr0, __ldg(M + x)) : thr0;
        const float2 sh = shrink2(fma2(ntau_v, smg[x], c_old), thr);
        const float2 c_new = make_float2(act0 ? sh.x : c_old.x, act1 ? sh.y : c_old.y);   // a stopped slice keeps its chi
        const float2 dc = sub2(c_new, c_old);
        dn = fma2(dc, dc, dn);
        cn = fma2(c_new, c_new, cn);
        __stcs(chiw + x, c_new);
        smg[x] = fma2(theta2, dc, c_new);
    }
    if (!last) {
#pragma unroll
        for (int m = 0; m < E; ++m) v[m] = smg[j + T * m];
        fft_line<NX, Cfg::LD>(v, smg, j, tw, WarpSync());
#pragma unroll
        for (int m = 0; m < E; ++m) __stcs(zr + j + T * m, v[m]);
    }
    float s4[4] = {dn.x, cn.x, dn.y, cn.y};
#pragma unroll
    for (int k = 0; k < 4; ++k) s4[k] = group_sum<T>(s4[k]);
    if (j == 0) {
#pragma unroll
        for (int k = 0; k < 4; ++k) red[g][k] = s4[k];
    }
    __syncthreads();
    if (threadIdx.x < 4) {
        const int k = threadIdx.x;
        float t = 0.f;
        for (int q = 0; q < G; ++q) t += red[q][k];
        const long long part = (long long)pair * a.nrowparts + blockIdx.x;
        if ((k < 2) ? act0 : act1) a.res_part[part * 4 + k] = t;
        if (want_gap && k < 2) a.gap_row[part * 2 + k] = 0.f;   // the gap has no regulariser term here (R9)
    }
}

// ------------------------------------------------------------------------------------------------ dual rows (literal path)
// W != I (or PD_OPT_FOURIER_DUAL = 0): p lives in the image domain, K is applied twice per iteration (PAPER.md:49
// literally).  Iteration n:  [sfd_cols<PLAIN>]  this kernel  [sfd_cols<PLAIN>]  sfd_rows.
//   u = K chibar_n: row FFT of Z gives (u_a, -u_b) (zero in iteration 0)
//   p_{n+1} = (p_n + sigma W (u - phi)) / (1 + sigma)                      [PAPER.md:49 line 1; R2, R3]
//   Z <- row FFT of W p_{n+1}        ;        data term of the gap 1/2 ||W(u - phi) - p_{n+1}||^2 per CTA
// Same structure as sfd_rows: read-only double-buffered p, spectrum parked in the exchange region.
template <int NX>
__global__ void __launch_bounds__(SfdRowCfg<NX>::THREADS, 4)
sfd_dual_rows_kernel(const StreamFdArgs a, const int n_arg) {
    const int n = n_arg >= 0 ? n_arg : *a.iter;
    using Cfg = SfdRowCfg<NX>;
    constexpr int E = Cfg::E, T = Cfg::T, G = Cfg::G;
    __shared__ float2 sm[G * Cfg::SM_PER_GROUP];
    __shared__ float2 tws[FftCfg<NX>::TW];
    __shared__ float red[G][2];

    const int pair = blockIdx.y, s0 = 2 * pair, s1 = s0 + 1;
    const bool act0 = n < a.stop_iter[s0];
    const bool act1 = (s1 < a.batch) && (n < a.stop_iter[s1]);
    if (!act0 && !act1) return;
    const bool last = (n + 1 == a.max_iters);
    const bool want_gap = last || (a.tol > 0.f && ((n + 1) % a.check_every) == 0);

    TwiddlesSmem<NX>::fill(tws, a.tw_row, threadIdx.x, Cfg::THREADS);
    const int g = threadIdx.x / T, j = threadIdx.x % T;
    const int y = blockIdx.x * G + g;
    float2 *smg = sm + g * Cfg::SM_PER_GROUP;
    TwiddlesSmem<NX> tw;
    tw.w = tws + j;
    const long long po = ((long long)pair * a.ny + y) * NX;
    float2 *zr = a.Z + po, *pw = a.phat[(n & 1) ^ 1] + po;
    const float2 *pr = a.phat[n & 1] + po, *phi = a.phihat + po, *W = a.W2 + po;

    float2 v[E];
    if (n > 0) {
#pragma unroll
        for (int m = 0; m < E; ++m) v[m] = __ldcs(zr + j + T * m);
    } else {
#pragma unroll
        for (int m = 0; m < E; ++m) v[m] = make_float2(0.f, 0.f);
    }
    __syncthreads();   // twiddle table
    if (n > 0) fft_line<NX, Cfg::LD>(v, smg, j, tw, WarpSync());
    __syncwarp();      // the second FFT stage of the other threads has read the region
#pragma unroll
    for (int m = 0; m < E; ++m) smg[j + T * m] = v[m];

    const float2 sig2 = splat(a.sigma), inv2 = splat(a.inv_one_plus_sigma), half2 = splat(0.5f);
    const float2 sgn = make_float2(1.f, -1.f);   // lane y of the transform carries -u_b
    float2 gap = make_float2(0.f, 0.f);
#pragma unroll
    for (int m = 0; m < E; ++m) {
        const int x = j + T * m;
        const float2 w = __ldg(W + x);
        const float2 res = mul2(w, sub2(mul2(sgn, smg[x]), __ldg(phi + x)));
        const float2 pn = mul2(fma2(sig2, res, __ldg(pr + x)), inv2);
        if (want_gap) {
            const float2 e = sub2(res, pn);
            gap = fma2(mul2(e, half2), e, gap);
        }
        __stcs(pw + x, pn);
        smg[x] = mul2(w, pn);
    }
#pragma unroll
    for (int m = 0; m < E; ++m) v[m] = smg[j + T * m];
    fft_line<NX, Cfg::LD>(v, smg, j, tw, WarpSync());
#pragma unroll
    for (int m = 0; m < E; ++m) __stcs(zr + j + T * m, v[m]);

    if (want_gap) {   // per-CTA partial sums, fixed order; read by sfd_gap_sum through gap_col (ncolparts = nrowparts)
        gap.x = group_sum<T>(gap.x);
        gap.y = group_sum<T>(gap.y);
        if (j == 0) { red[g][0] = gap.x; red[g][1] = gap.y; }
        __syncthreads();
        if (threadIdx.x < 2) {
            float t = 0.f;
            for (int q = 0; q < G; ++q) t += red[q][threadIdx.x];
            a.gap_col[n & 1][((long long)pair * a.ncolparts + blockIdx.x) * 2 + threadIdx.x] = t;
        }
    }
}

// ------------------------------------------------------------------------------------------------ loop control
// Last node of the graphed iteration body (one CTA): n <- n + 1, and the WHILE node runs the body again only if the
// count allows it and some slice is still active -- the paper's per-slice "control of the calculation end points"
// extended to the launch sequence itself: once every slice has stopped nothing is launched any more,
// and the host is never asked.  The stop decision of iteration n-1 is taken inside the column kernel of
// iteration n, so the loop runs one (empty) iteration past the last stop.
__global__ void __launch_bounds__(256)
sfd_loop_ctl_kernel(const StreamFdArgs a, const cudaGraphConditionalHandle handle) {
    const int n = *a.iter + 1;
    int active = 0;
    for (int b = threadIdx.x; b < a.batch; b += 256) active |= (n < a.stop_iter[b]);
    active = __syncthreads_or(active);
    if (threadIdx.x == 0) {
        *a.iter = n;
        cudaGraphSetConditional(handle, (n < a.max_iters && active) ? 1u : 0u);
    }
}

// ------------------------------------------------------------------------------------------------ finish
// chi_N of every slice -> the caller's planes (S7); column... block 0 of the pair: relgap of slices that ran to
// max_iters (the others recorded theirs when they stopped), relres, iters_done.
__global__ void __launch_bounds__(256)
sfd_finish_kernel(const StreamFdArgs a) {
    const int pair = blockIdx.y, s0 = 2 * pair, s1 = s0 + 1;
    const bool has_b = s1 < a.batch;
    const long long P = (long long)a.nx * a.ny;
    // the last row kernel that ran for this pair was iteration max(stop) - 1, which wrote buffer max(stop) % 3
    const int st0 = a.stop_iter[s0], st1 = has_b ? a.stop_iter[s1] : 0;
    const float2 *c2 = a.chi3[(st0 > st1 ? st0 : st1) % 3] + (long long)pair * P;
    float *oa = a.chi_out + (long long)s0 * P, *ob = a.chi_out + (long long)s1 * P;
    const float ia = 1.f / a.cscale[s0], ib = has_b ? 1.f / a.cscale[s1] : 0.f;   // back to the caller's units (exact: powers of two)
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < P; i += (long long)gridDim.x * blockDim.x) {
        const float2 c = __ldcs(c2 + i);
        oa[i] = ia * c.x;
        if (has_b) ob[i] = ib * c.y;
    }
    if (blockIdx.x == 0 && threadIdx.x < 2 && (threadIdx.x == 0 || has_b)) {
        const int s = threadIdx.x, b = s ? s1 : s0;
        const int stop = a.stop_iter[b];
        const float P0 = a.P0[b];
        if (stop >= a.max_iters && a.max_iters > 0 && P0 > 0.f) {
            const float2 g = sfd_gap_sum(a, pair, (a.max_iters - 1) & 1);
            a.relgap[b] = (s ? g.y : g.x) / P0;
        }
        float dn = 0.f, cn = 0.f;
        if (stop > 0) {
            const float *rp = a.res_part + (long long)pair * a.nrowparts * 4 + 2 * s;
            for (int k = 0; k < a.nrowparts; ++k) { dn += rp[4 * k]; cn += rp[4 * k + 1]; }
        }
        a.relres[b] = (cn > 0.f) ? sqrtf(dn) / sqrtf(cn) : 0.f;
        a.iters_done[b] = (P0 == 0.f && !(a.tol > 0.f)) ? a.max_iters : min(stop, a.max_iters);
    }
}

}  // namespace pdk
