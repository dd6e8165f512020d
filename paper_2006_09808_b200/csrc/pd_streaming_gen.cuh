// pd_streaming_gen.cuh -- streaming variant for slice sizes that are NOT powers of two: the paper's own matrices are
// 256 x 258 and 128 x 132.  Any even nx, ny in [4, 1024] is accepted.
//
// The iteration is the literal one of PAPER.md:49 (p in the image domain, K = F^-1 D F applied twice per iteration), on
// the pair-interleaved float2 planes and with the launch sequence of the literal path of pd_streaming_fd.cuh:
//   gen_cols (K1; carries the stop decision of the previous iteration)   [not in iteration 0: chibar_0 = 0]
//   gen_dual_rows : u = K chibar_n (finish) ; p_{n+1} = (p_n + sigma W (u - phi))/(1 + sigma) ; start K (W p_{n+1})
//   gen_cols (K2)
//   gen_rows      : v = K W p_{n+1} (finish) ; q-update ; chi-update ; over-relaxation ; start K chibar_{n+1}
// sfd_scale / sfd_finish / sfd_loop_ctl and the graphed loop are shared with the power-of-two path.
//
// Line transform: a length-N DFT, N = N1 * N2 (the most balanced factorisation, chosen by pd_plan: 258 = 6 x 43,
// 132 = 11 x 12), as two DENSE stages in shared memory (Cooley-Tukey with arbitrary factors):
//   Y[n1][k2] = W_N^(n1 k2) sum_n2 x[n1 + N1 n2] W_N2^(n2 k2)          N * N2 complex multiply-adds
//   X[k2 + N2 k1] = sum_n1 Y[n1][k2] W_N1^(n1 k1)                       N * N1
// from the plan's double-precision table W_N^e.  One warp per line, no register arrays, every index a run-time value:
// about five times the arithmetic of a radix-2 line of the same length -- written for generality, not for the roofline
// (the tuned kernels of pd_streaming_fd.cuh stay the path of every power-of-two size).
#pragma once
#include "pd_streaming_fd.cuh"

namespace pdk {

constexpr int kGenRows = 4;      // rows per CTA of the row kernels
constexpr int kGenWPR = 2;       // warps per row in the row kernels: the paper's stacks are small (13 and 21 slice pairs), one warp
                                 // per row left the GPU at 22 warps per SM; the two warps of a row meet at a named barrier
constexpr int kGenLT = 32 * kGenWPR;
constexpr int kGenColsB = 8;     // adjacent columns per CTA of the column kernel (64-byte segments)

struct GenDims { int n1x, n2x, n1y, n2y; };   // nx = n1x * n2x, ny = n1y * n2y

// The twiddle table W_N^e sits in shared memory with one padding slot after every 16 entries: the lanes of a warp read
// W[(lane-dependent multiple of a stride) mod N], and strides that are multiples of 8 or 16 entries (N2 = 16: every
// access; N = 258: every eighth n2) would otherwise land in one or two banks (measured: 20 cycles per warp instruction).
__host__ __device__ constexpr int gen_wsize(int n) { return n + (n >> 4) + 1; }
__device__ __forceinline__ int gen_wp(const int e) { return e + (e >> 4); }

// sum_k x[k * xs] W[(k * step) mod N], k = 0..cnt-1, with eight independent accumulation chains (two elements per trip,
// every product its own chain): the loop is bound by the latency of dependent FMAs and shared-memory loads, not by their count
__device__ __forceinline__ float2 gen_dot(const float2 *W, const int N, const float2 *x, const int xs, const int cnt, const int step) {
    float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f, b0 = 0.f, b1 = 0.f, b2 = 0.f, b3 = 0.f;
    int e = 0, k = 0;
    for (; k + 1 < cnt; k += 2) {
        int e1 = e + step;
        if (e1 >= N) e1 -= N;
        const float2 x0 = x[k * xs], w0 = W[gen_wp(e)], x1 = x[(k + 1) * xs], w1 = W[gen_wp(e1)];
        e = e1 + step;
        if (e >= N) e -= N;
        a0 = fmaf(x0.x, w0.x, a0); a1 = fmaf(-x0.y, w0.y, a1); a2 = fmaf(x0.x, w0.y, a2); a3 = fmaf(x0.y, w0.x, a3);
        b0 = fmaf(x1.x, w1.x, b0); b1 = fmaf(-x1.y, w1.y, b1); b2 = fmaf(x1.x, w1.y, b2); b3 = fmaf(x1.y, w1.x, b3);
    }
    if (k < cnt) {
        const float2 x0 = x[k * xs], w0 = W[gen_wp(e)];
        a0 = fmaf(x0.x, w0.x, a0); a1 = fmaf(-x0.y, w0.y, a1); a2 = fmaf(x0.x, w0.y, a2); a3 = fmaf(x0.y, w0.x, a3);
    }
    return make_float2((a0 + b0) + (a1 + b1), (a2 + b2) + (a3 + b3));
}

// Forward DFT of one line by LT cooperating threads (one or two warps).  W: padded table W_N^e (shared memory).
// src -> tmp -> dst; src and dst may be the same buffer.  sync() synchronises the LT threads; the call ends with one.
template <int LT, class Sync>
__device__ __forceinline__ void gen_line_dft(const float2 *W, const int N, const int N1, const int N2, const float2 *src,
                                             float2 *tmp, float2 *dst, const int lane, const Sync sync) {
    for (int o = lane; o < N; o += LT) {
        const int n1 = o / N2, k2 = o - n1 * N2;
        // Y[n1][k2] = W_N^(n1 k2) sum_n2 x[n1 + N1 n2] W_N2^(n2 k2),  W_N2^(n2 k2) = W_N^(n2 k2 N1)
        tmp[o] = cmul(gen_dot(W, N, src + n1, N1, N2, k2 * N1), W[gen_wp(n1 * k2)]);
    }
    sync();
    for (int o = lane; o < N; o += LT) {
        const int k1 = o / N2, k2 = o - k1 * N2;
        // X[k2 + N2 k1] = sum_n1 Y[n1][k2] W_N1^(n1 k1),  W_N1^(n1 k1) = W_N^(n1 k1 N2)
        dst[k2 + N2 * k1] = gen_dot(W, N, tmp + k2, N2, N1, k1 * N2);
    }
    sync();
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// ------------------------------------------------------------------------------------------------ init
// Interleave phi (normalised, pair_scale), W and M; zero p_0, chi_0, chi_{-1}, q_0; partial sums of
// 1/2 ||W phi||^2 per (pair, row block).  One warp per row.
__global__ void __launch_bounds__(32 * kGenRows)
gen_init_kernel(const StreamFdArgs a) {
    __shared__ float red[kGenRows][2];
    const int pair = blockIdx.y, s0 = 2 * pair, s1 = s0 + 1;
    const bool has_b = s1 < a.batch;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int y = blockIdx.x * kGenRows + warp, nx = a.nx;
    const long long P = (long long)nx * a.ny;
    float acc0 = 0.f, acc1 = 0.f;
    if (y < a.ny) {
        const long long rowoff = (long long)y * nx, po = (long long)pair * P + rowoff;
        const float ca = a.cscale[s0], cb = has_b ? a.cscale[s1] : 0.f;
        const float2 zero = make_float2(0.f, 0.f);
        for (int x = lane; x < nx; x += 32) {
            const float va = ca * a.field[(long long)s0 * P + rowoff + x];
            const float vb = has_b ? cb * a.field[(long long)s1 * P + rowoff + x] : 0.f;
            float wa = 1.f, wb = has_b ? 1.f : 0.f;
            if (a.weight) { wa = a.weight[(long long)s0 * P + rowoff + x]; wb = has_b ? a.weight[(long long)s1 * P + rowoff + x] : 0.f; }
            a.phihat[po + x] = make_float2(va, vb);
            a.W2[po + x] = make_float2(wa, wb);
            float ma = 1.f, mb = 1.f;
            if (a.mask) { ma = a.mask[s0 * a.mask_bstride + rowoff + x]; mb = has_b ? a.mask[s1 * a.mask_bstride + rowoff + x] : 0.f; }
            a.M2[po + x] = make_float2(ma, mb);
            a.phat[0][po + x] = zero; a.chi3[0][po + x] = zero; a.chi3[2][po + x] = zero;
            a.qx2[0][po + x] = zero; a.qy2[0][po + x] = zero; a.Z[po + x] = zero;
            acc0 = fmaf(wa * va, wa * va, acc0);
            acc1 = fmaf(wb * vb, wb * vb, acc1);
        }
    }
    acc0 = warp_sum(acc0);
    acc1 = warp_sum(acc1);
    if (lane == 0) { red[warp][0] = acc0; red[warp][1] = acc1; }
    __syncthreads();
    if (threadIdx.x < 2) {
        float t = 0.f;
        for (int k = 0; k < kGenRows; ++k) t += red[k][threadIdx.x];
        a.p0_part[((long long)pair * a.nrowparts + blockIdx.x) * 2 + threadIdx.x] = t;
    }
}

// P0 of every slice and its per-slice state (one thread per slice)
__global__ void __launch_bounds__(128)
gen_init_finish_kernel(const StreamFdArgs a) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < a.batch) {
        float t = 0.f;
        const float *pp = a.p0_part + (long long)(b >> 1) * a.nrowparts * 2 + (b & 1);
        for (int k = 0; k < a.nrowparts; ++k) t += pp[2 * k];
        const float P0 = 0.5f * t;
        a.P0[b] = P0;
        a.relgap[b] = 0.f;
        a.relres[b] = 0.f;
        a.stop_iter[b] = (P0 == 0.f) ? 0 : a.max_iters;   // R13b: an all-zero slice is never scheduled
    }
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < (long long)a.npairs * a.nrowparts * 4;
         k += (long long)gridDim.x * blockDim.x)
        a.res_part[k] = 0.f;
}

// ------------------------------------------------------------------------------------------------ column kernel
// Z <- column DFT of conj(D/(nx ny) * column DFT of Z): one application of K between two row passes (the row kernels'
// transforms finish it).  kGenColsB adjacent columns per CTA, one warp per column at a time.  With do_decide: the stop
// decision of iteration n-1 first (as sfd_cols_kernel: every CTA reduces the same partial sums in the same order).
__global__ void __launch_bounds__(32 * kGenColsB)
gen_cols_kernel(const StreamFdArgs a, const GenDims gd, const int n_arg, const int do_decide) {
    const int n = n_arg >= 0 ? n_arg : *a.iter;
    if (do_decide && n == 0) return;   // chibar_0 = 0: the first K application of iteration 0 is skipped
    extern __shared__ __align__(16) unsigned char gen_smem[];
    const int nx = a.nx, ny = a.ny;
    float2 *W = reinterpret_cast<float2 *>(gen_smem);          // [gen_wsize(ny)], padded (gen_wp)
    float2 *buf = W + gen_wsize(ny);                           // [kGenColsB][2][ny]
    __shared__ float dec[2];

    const int pair = blockIdx.y, s0 = 2 * pair, s1 = s0 + 1;
    const bool has_b = s1 < a.batch;
    int stop0 = a.stop_iter[s0], stop1 = has_b ? a.stop_iter[s1] : 0;
    if (n >= stop0 && n >= stop1) return;
    const bool decide = do_decide && n > 0 && a.tol > 0.f && (n % a.check_every) == 0;
    if (decide) {
        if (threadIdx.x == 0) {
            const float2 g = sfd_gap_sum(a, pair, (n - 1) & 1);
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
        __syncthreads();
        if (dec[0] != 0.f) stop0 = n;
        if (dec[1] != 0.f) stop1 = n;
        if (n >= stop0 && n >= stop1) return;
    }
    for (int i = threadIdx.x; i < ny; i += blockDim.x) W[gen_wp(i)] = __ldg(a.tw_col + i);
    const int x0 = blockIdx.x * kGenColsB;
    const int ncols = nx - x0 < kGenColsB ? nx - x0 : kGenColsB;
    float2 *zb = a.Z + (long long)pair * nx * ny + x0;
    // tile [ny][ncols] -> column-major lines: consecutive threads read consecutive columns of one row
    for (int i = threadIdx.x; i < ny * kGenColsB; i += blockDim.x) {
        const int y = i / kGenColsB, c = i - y * kGenColsB;
        if (c < ncols) buf[(c * 2) * ny + y] = __ldcs(zb + (long long)y * nx + c);
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (warp < ncols) {
        float2 *l0 = buf + (warp * 2) * ny, *l1 = l0 + ny;
        gen_line_dft<32>(W, ny, gd.n1y, gd.n2y, l0, l1, l0, lane, WarpSync());
        const float *dcol = a.Dtab + x0 + warp;
        for (int y = lane; y < ny; y += 32) {
            const float d = __ldg(dcol + (long long)y * nx);
            const float2 v = l0[y];
            l0[y] = make_float2(d * v.x, -d * v.y);   // conj(D z^): the next forward transform is the conjugate of the inverse
        }
        __syncwarp();
        gen_line_dft<32>(W, ny, gd.n1y, gd.n2y, l0, l1, l0, lane, WarpSync());
    }
    __syncthreads();
    for (int i = threadIdx.x; i < ny * kGenColsB; i += blockDim.x) {
        const int y = i / kGenColsB, c = i - y * kGenColsB;
        if (c < ncols) __stcs(zb + (long long)y * nx + c, buf[(c * 2) * ny + y]);
    }
}

// ------------------------------------------------------------------------------------------------ dual rows
// u = K chibar_n: the row DFT of Z gives (u_a, -u_b) (zero in iteration 0) ; p_{n+1} = (p_n + sigma W (u - phi))/(1 + sigma)
// [PAPER.md:49 line 1; R2, R3] ; Z <- row DFT of W p_{n+1} ; data term of the gap 1/2 ||W(u - phi) - p_{n+1}||^2.
__global__ void __launch_bounds__(kGenLT * kGenRows)
gen_dual_rows_kernel(const StreamFdArgs a, const GenDims gd, const int n_arg) {
    const int n = n_arg >= 0 ? n_arg : *a.iter;
    extern __shared__ __align__(16) unsigned char gen_smem[];
    const int nx = a.nx;
    float2 *W = reinterpret_cast<float2 *>(gen_smem);          // [gen_wsize(nx)], padded (gen_wp)
    __shared__ float red[kGenRows * kGenWPR][2];
    const int pair = blockIdx.y, s0 = 2 * pair, s1 = s0 + 1;
    const bool act0 = n < a.stop_iter[s0];
    const bool act1 = (s1 < a.batch) && (n < a.stop_iter[s1]);
    if (!act0 && !act1) return;
    const bool last = (n + 1 == a.max_iters);
    const bool want_gap = last || (a.tol > 0.f && ((n + 1) % a.check_every) == 0);
    for (int i = threadIdx.x; i < nx; i += blockDim.x) W[gen_wp(i)] = __ldg(a.tw_row + i);
    __syncthreads();
    const int warp = threadIdx.x >> 5, grp = threadIdx.x / kGenLT, lane = threadIdx.x % kGenLT;   // grp: the row of this thread
    const int y = blockIdx.x * kGenRows + grp;
    float2 *l0 = W + gen_wsize(nx) + (grp * 2) * nx, *l1 = l0 + nx;
    const NamedSync rowsync{1 + grp, kGenLT};
    float2 gap = make_float2(0.f, 0.f);
    if (y < a.ny) {
        const long long po = ((long long)pair * a.ny + y) * nx;
        float2 *zr = a.Z + po, *pw = a.phat[(n & 1) ^ 1] + po;
        const float2 *pr = a.phat[n & 1] + po, *phi = a.phihat + po, *W2 = a.W2 + po;
        if (n > 0) {
            for (int x = lane; x < nx; x += kGenLT) l0[x] = __ldcs(zr + x);
            rowsync();
            gen_line_dft<kGenLT>(W, nx, gd.n1x, gd.n2x, l0, l1, l0, lane, rowsync);
        } else {
            for (int x = lane; x < nx; x += kGenLT) l0[x] = make_float2(0.f, 0.f);
        }
        const float2 sig2 = splat(a.sigma), inv2 = splat(a.inv_one_plus_sigma), half2 = splat(0.5f);
        const float2 sgn = make_float2(1.f, -1.f);   // lane y of the transform carries -u_b
        for (int x = lane; x < nx; x += kGenLT) {
            const float2 w = __ldg(W2 + x);
            const float2 res = mul2(w, sub2(mul2(sgn, l0[x]), __ldg(phi + x)));
            const float2 pn = mul2(fma2(sig2, res, __ldg(pr + x)), inv2);
            if (want_gap) {
                const float2 e = sub2(res, pn);
                gap = fma2(mul2(e, half2), e, gap);
            }
            __stcs(pw + x, pn);
            l0[x] = mul2(w, pn);
        }
        rowsync();
        gen_line_dft<kGenLT>(W, nx, gd.n1x, gd.n2x, l0, l1, l0, lane, rowsync);
        for (int x = lane; x < nx; x += kGenLT) __stcs(zr + x, l0[x]);
    }
    if (want_gap) {   // per-CTA partial sums, fixed order; read by sfd_gap_sum through gap_col (ncolparts = nrowparts)
        gap.x = warp_sum(gap.x);
        gap.y = warp_sum(gap.y);
        if ((lane & 31) == 0) { red[warp][0] = gap.x; red[warp][1] = gap.y; }
        __syncthreads();
        if (threadIdx.x < 2) {
            float t = 0.f;
            for (int q = 0; q < kGenRows * kGenWPR; ++q) t += red[q][threadIdx.x];
            a.gap_col[n & 1][((long long)pair * a.ncolparts + blockIdx.x) * 2 + threadIdx.x] = t;
        }
    }
}

// ------------------------------------------------------------------------------------------------ primal rows
// v = K W p_{n+1}: the row DFT of Z gives (v_a, -v_b).  Then, per pixel of the row (PAPER.md:49 lines 2-4):
//   q_{n+1} = proj_alpha(q_n + sigma M G chibar_n) for the own row and, redundantly, its qy for the row above
//   d = G^T (M q_{n+1}) ; chi_{n+1} = chi_n - tau (v + d) ; chibar_{n+1} = chi_{n+1} + theta (chi_{n+1} - chi_n)
// or, with the l1 regulariser, chi_{n+1} = shrink(chi_n - tau v, tau alpha M).  chibar_n is recomputed from chi_n and
// chi_{n-1} wherever it is needed (as in sfd_rows_kernel); neighbours are plain (cached) loads.  Z <- row DFT of chibar_{n+1}.
__global__ void __launch_bounds__(kGenLT * kGenRows)
gen_rows_kernel(const StreamFdArgs a, const GenDims gd, const int n_arg) {
    const int n = n_arg >= 0 ? n_arg : *a.iter;
    extern __shared__ __align__(16) unsigned char gen_smem[];
    const int nx = a.nx, ny = a.ny;
    float2 *W = reinterpret_cast<float2 *>(gen_smem);          // [gen_wsize(nx)], padded (gen_wp)
    __shared__ float red[kGenRows * kGenWPR][6];
    const int pair = blockIdx.y, s0 = 2 * pair, s1 = s0 + 1;
    const bool act0 = n < a.stop_iter[s0];
    const bool act1 = (s1 < a.batch) && (n < a.stop_iter[s1]);
    if (!act0 && !act1) return;
    const bool last = (n + 1 == a.max_iters);
    const bool want_gap = last || (a.tol > 0.f && ((n + 1) % a.check_every) == 0);
    for (int i = threadIdx.x; i < nx; i += blockDim.x) W[gen_wp(i)] = __ldg(a.tw_row + i);
    __syncthreads();
    const int warp = threadIdx.x >> 5, grp = threadIdx.x / kGenLT, lane = threadIdx.x % kGenLT;   // grp: the row of this thread
    const int y = blockIdx.x * kGenRows + grp;
    float2 *l0 = W + gen_wsize(nx) + (grp * 2) * nx, *l1 = l0 + nx;
    const NamedSync rowsync{1 + grp, kGenLT};
    const float2 zero = make_float2(0.f, 0.f);
    float2 gap = zero, dn = zero, cn = zero;
    if (y < ny) {
        const long long po = ((long long)pair * ny + y) * nx;
        const int rd = n & 1, wr = rd ^ 1;
        float2 *zr = a.Z + po;
        const float2 *qxr = a.qx2[rd] + po, *qyr = a.qy2[rd] + po, *M = a.M2 + po;
        float2 *qxw = a.qx2[wr] + po, *qyw = a.qy2[wr] + po, *chiw = a.chi3[(n + 1) % 3] + po;
        const float2 *chn = a.chi3[n % 3] + po, *chp = a.chi3[(n + 2) % 3] + po;   // chi_n, chi_{n-1}
        const bool has_up = y > 0, has_down = y < ny - 1;
        for (int x = lane; x < nx; x += kGenLT) l0[x] = __ldcs(zr + x);
        rowsync();
        gen_line_dft<kGenLT>(W, nx, gd.n1x, gd.n2x, l0, l1, l0, lane, rowsync);

        const float2 sig2 = splat(a.sigma), theta2 = splat(a.theta);
        const float2 alpha = make_float2(a.alpha * a.cscale[s0], (s1 < a.batch) ? a.alpha * a.cscale[s1] : 0.f);
        const float2 alpha_sq = mul2(alpha, alpha), thr0 = mul2(splat(a.tau), alpha);
        const bool aniso = a.aniso != 0;
        const float2 ntau2 = splat(-a.tau), ntau_v = make_float2(-a.tau, a.tau);
        const float2 actm = make_float2(act0 ? 1.f : 0.f, act1 ? 1.f : 0.f);
        // chibar_n = chi_n + theta (chi_n - chi_{n-1}), the operations that produced it in iteration n-1 (PAPER.md:49 line 4)
        auto cbar_at = [&](const int off) {
            const float2 c = __ldg(chn + off);
            return fma2(theta2, sub2(c, __ldg(chp + off)), c);
        };
        for (int x = lane; x < nx; x += kGenLT) {
            const float2 c_old = __ldg(chn + x), mm = __ldg(M + x);
            float2 c_new;
            if (a.reg_l1) {
                const float2 sh = shrink2(fma2(ntau_v, l0[x], c_old), mul2(thr0, mm));
                c_new = make_float2(act0 ? sh.x : c_old.x, act1 ? sh.y : c_old.y);
            } else {
                const bool has_right = x < nx - 1;
                const float2 c0 = cbar_at(x);
                const float2 cr = has_right ? cbar_at(x + 1) : c0;        // Neumann: gx = 0 in the last column
                const float2 cd = has_down ? cbar_at(x + nx) : c0;       // Neumann: gy = 0 in the last row
                const float2 gx = mul2(mm, sub2(cr, c0)), gy = mul2(mm, sub2(cd, c0));
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
                // (M qx_{n+1})[y][x-1] and (M qy_{n+1})[y-1][x], recomputed from read-only data
                float2 mqx_left = zero, mqy_up = zero;
                if (x > 0) {
                    const float2 ml = __ldg(M + x - 1), cl = cbar_at(x - 1);
                    const float2 cld = has_down ? cbar_at(x - 1 + nx) : cl;
                    float2 lx = fma2(sig2, mul2(ml, sub2(c0, cl)), __ldg(qxr + x - 1));
                    float2 ly = fma2(sig2, mul2(ml, sub2(cld, cl)), __ldg(qyr + x - 1));
                    sfd_project(lx, ly, alpha, alpha_sq, aniso);
                    mqx_left = mul2(ml, lx);
                }
                if (has_up) {
                    const float2 mu = __ldg(M - nx + x), cu = cbar_at(x - nx);
                    const float2 cur = has_right ? cbar_at(x - nx + 1) : cu;
                    float2 ux = fma2(sig2, mul2(mu, sub2(cur, cu)), __ldg(qxr - nx + x));
                    float2 uy = fma2(sig2, mul2(mu, sub2(c0, cu)), __ldg(qyr - nx + x));
                    sfd_project(ux, uy, alpha, alpha_sq, aniso);
                    mqy_up = mul2(mu, uy);
                }
                // d = G^T (M q) = -div(M q): qx is 0 in the last column and qy in the last row, so no predicate
                const float2 d = add2(sub2(mqx_left, mul2(mm, tx)), sub2(mqy_up, mul2(mm, ty)));
                const float2 step = fma2(ntau2, d, mul2(ntau_v, l0[x]));
                c_new = fma2(actm, step, c_old);   // a lane whose slice has stopped keeps its chi
            }
            const float2 dc = sub2(c_new, c_old);
            dn = fma2(dc, dc, dn);
            cn = fma2(c_new, c_new, cn);
            __stcs(chiw + x, c_new);
            l0[x] = fma2(theta2, dc, c_new);
        }
        if (!last) {
            rowsync();
            gen_line_dft<kGenLT>(W, nx, gd.n1x, gd.n2x, l0, l1, l0, lane, rowsync);
            for (int x = lane; x < nx; x += kGenLT) __stcs(zr + x, l0[x]);
        }
    }
    float s6[6] = {gap.x, gap.y, dn.x, cn.x, dn.y, cn.y};
#pragma unroll
    for (int k = 0; k < 6; ++k) s6[k] = warp_sum(s6[k]);
    if ((lane & 31) == 0) {
#pragma unroll
        for (int k = 0; k < 6; ++k) red[warp][k] = s6[k];
    }
    __syncthreads();
    if (threadIdx.x < 6) {
        const int k = threadIdx.x;
        float t = 0.f;
        for (int q = 0; q < kGenRows * kGenWPR; ++q) t += red[q][k];
        const long long part = (long long)pair * a.nrowparts + blockIdx.x;
        if (k < 2) { if (want_gap) a.gap_row[part * 2 + k] = t; }
        else if ((k < 4) ? act0 : act1) a.res_part[part * 4 + (k - 2)] = t;
    }
}

}  // namespace pdk
