// pd_streaming.cuh -- streaming variant of the PD iteration for sm_100a.
//
// One iteration = four launches over the whole batch:
//   dual_rows   : finish K1 = F^-1 D F chibar_n (inverse row pass), p-update, q-update, gap sums,
//                 forward row pass of W p_{n+1}                              (PAPER.md:49 lines 1-2)
//   dipole_cols : forward column FFT, multiply by D, inverse column FFT
//   primal_rows : finish K2 = F^-1 D F (W p_{n+1}), G^T M q_{n+1}, chi-update, over-relaxation,
//                 residual sums, forward row pass of chibar_{n+1}            (PAPER.md:49 lines 3-4)
//   dipole_cols : same kernel, for the next K1.
//
// Two slices share one complex transform: z = slice_{2j} + i*slice_{2j+1}.  D is real and even, so
// F^-1 D F z = K(slice_{2j}) + i*K(slice_{2j+1}) exactly.
// Spectra live in Z[pair][ny][nx] (float2).  Between the column kernel and the next row kernel the data is
// kept in the "swapped" convention of the forward-only FFT (fft_regs.cuh): after the row pass the real part
// of the result sits in .y and the imaginary part in .x.
#pragma once
#include "fft_regs.cuh"

namespace pdk {

struct SolveArgs {
    // geometry
    int nx, ny, batch, npairs;
    // inputs (device)
    const float *field;   // phi
    const float *mask;    // M or nullptr
    const float *weight;  // W or nullptr
    long long mask_bstride;  // 0 when one mask is shared by all slices
    // state (device)
    float *chi;      // = chi_out
    float *chibar;
    float *p, *qx, *qy;
    float2 *Z;       // [npairs][ny][nx]
    const float *Dtab;          // D / (nx*ny), [ny][nx]
    const float2 *tw_row, *tw_col;  // exp(-2 pi i n / nx), exp(-2 pi i n / ny)
    // per-slice state variables
    int *stop_iter;       // slice b is active in iteration n (0-based) iff n < stop_iter[b]
    float *P0;            // 1/2 ||W phi||^2
    float *relgap, *relres;
    float *gap_part;      // [batch][nparts]
    float *res_part;      // [batch][nparts][2]  (||chi+ - chi||^2, ||chi+||^2)
    int nparts;           // row-kernel CTAs per pair
    // parameters
    float alpha, sigma, tau, theta, inv_one_plus_sigma, tol;
    int aniso, check_every, max_iters;
};

template <int T>
__device__ __forceinline__ float group_sum(float v) {
#pragma unroll
    for (int o = T / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Row kernels: G lines per CTA, one line (pair j, row y) per group of T threads inside one warp.
template <int NX> struct RowCfg {
    static constexpr int E = FftCfg<NX>::E, T = FftCfg<NX>::T;
    static constexpr int THREADS = 128;
    static constexpr int G = THREADS / T;      // rows per CTA
    static constexpr int LD = T + 1;           // padded exchange rows: conflict-free 64-bit accesses
    static constexpr int SM_PER_GROUP = E * LD;
};

// ------------------------------------------------------------------------------------------------ dual step
template <int NX>
__global__ void __launch_bounds__(RowCfg<NX>::THREADS)
dual_rows_kernel(const SolveArgs a, const int n_iter) {
    using Cfg = RowCfg<NX>;
    constexpr int E = Cfg::E, T = Cfg::T, G = Cfg::G;
    __shared__ float2 sm[G * Cfg::SM_PER_GROUP];
    __shared__ float red[G][2];

    const int pair = blockIdx.y;
    const int s0 = 2 * pair, s1 = s0 + 1;
    const bool act0 = n_iter < a.stop_iter[s0];
    const bool act1 = (s1 < a.batch) && (n_iter < a.stop_iter[s1]);
    if (!act0 && !act1) return;

    const int g = threadIdx.x / T, j = threadIdx.x % T;
    const int y = blockIdx.x * G + g;
    float2 *smg = sm + g * Cfg::SM_PER_GROUP;
    Twiddles<NX> tw;
    tw.load(a.tw_row, j);

    const long long P = (long long)a.nx * a.ny;
    const long long rowoff = (long long)y * NX;

    // ---- u = K chibar_n : inverse row pass (data arrives column-transformed and swapped)
    float2 v[E];
    {
        const float2 *zr = a.Z + (long long)pair * P + rowoff;
#pragma unroll
        for (int m = 0; m < E; ++m) v[m] = zr[j + T * m];
    }
    fft_line<NX, Cfg::LD>(v, smg, j, tw, WarpSync());
    // now: u(slice s0) = v.y, u(slice s1) = v.x at x = j + T*m

    float gap[2] = {0.f, 0.f};
    float2 out[E];
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        const bool act = s ? act1 : act0;
        const int b = s ? s1 : s0;
        const long long base = (long long)b * P + rowoff;
        if (act) {
            const float *phi = a.field + base;
            float *pp = a.p + base;
            const float *wt = a.weight ? a.weight + base : nullptr;
            const float *mk = a.mask ? a.mask + (long long)b * a.mask_bstride + rowoff : nullptr;
            const float *cb = a.chibar + base;
            float *qxp = a.qx + base, *qyp = a.qy + base;
            const bool has_down = y < a.ny - 1;
            // p_{n+1} = (p_n + sigma*W(K chibar_n - phi)) / (1 + sigma)            [PAPER.md:49 line 1, R2/R3]
            float c0[E], cd[E];
#pragma unroll
            for (int m = 0; m < E; ++m) {
                const int x = j + T * m;
                c0[m] = cb[x];
                cd[m] = has_down ? cb[x + NX] : 0.f;
            }
#pragma unroll
            for (int m = 0; m < E; ++m) {
                const int x = j + T * m;
                const float u = s ? v[m].x : v[m].y;
                const float w = wt ? wt[x] : 1.f;
                const float r = w * (u - phi[x]);
                const float pn = (pp[x] + a.sigma * r) * a.inv_one_plus_sigma;
                const float e = r - pn;
                gap[s] = fmaf(0.5f * e, e, gap[s]);
                pp[x] = pn;
                if (s) out[m].y = w * pn; else out[m].x = w * pn;
            }
            // q_{n+1} = proj_alpha(q_n + sigma*M G chibar_n)                           [PAPER.md:49 line 2, R4/R7]
#pragma unroll
            for (int m = 0; m < E; ++m) {
                const int x = j + T * m;
                // right neighbour chibar[y][x+1]: lane j+1 (same m), or lane 0 at m+1 when j == T-1
                const float give = (j == 0 && m + 1 < E) ? c0[(m + 1 < E) ? m + 1 : m] : c0[m];
                const float cr = __shfl_sync(0xffffffffu, give, (j + 1) & (T - 1), T);
                const float mm = mk ? mk[x] : 1.f;
                const float gx = (x < NX - 1) ? mm * (cr - c0[m]) : 0.f;
                const float gy = has_down ? mm * (cd[m] - c0[m]) : 0.f;
                float tx = fmaf(a.sigma, gx, qxp[x]);
                float ty = fmaf(a.sigma, gy, qyp[x]);
                float gn;
                if (a.aniso) {
                    tx = fminf(fmaxf(tx, -a.alpha), a.alpha);
                    ty = fminf(fmaxf(ty, -a.alpha), a.alpha);
                    gn = fabsf(gx) + fabsf(gy);
                } else {
                    const float nrm = sqrtf(tx * tx + ty * ty);
                    const float sc = (nrm > a.alpha) ? a.alpha / nrm : 1.f;
                    tx *= sc;
                    ty *= sc;
                    gn = sqrtf(gx * gx + gy * gy);
                }
                qxp[x] = tx;
                qyp[x] = ty;
                gap[s] += a.alpha * gn - gx * tx - gy * ty;
            }
        } else {
#pragma unroll
            for (int m = 0; m < E; ++m) { if (s) out[m].y = 0.f; else out[m].x = 0.f; }
        }
    }

    // ---- forward row pass of z = W p(s0) + i W p(s1) for K2
    fft_line<NX, Cfg::LD>(out, smg, j, tw, WarpSync());
    {
        float2 *zr = a.Z + (long long)pair * P + rowoff;
#pragma unroll
        for (int m = 0; m < E; ++m) zr[j + T * m] = out[m];
    }

    // ---- per-CTA gap partial sums, fixed order (deterministic stopping)
    gap[0] = group_sum<T>(gap[0]);
    gap[1] = group_sum<T>(gap[1]);
    if (j == 0) { red[g][0] = gap[0]; red[g][1] = gap[1]; }
    __syncthreads();
    if (threadIdx.x < 2) {
        const int s = threadIdx.x;
        const int b = s ? s1 : s0;
        if (s ? act1 : act0) {
            float acc = 0.f;
            for (int k = 0; k < G; ++k) acc += red[k][s];
            a.gap_part[(long long)b * a.nparts + blockIdx.x] = acc;
        }
    }
}

// ------------------------------------------------------------------------------------------------ primal step
template <int NX>
__global__ void __launch_bounds__(RowCfg<NX>::THREADS)
primal_rows_kernel(const SolveArgs a, const int n_iter) {
    using Cfg = RowCfg<NX>;
    constexpr int E = Cfg::E, T = Cfg::T, G = Cfg::G;
    __shared__ float2 sm[G * Cfg::SM_PER_GROUP];
    __shared__ float red[G][4];

    const int pair = blockIdx.y;
    const int s0 = 2 * pair, s1 = s0 + 1;
    const bool act0 = n_iter < a.stop_iter[s0];
    const bool act1 = (s1 < a.batch) && (n_iter < a.stop_iter[s1]);
    if (!act0 && !act1) return;

    const int g = threadIdx.x / T, j = threadIdx.x % T;
    const int y = blockIdx.x * G + g;
    float2 *smg = sm + g * Cfg::SM_PER_GROUP;
    Twiddles<NX> tw;
    tw.load(a.tw_row, j);

    const long long P = (long long)a.nx * a.ny;
    const long long rowoff = (long long)y * NX;

    // ---- v = K (W p_{n+1}) : inverse row pass
    float2 v[E];
    {
        const float2 *zr = a.Z + (long long)pair * P + rowoff;
#pragma unroll
        for (int m = 0; m < E; ++m) v[m] = zr[j + T * m];
    }
    fft_line<NX, Cfg::LD>(v, smg, j, tw, WarpSync());

    float acc[2][2] = {{0.f, 0.f}, {0.f, 0.f}};
    float2 out[E];
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        const bool act = s ? act1 : act0;
        const int b = s ? s1 : s0;
        const long long base = (long long)b * P + rowoff;
        if (act) {
            const float *mk = a.mask ? a.mask + (long long)b * a.mask_bstride + rowoff : nullptr;
            const float *qxp = a.qx + base, *qyp = a.qy + base;
            float *chip = a.chi + base, *cbp = a.chibar + base;
            const bool has_up = y > 0, has_down = y < a.ny - 1;
            float mqx[E];
#pragma unroll
            for (int m = 0; m < E; ++m) {
                const int x = j + T * m;
                mqx[m] = (mk ? mk[x] : 1.f) * qxp[x];
            }
#pragma unroll
            for (int m = 0; m < E; ++m) {
                const int x = j + T * m;
                // left neighbour (M qx)[y][x-1]: lane j-1 (same m), or lane T-1 at m-1 when j == 0
                const float give = (j == T - 1 && m > 0) ? mqx[m > 0 ? m - 1 : 0] : mqx[m];
                const float left = __shfl_sync(0xffffffffu, give, (j + T - 1) & (T - 1), T);
                const float mm = mk ? mk[x] : 1.f;
                const float mqy = mm * qyp[x];
                const float mqy_up = has_up ? (mk ? mk[x - NX] : 1.f) * qyp[x - NX] : 0.f;
                // d = G^T (M q) = -div(M q)                                           [PAPER.md:49 line 3, R7]
                float d = 0.f;
                if (x > 0) d += left;
                if (x < NX - 1) d -= mqx[m];
                if (has_up) d += mqy_up;
                if (has_down) d -= mqy;
                const float kv = s ? v[m].x : v[m].y;
                const float c_old = chip[x];
                // chi_{n+1} = chi_n - tau*K(W p_{n+1}) - tau*G^T M q_{n+1}
                const float c_new = fmaf(-a.tau, d, fmaf(-a.tau, kv, c_old));
                const float dc = c_new - c_old;
                acc[s][0] = fmaf(dc, dc, acc[s][0]);
                acc[s][1] = fmaf(c_new, c_new, acc[s][1]);
                // chibar_{n+1} = chi_{n+1} + theta*(chi_{n+1} - chi_n)               [PAPER.md:49 line 4]
                const float cbar = fmaf(a.theta, dc, c_new);
                chip[x] = c_new;
                cbp[x] = cbar;
                if (s) out[m].y = cbar; else out[m].x = cbar;
            }
        } else {
#pragma unroll
            for (int m = 0; m < E; ++m) { if (s) out[m].y = 0.f; else out[m].x = 0.f; }
        }
    }

    // ---- forward row pass of z = chibar(s0) + i chibar(s1) for the next K1
    fft_line<NX, Cfg::LD>(out, smg, j, tw, WarpSync());
    {
        float2 *zr = a.Z + (long long)pair * P + rowoff;
#pragma unroll
        for (int m = 0; m < E; ++m) zr[j + T * m] = out[m];
    }

#pragma unroll
    for (int s = 0; s < 2; ++s)
#pragma unroll
        for (int q = 0; q < 2; ++q) acc[s][q] = group_sum<T>(acc[s][q]);
    if (j == 0) { red[g][0] = acc[0][0]; red[g][1] = acc[0][1]; red[g][2] = acc[1][0]; red[g][3] = acc[1][1]; }
    __syncthreads();
    if (threadIdx.x < 4) {
        const int s = threadIdx.x >> 1, q = threadIdx.x & 1;
        const int b = s ? s1 : s0;
        if (s ? act1 : act0) {
            float t = 0.f;
            for (int k = 0; k < G; ++k) t += red[k][threadIdx.x];
            a.res_part[((long long)b * a.nparts + blockIdx.x) * 2 + q] = t;
        }
    }
}

// ------------------------------------------------------------------------------------------------ column pass
// CTA = 16 adjacent columns x T threads each.  Forward column FFT, * D/(nx*ny), swap (=inverse), forward column FFT.
// After the first dual step of an iteration (finalize_gap != 0) the CTA of column block 0 also reduces the gap
// partials of its pair in fixed order and raises the per-slice stop flag on the device.
template <int NY> struct ColCfg {
    static constexpr int E = FftCfg<NY>::E, T = FftCfg<NY>::T;
    static constexpr int COLS = 16;
    static constexpr int THREADS = COLS * T;
    static constexpr int CS = NY + 1;  // odd column stride (float2): conflict-free across the 16 columns of a half-warp
    static constexpr int SMEM_BYTES = COLS * CS * (int)sizeof(float2);
};

template <int NY>
__global__ void __launch_bounds__(ColCfg<NY>::THREADS)
dipole_cols_kernel(const SolveArgs a, const int n_iter, const int finalize_gap) {
    using Cfg = ColCfg<NY>;
    constexpr int E = Cfg::E, T = Cfg::T;
    extern __shared__ float2 smc[];

    const int pair = blockIdx.y;
    const int s0 = 2 * pair, s1 = s0 + 1;
    const bool act0 = n_iter < a.stop_iter[s0];
    const bool act1 = (s1 < a.batch) && (n_iter < a.stop_iter[s1]);
    if (!act0 && !act1) return;

    const int c = threadIdx.x & (Cfg::COLS - 1), j = threadIdx.x / Cfg::COLS;
    const int kx = blockIdx.x * Cfg::COLS + c;
    const int nx = a.nx;
    Twiddles<NY> tw;
    tw.load(a.tw_col, j);
    float2 *zc = a.Z + (long long)pair * nx * NY + kx;
    float2 *smg = smc + c * Cfg::CS;

    float2 v[E];
#pragma unroll
    for (int m = 0; m < E; ++m) v[m] = zc[(long long)(j + T * m) * nx];
    fft_line<NY, T>(v, smg, j, tw, BlockSync());
    const float *dcol = a.Dtab + kx;
#pragma unroll
    for (int m = 0; m < E; ++m) {
        const float d = __ldg(dcol + (long long)(j + T * m) * nx);
        v[m] = make_float2(v[m].y * d, v[m].x * d);  // multiply by D and swap re/im: next forward FFT acts as the inverse
    }
    fft_line<NY, T>(v, smg, j, tw, BlockSync());
#pragma unroll
    for (int m = 0; m < E; ++m) zc[(long long)(j + T * m) * nx] = v[m];

    if (finalize_gap && blockIdx.x == 0 && threadIdx.x < 2) {
        const int s = threadIdx.x;
        const int b = s ? s1 : s0;
        if (s ? act1 : act0) {
            float t = 0.f;
            for (int k = 0; k < a.nparts; ++k) t += a.gap_part[(long long)b * a.nparts + k];
            const float P0 = a.P0[b];
            const float rg = P0 > 0.f ? t / P0 : 0.f;
            a.relgap[b] = rg;
            if (a.tol > 0.f && ((n_iter + 1) % a.check_every) == 0 && rg < a.tol) a.stop_iter[b] = n_iter + 1;
        }
    }
}

// ------------------------------------------------------------------------------------------------ init / finish
// One CTA per slice: P0 = 1/2 ||W phi||^2 (fixed-order reduction), reset of the per-slice state variables.
__global__ void __launch_bounds__(256)
init_slices_kernel(const SolveArgs a) {
    __shared__ float red[256];
    const int b = blockIdx.x;
    const long long P = (long long)a.nx * a.ny;
    const float *phi = a.field + (long long)b * P;
    const float *wt = a.weight ? a.weight + (long long)b * P : nullptr;
    float acc = 0.f;
    for (long long i = threadIdx.x; i < P; i += 256) {
        const float t = (wt ? wt[i] : 1.f) * phi[i];
        acc = fmaf(t, t, acc);
    }
    red[threadIdx.x] = acc;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const float P0 = 0.5f * red[0];
        a.P0[b] = P0;
        a.relgap[b] = 0.f;
        a.relres[b] = 0.f;
        // reading R13b: for an all-zero slice every iteration is a no-op (chi stays 0); it is never scheduled, so that
        // rounding cross-talk from its pair partner cannot leak into it.  finish_slices_kernel reports its count.
        a.stop_iter[b] = (P0 == 0.f) ? 0 : a.max_iters;
    }
    for (int k = threadIdx.x; k < a.nparts; k += 256) {
        a.gap_part[(long long)b * a.nparts + k] = 0.f;
        a.res_part[((long long)b * a.nparts + k) * 2 + 0] = 0.f;
        a.res_part[((long long)b * a.nparts + k) * 2 + 1] = 0.f;
    }
}

__global__ void finish_slices_kernel(const SolveArgs a, int *iters_done) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= a.batch) return;
    float dn = 0.f, cn = 0.f;
    for (int k = 0; k < a.nparts; ++k) {
        dn += a.res_part[((long long)b * a.nparts + k) * 2 + 0];
        cn += a.res_part[((long long)b * a.nparts + k) * 2 + 1];
    }
    int it = min(a.stop_iter[b], a.max_iters);
    if (a.P0[b] == 0.f && !(a.tol > 0.f)) it = a.max_iters;  // R13b: "runs N no-op iterations" when no tolerance is set
    iters_done[b] = it;
    a.relres[b] = (cn > 0.f) ? sqrtf(dn) / sqrtf(cn) : 0.f;
}

}  // namespace pdk
