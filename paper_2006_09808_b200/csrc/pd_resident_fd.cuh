// pd_resident_fd.cuh -- resident variant with the dual variable p kept in the FOURIER domain (W = identity).
//
// With W = I the p-update of PAPER.md:49 line 1 is linear and pointwise, so it commutes with the FFT:
//     p^_{n+1} = (p^_n + sigma (D X^_n - phi^)) / (1 + sigma),   X^_n = F chibar_n,   phi^ = F phi,
// and K p_{n+1} = F^-1 (D p^_{n+1}).  One iteration then needs ONE forward 2-D FFT (of chibar_n) and ONE inverse
// (of D p^_{n+1}) instead of two round trips: 4 FFT passes, 2 transposes and 2 cluster barriers per iteration instead
// of 8 / 4 / 4 (pd_resident.cuh, which stays the path for W != I).  The iterates chi_n are the same up to rounding
// order.
//
// The data term of the gap (R9), 1/2 ||r - p_{n+1}||^2 = ||p_{n+1} - p_n||^2 / (2 sigma^2), is taken in the
// Fourier domain by Parseval.  Two slices share one complex transform z = a + i b, so the per-slice sums need
//     sum_x a^2 = 1/2 (sum |z|^2 + Re sum z^2),  sum_x b^2 = 1/2 (sum |z|^2 - Re sum z^2),
//     sum_x z^2 = N^-2 sum_k Z(k) Z(-k):
// every CTA therefore owns its columns in MIRROR PAIRS (kx, N - kx), so that Z(-k) is in its own shared memory.
//
// Layout in time, per pair and iteration n (phases separated by ONE cluster barrier each):
//   column phase n : X^_n = column FFT of Z ; p^ update ; Z <- column FFT of conj(D/N^2 p^_{n+1})
//   q-update n     : q_{n+1} = proj_alpha(q_n + sigma M G chibar_n)                       (PAPER.md:49 line 2)
//   -- cluster barrier, stop decision (same in every CTA) --
//   row phase n    : v = conj(row FFT of Z) = K p_{n+1} ; chi_{n+1} = chi_n - tau (v + G^T M q_{n+1}) ;
//                    chibar_{n+1} ; Z <- row FFT of chibar_{n+1}                          (PAPER.md:49 lines 3-4)
//   -- cluster barrier --
#pragma once
#include "pd_resident.cuh"

namespace pdk {

struct ResidentFdArgs {
    int batch, npairs, max_iters, check_every;
    float alpha, sigma, tau, theta, inv_one_plus_sigma, tol;
    const float *field, *mask;
    long long mask_bstride;
    float *chi_out;
    float2 *Z, *qy, *chi, *chibar, *M2, *phihat;  // per-cluster scratch, each [nclusters][N*N]
    const float *Dpriv;    // D/(N*N) in the column phase's thread-private order: [C][E][NT]
    const float2 *tw_tab;  // exp(-2 pi i n / N)
    float *part;           // [nclusters][C][8] per-CTA partial sums
    int *iters_done;
    float *relgap, *relres;
};
constexpr int kResidentFdScratchArrays = 6;

// Column kx owned by (cluster rank, column group cgi in {0,1}, slot cc in 0..15): the low half [16 rank, 16 rank + 16)
// and its mirror images N - kx; the two self-mirrored columns 0 and N/2 both sit in rank 0, slot 0.
// The host builds Dpriv with the same function (pd_api.cu).
__host__ __device__ constexpr int fd_column_of(int N, int rank, int cgi, int cc) {
    const int lo = 16 * rank + cc;
    return cgi == 0 ? lo : (lo == 0 ? N / 2 : N - lo);
}

// ------------------------------------------------------------------------------------------------ column phase
// Thread (column kx, slot j) holds ky = j + T m.  zc = &Z[kx]; dpriv / phh / ph_s already offset by the thread id.
//   X^ = column FFT of Z (zero when `first`: chibar_0 = 0)
//   p^_{n+1} = (p^_n + sigma (D X^ - phi^)) / (1 + sigma)                 [PAPER.md:49 line 1 in the Fourier domain]
//   Z <- column FFT of conj(D/N^2 p^_{n+1})   (= conjugate of the inverse transform, finished by the row phase)
// With want_gap: S1 += sum |dp|^2, S2 += Re sum dp(k) dp(-k), dp = p^_{n+1} - p^_n (mirror column in smg_mirror).
template <int N, int NT, class Tw>
__device__ __forceinline__ void dual_fd_col(float2 *zc, const float *__restrict__ dpriv, const float2 *phh,
                                            float2 *ph_s, const int j, float2 *smg, const float2 *smg_mirror,
                                            const Tw &tw, const ResidentFdArgs &a, const bool first,
                                            const bool want_gap, float &S1, float &S2,
                                            const float2 (&pht)[FftCfg<N>::E]) {
    constexpr int E = FftCfg<N>::E, T = FftCfg<N>::T;
    float2 v[E];
    float dv[E];
#pragma unroll
    for (int m = 0; m < E; ++m) dv[m] = __ldg(dpriv + m * NT);
    if (!first) {
#pragma unroll
        for (int m = 0; m < E; ++m) v[m] = ldcg2(zc + (j + T * m) * N);
        fft_line<N, T>(v, smg, j, tw, BlockSync());
    } else {
#pragma unroll
        for (int m = 0; m < E; ++m) v[m] = make_float2(0.f, 0.f);
    }
    const float2 sig2 = splat(a.sigma), inv2 = splat(a.inv_one_plus_sigma);
    constexpr float NN = (float)N * (float)N;
    if (want_gap) __syncthreads();   // the exchange region is free (readers of the FFT above are done)
#pragma unroll
    for (int m = 0; m < E; ++m) {
        const float d = dv[m];
        const float2 phat = pht[m];   // phi^, loaded by the caller while it waited at the cluster barrier
        const float2 pold = ph_s[m * NT];
        const float2 res = sub2(mul2(splat(d * NN), v[m]), phat);
        const float2 pn = mul2(fma2(sig2, res, pold), inv2);
        if (want_gap) {
            const float2 dp = sub2(pn, pold);
            S1 = fmaf(dp.x, dp.x, fmaf(dp.y, dp.y, S1));
            smg[j + T * m] = dp;
        }
        ph_s[m * NT] = pn;
        v[m] = make_float2(d * pn.x, -d * pn.y);
    }
    if (want_gap) {
        __syncthreads();
#pragma unroll
        for (int m = 0; m < E; ++m) {
            const int ky = j + T * m;
            const float2 dp = smg[ky];
            const float2 dm = smg_mirror[(N - ky) & (N - 1)];
            S2 = fmaf(dp.x, dm.x, fmaf(-dp.y, dm.y, S2));
        }
    }
    fft_line<N, T>(v, smg, j, tw, BlockSync());
#pragma unroll
    for (int m = 0; m < E; ++m) zc[(j + T * m) * N] = v[m];
}

// ------------------------------------------------------------------------------------------------ row phase
// v = K p_{n+1}: the row FFT of Z gives conj(v_a + i v_b) = (v_a, -v_b).
// chi_{n+1} = chi_n - tau v - tau d ; chibar_{n+1} = chi_{n+1} + theta (chi_{n+1} - chi_n) ; Z <- row FFT of chibar_{n+1}.
template <int N, int NT, int LDR, class Tw>
__device__ __forceinline__ void primal_fd_row(const RowPtrs &r, const ResidentFdArgs &a, const int j, float2 *smg,
                                              const Tw &tw, const float2 (&d)[FftCfg<N>::E], float *out_a,
                                              float *out_b, float2 &dn, float2 &cn, const bool need_next) {
    constexpr int E = FftCfg<N>::E, T = FftCfg<N>::T;
    float2 v[E];
#pragma unroll
    for (int m = 0; m < E; ++m) v[m] = ldcg2(r.Z + j + T * m);
    fft_line<N, LDR>(v, smg, j, tw, WarpSync());
    const float2 ntau2 = splat(-a.tau), ntau_v = make_float2(-a.tau, a.tau), theta2 = splat(a.theta);
    constexpr int CH = 8;   // chi is loaded a chunk ahead of the stores (see q_update_row)
    float2 cov[CH];
#pragma unroll
    for (int m = 0; m < E; ++m) {
        const int x = j + T * m;
        if (m % CH == 0) {
#pragma unroll
            for (int k = 0; k < CH; ++k) cov[k] = ldcg2(r.chi + x + T * k);
        }
        const float2 c_old = cov[m % CH];
        const float2 c_new = fma2(ntau2, d[m], fma2(ntau_v, v[m], c_old));
        const float2 dc = sub2(c_new, c_old);
        dn = fma2(dc, dc, dn);
        cn = fma2(c_new, c_new, cn);
        const float2 cbar = fma2(theta2, dc, c_new);
        r.chi[x] = c_new;
        r.chibar[x] = cbar;
        v[m] = cbar;
        if (out_a) out_a[x] = c_new.x;
        if (out_b) out_b[x] = c_new.y;
    }
    if (need_next) {
        fft_line<N, LDR>(v, smg, j, tw, WarpSync());
#pragma unroll
        for (int m = 0; m < E; ++m) r.Z[j + T * m] = v[m];
    }
}

// ------------------------------------------------------------------------------------------------ the kernel
template <int N, int C, int NT, int MINB, bool ANISO>
__global__ void __launch_bounds__(NT, MINB)
resident_fd_kernel(const ResidentFdArgs a) {
    using Cfg = ResCfg<N, C, NT>;
    constexpr int E = Cfg::E, T = Cfg::T, RPC = Cfg::RPC, P = N * N;
    static_assert(RPC == 32 && Cfg::NCG == 2 && Cfg::COLS == 16, "mirror-pair column ownership needs 2 groups of 16 columns");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *exch = reinterpret_cast<float2 *>(smem_raw);
    float2 *tws = exch + Cfg::EXCH;
    float2 *ph_sm = tws + E * T;          // p^ in the column phase's thread-private order
    float2 *qx_sm = ph_sm + Cfg::PRIV;    // qx in the row phase's thread-private order
    float *red = reinterpret_cast<float *>(qx_sm + Cfg::PRIV);
    float *dec = red + Cfg::NWARPS * 8;   // [0..1] P0 ; [2..3] gap ; [4..7] scratch of the gap combination

    const int tid = threadIdx.x;
    const int rank = (C == 1) ? 0 : (int)cluster_ctarank();
    const int cid = (C == 1) ? (int)blockIdx.x : (int)cluster_id_x();
    const int ncl = (C == 1) ? (int)gridDim.x : (int)num_clusters_x();

    TwiddlesSmem<N>::fill(tws, a.tw_tab, tid, NT);
    __syncthreads();

    // row role: group g owns row y ; column role: thread owns column kx, slot cj
    const int g = tid / T, j = tid % T;
    const int row0 = rank * RPC;
    const int y = row0 + g;
    float2 *smg_row = exch + g * (E * Cfg::LDR);
    TwiddlesSmem<N> tw_row;
    tw_row.w = tws + j;
    const int cgi = tid / (Cfg::COLS * T), cc = tid % Cfg::COLS, cj = (tid / Cfg::COLS) % T;
    const int kx = fd_column_of(N, rank, cgi, cc);
    const bool self_mirror = (rank == 0 && cc == 0);   // kx = 0 and kx = N/2
    float2 *smg_col = exch + (cgi * Cfg::COLS + cc) * Cfg::CS;
    const float2 *smg_mir = self_mirror ? smg_col : exch + ((1 - cgi) * Cfg::COLS + cc) * Cfg::CS;
    TwiddlesSmem<N> tw_col;
    tw_col.w = tws + cj;

    const long long soff = (long long)cid * P;
    RowPtrs r;
    r.Z = a.Z + soff + y * N; r.qy = a.qy + soff + y * N; r.chi = a.chi + soff + y * N;
    r.chibar = a.chibar + soff + y * N; r.phi2 = nullptr; r.M2 = a.M2 + soff + y * N; r.W2 = nullptr;
    r.p_s = nullptr; r.qx_s = qx_sm + tid;
    float2 *zcol = a.Z + soff + kx;
    float2 *phh = a.phihat + soff + rank * (RPC * N) + tid;   // [m * NT] per thread
    const float *dpriv = a.Dpriv + rank * (RPC * N) + tid;
    float2 *ph_s = ph_sm + tid;
    float *part = a.part + (long long)cid * C * 8;
    // 1/2 sum_x e^2 = S / (4 N^2 sigma^2) with S = S1 +- S2 (Parseval, header comment)
    const float gap_scale = 0.25f / ((float)N * (float)N * a.sigma * a.sigma);

    // ResidentArgs view for the shared q-update (same fields, same meaning)
    ResidentArgs qa;
    qa.alpha = a.alpha; qa.sigma = a.sigma;

    for (int pair = cid; pair < a.npairs; pair += ncl) {
        const int s0 = 2 * pair, s1 = s0 + 1;
        const bool has_b = s1 < a.batch;
        const float2 zero = make_float2(0.f, 0.f);

        // ---- S7 load: my row of field and mask -> interleaved scratch, zero state, P0 partial sums, row FFT of phi
        {
            const float *fa = a.field + (long long)s0 * P + y * N;
            const float *fb = a.field + (long long)s1 * P + y * N;
            const float *ma = a.mask ? a.mask + s0 * a.mask_bstride + y * N : nullptr;
            const float *mb = a.mask ? a.mask + s1 * a.mask_bstride + y * N : nullptr;
            float acc[2] = {0.f, 0.f};
            float2 v[E];
#pragma unroll
            for (int m = 0; m < E; ++m) {
                const int x = j + T * m;
                const float va = fa[x], vb = has_b ? fb[x] : 0.f;
                v[m] = make_float2(va, vb);
                (a.M2 + soff + y * N)[x] = make_float2(ma ? ma[x] : 1.f, has_b ? (mb ? mb[x] : 1.f) : 0.f);
                r.qy[x] = zero; r.chi[x] = zero; r.chibar[x] = zero;
                acc[0] = fmaf(va, va, acc[0]);
                acc[1] = fmaf(vb, vb, acc[1]);
                ph_s[m * NT] = zero; r.qx_s[m * NT] = zero;
            }
            fft_line<N, Cfg::LDR>(v, smg_row, j, tw_row, WarpSync());
#pragma unroll
            for (int m = 0; m < E; ++m) r.Z[j + T * m] = v[m];
            const float t = block_sum<NT, 2>(acc, red);
            if (tid < 2) part[rank * 8 + tid] = t;
        }
        cluster_sync_all<C>();
        if (tid < 2) {
            float t = 0.f;
            for (int q = 0; q < C; ++q) t += __ldcg(part + q * 8 + tid);
            dec[tid] = 0.5f * t;
        }
        // ---- phi^ = column FFT of the row-transformed field, kept in the column phase's private order
        {
            float2 v[E];
#pragma unroll
            for (int m = 0; m < E; ++m) v[m] = ldcg2(zcol + (cj + T * m) * N);
            fft_line<N, T>(v, smg_col, cj, tw_col, BlockSync());   // its __syncthreads also publish dec[]
#pragma unroll
            for (int m = 0; m < E; ++m) phh[m * NT] = v[m];
        }
        const float P0a = dec[0], P0b = dec[1];
        // R13b: an all-zero slice is never scheduled (every iteration would be a no-op)
        int stop_a = (P0a == 0.f) ? 0 : a.max_iters;
        int stop_b = (!has_b || P0b == 0.f) ? 0 : a.max_iters;
        float gap_a = 0.f, gap_b = 0.f;
        if (stop_a == 0) for (int i = tid; i < RPC * N; i += NT) a.chi_out[(long long)s0 * P + row0 * N + i] = 0.f;
        if (has_b && stop_b == 0) for (int i = tid; i < RPC * N; i += NT) a.chi_out[(long long)s1 * P + row0 * N + i] = 0.f;

        float2 pht[E];
        for (int n = 0; n < a.max_iters; ++n) {
            const bool act_a = n < stop_a, act_b = n < stop_b;
            if (!act_a && !act_b) break;
            const bool last = (n + 1 == a.max_iters);
            const bool check = a.tol > 0.f && ((n + 1) % a.check_every) == 0;
            const bool want_gap = check || last;

            // (1) column phase: p^_{n+1} and the spectrum of K p_{n+1}
            float S1 = 0.f, S2 = 0.f;
            if (n == 0) {
#pragma unroll
                for (int m = 0; m < E; ++m) pht[m] = ldcg2(phh + m * NT);
            }
            dual_fd_col<N, NT>(zcol, dpriv, phh, ph_s, cj, smg_col, smg_mir, tw_col, a, n == 0, want_gap, S1, S2, pht);
            // (2) q-update from chibar_n (chibar_0 = 0 and q_0 = 0: nothing to do in the first iteration)
            float2 gap = zero;
            if (n > 0) q_update_row<N, NT, ANISO>(r, qa, y, j, want_gap, gap);
            if (want_gap) {
                float acc[4] = {S1, S2, gap.x, gap.y};
                const float t = block_sum<NT, 4>(acc, red);
                if (tid < 4) dec[4 + tid] = t;
                __syncthreads();
                if (tid < 2) part[rank * 8 + 2 + tid] = gap_scale * (dec[4] + (tid ? -dec[5] : dec[5])) + dec[6 + tid];
            }
            cluster_sync_all<C>();
            // every CTA reduces the same gap partials in the same order: same stop decision everywhere
            if (want_gap) {
                if (tid < 2) {
                    float t = 0.f;
                    for (int q = 0; q < C; ++q) t += __ldcg(part + q * 8 + 2 + tid);
                    dec[2 + tid] = t;
                }
                __syncthreads();
                if (act_a) { gap_a = dec[2] / P0a; if (check && gap_a < a.tol) stop_a = n + 1; }
                if (act_b) { gap_b = dec[3] / P0b; if (check && gap_b < a.tol) stop_b = n + 1; }
            }
            // (3) row phase: divergence of M q_{n+1}, primal step, over-relaxation, row FFT of chibar_{n+1}
            {
                float2 d[E];
                d_term_row<N, NT>(r, y, j, d);
                float *out_a = (act_a && n + 1 >= stop_a) ? a.chi_out + (long long)s0 * P + y * N : nullptr;
                float *out_b = (act_b && n + 1 >= stop_b) ? a.chi_out + (long long)s1 * P + y * N : nullptr;
                const bool need_next = (n + 1 < a.max_iters) && (n + 1 < stop_a || n + 1 < stop_b);
                float2 dn = zero, cn = zero;
                primal_fd_row<N, NT, Cfg::LDR>(r, a, j, smg_row, tw_row, d, out_a, out_b, dn, cn, need_next);
                if (out_a || out_b) {   // residual of the final iterate (reported, not used for stopping)
                    float acc[4] = {dn.x, cn.x, dn.y, cn.y};
                    const float t = block_sum<NT, 4>(acc, red);
                    if (tid < 4 && ((tid < 2) ? out_a != nullptr : out_b != nullptr)) part[rank * 8 + 4 + tid] = t;
                }
            }
            // the next column phase's thread-private operand phi^ travels while the cluster barrier is waited for
            cluster_arrive<C>();
#pragma unroll
            for (int m = 0; m < E; ++m) pht[m] = ldcg2(phh + m * NT);
            cluster_wait<C>();
        }
        // ---- per-slice state variables
        if (rank == 0 && tid < 2 && (tid == 0 || has_b)) {
            const int b = tid ? s1 : s0;
            const int stop = tid ? stop_b : stop_a;
            const float P0 = tid ? P0b : P0a;
            float dn = 0.f, cn = 0.f;
            if (stop > 0) {
                for (int q = 0; q < C; ++q) {
                    dn += __ldcg(part + q * 8 + 4 + 2 * tid);
                    cn += __ldcg(part + q * 8 + 5 + 2 * tid);
                }
            }
            a.iters_done[b] = (P0 == 0.f && !(a.tol > 0.f)) ? a.max_iters : min(stop, a.max_iters);
            a.relgap[b] = tid ? gap_b : gap_a;
            a.relres[b] = (cn > 0.f) ? sqrtf(dn) / sqrtf(cn) : 0.f;
        }
        cluster_sync_all<C>();   // scratch and partials are reused by the next pair
    }
}

}  // namespace pdk
