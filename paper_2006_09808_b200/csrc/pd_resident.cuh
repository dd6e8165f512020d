// pd_resident.cuh -- resident variant of the PD iteration for square slices <= 256x256.
//
// ONE launch per pd_solve.  A thread-block cluster of C CTAs owns one slice pair for ALL its iterations
// (the paper's "one GPU thread per slice controls the end point", recast as a cluster per pair).
// CTA r of the cluster owns rows [r*N/C, (r+1)*N/C) in the row phases and the same range of columns in the
// column phases; inside the CTA every group of T threads owns ONE row and every thread one column slot, for the
// whole kernel.  The phases of an iteration are separated by hardware cluster barriers instead of kernel
// boundaries, and the work that does not depend on the other CTAs' spectrum (the q-update, the divergence term)
// is placed between the arrive and the wait of those barriers.
//
// Where the state lives: p and qx, which only their owning thread ever touches, stay in shared memory for all
// iterations; chi, chibar, qy, phi, M and the spectrum Z live in a per-CLUSTER scratch that is reused for every
// pair the cluster processes: nclusters * 7 arrays * N*N*8 B (55 MB at 256x256 with 15 clusters), which stays
// resident in the 126 MB L2.  HBM is touched only when a pair is loaded (field, mask) and when chi is stored.
// Per-slice stopping needs no flag exchange: every CTA reduces the same per-CTA partial sums in the same fixed
// order and reaches the same decision; a slice that has stopped keeps iterating in its lane (its results are
// already stored and are not written again).
//
// Arithmetic: two slices share one complex transform (lane x = slice 2j, lane y = slice 2j+1) and all elementwise
// updates run on both lanes at once with Blackwell's packed fp32x2 instructions (FADD2/FMUL2/FFMA2).
// The inverse transform is conj(FFT(conj(.))): the column phase multiplies by (D, -D), so after the next row pass
// lane y carries MINUS its value.  The dual-side arrays (p, phi) are therefore kept with lane y negated; after the
// second K of the iteration the sign is back (K is real), so chi, chibar, q and M are in plain convention.
#pragma once
#include "fft_regs.cuh"

namespace pdk {

struct ResidentArgs {
    int batch, npairs, max_iters, check_every;
    float alpha, sigma, tau, theta, inv_one_plus_sigma, tol;
    const float *field, *mask, *weight;
    long long mask_bstride;
    float *chi_out;
    float2 *Z, *qy, *chi, *chibar, *phi2, *M2, *W2;  // per-cluster scratch, each [nclusters][N*N]
    const float *Dtab;     // D/(N*N), [N][N]
    const float2 *tw_tab;  // exp(-2 pi i n / N)
    float *part;           // [nclusters][C][8] per-CTA partial sums
    int *iters_done;
    float *relgap, *relres;
};
constexpr int kResidentScratchArrays = 7;

__device__ __forceinline__ unsigned cluster_ctarank() {
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ unsigned cluster_id_x() {
    unsigned r;
    asm volatile("mov.u32 %0, %%clusterid.x;" : "=r"(r));
    return r;
}
__device__ __forceinline__ unsigned num_clusters_x() {
    unsigned r;
    asm volatile("mov.u32 %0, %%nclusterid.x;" : "=r"(r));
    return r;
}
// Split cluster barrier: arrive releases this thread's global/shared writes to the cluster, wait acquires the others'.
template <int C>
__device__ __forceinline__ void cluster_arrive() {
    if constexpr (C > 1) asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
}
template <int C>
__device__ __forceinline__ void cluster_wait() {
    if constexpr (C == 1) {
        __syncthreads();
    } else {
        asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
    }
}
template <int C>
__device__ __forceinline__ void cluster_sync_all() {
    cluster_arrive<C>();
    cluster_wait<C>();
}

// packed fp32x2 helpers (sm_100: FADD2 / FMUL2 / FFMA2)
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 sub2(float2 a, float2 b) { return __ffma2_rn(b, make_float2(-1.f, -1.f), a); }
__device__ __forceinline__ float2 splat(float s) { return make_float2(s, s); }
__device__ __forceinline__ float2 shfl2(float2 v, int src, int width) {
    return make_float2(__shfl_sync(0xffffffffu, v.x, src, width), __shfl_sync(0xffffffffu, v.y, src, width));
}
__device__ __forceinline__ float2 ldcg2(const float2 *p) { return __ldcg(p); }

// alpha / |t| for the isotropic projection, n2 = |t|^2 (PAPER.md:49 line 2; R17).  FAST = false: IEEE square root and
// division.  FAST = true: alpha * rsqrt(n2) and sqrt.approx with the hardware approximations (2 ulp, denormals flushed).
// Which kernels use which, and the measured difference: DESIGN.md R17, profiles/r02/README.md.
#ifndef PD_RESIDENT_FAST_PROJECTION
#define PD_RESIDENT_FAST_PROJECTION 1
#endif
#ifndef PD_STREAMING_FAST_PROJECTION
#define PD_STREAMING_FAST_PROJECTION 1
#endif
constexpr bool kResidentFastProj = PD_RESIDENT_FAST_PROJECTION != 0, kStreamingFastProj = PD_STREAMING_FAST_PROJECTION != 0;
template <bool FAST>
__device__ __forceinline__ float proj_scale(const float alpha, const float n2) {
    if constexpr (FAST) {
        // ONE MUFU instruction (rsqrtf() wraps it in a denormal rescue of four more).  A denormal |t|^2 is flushed to 0,
        // rsqrt gives inf and min(1, alpha inf) leaves such a t (|t| < 1e-19) unscaled: the same as |t| <= alpha.
        float r;
        asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(n2));
        return alpha * r;
    } else {
        return __fdiv_rn(alpha, __fsqrt_rn(n2));
    }
}
// min(1, alpha / |t|): the factor of the isotropic projection, R13-safe (alpha = 0 gives 0; |t| = 0 gives 1 on a zero vector)
template <bool FAST>
__device__ __forceinline__ float proj_factor(const float alpha, const float alpha_sq, const float n2) {
    if constexpr (FAST) return fminf(proj_scale<true>(alpha, n2), 1.f);   // fminf(NaN, 1) = 1 covers 0 * inf
    else return (n2 > alpha_sq) ? proj_scale<false>(alpha, n2) : 1.f;
}
template <bool FAST>
__device__ __forceinline__ float gap_sqrt(const float x) {
    if constexpr (FAST) {
        float r;
        asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
        return r;
    } else {
        return __fsqrt_rn(x);
    }
}

// Per-slice normalisation: two real slices ride one complex transform, and the twiddle
// multiplications mix the lanes' rounding errors, so a weak slice would inherit the absolute error of a strong partner.
// Every slice is therefore scaled by a power of two c = 2^-e that brings its r.m.s. field into [1, 2).  The iteration is
// exactly invariant under (phi, alpha) -> (c phi, c alpha) -- chi, p, q scale by c -- and a power of two is exact in
// floating point, so a slice's result does not depend on c; chi is multiplied by 1/c when it is stored.
// `sumsq` = sum of phi^2 over the slice's `npix` pixels.
__device__ __forceinline__ float pair_scale(const float sumsq, const float npix) {
    if (!(sumsq > 0.f) || !(sumsq < 3.0e38f)) return 1.f;
    int e = ilogbf(sumsq / npix) >> 1;   // floor(log2(rms))
    e = e < -60 ? -60 : (e > 60 ? 60 : e);
    return ldexpf(1.f, -e);
}

template <int N, int C, int NT>
struct ResCfg {
    static constexpr int E = FftCfg<N>::E, T = FftCfg<N>::T;
    static constexpr int RPC = N / C;             // rows (and columns) owned by one CTA
    static constexpr int NG = NT / T;             // row groups
    static constexpr int LDR = T + 1;             // padded exchange row (row phases)
    static constexpr int COLS = 16;               // adjacent columns per column group
    static constexpr int NCG = NT / (COLS * T);   // column groups
    static constexpr int CS = N + 1;              // odd column stride (column phases)
    static constexpr int EXCH_ROW = NG * E * LDR;
    static constexpr int EXCH_COL = NCG * COLS * CS;
    static constexpr int EXCH = EXCH_ROW > EXCH_COL ? EXCH_ROW : EXCH_COL;  // float2 elements
    static constexpr int NWARPS = NT / 32;
    static constexpr int PRIV = E * NT;           // one thread-private array: E float2 per thread, [m][tid]
    static constexpr int SMEM_BYTES = (EXCH + E * T + 2 * PRIV) * 8 + NWARPS * 8 * 4 + 64;
    // one row per group and one column slot per thread, for the whole kernel
    static_assert(NG == RPC && NCG * COLS == RPC, "resident configuration: NT must equal (N/C)*T");
};

// CTA-wide sum of K per-thread values, fixed order; result valid in threads 0..K-1 (as their own k).
template <int NT, int K>
__device__ __forceinline__ float block_sum(float (&val)[K], float *red /*[NT/32][8]*/) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        float v = val[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) red[warp * 8 + k] = v;
    }
    __syncthreads();
    float out = 0.f;
    if (threadIdx.x < K) {
        for (int w = 0; w < NT / 32; ++w) out += red[w * 8 + threadIdx.x];
    }
    __syncthreads();
    return out;
}

// Everything a thread needs for its row (row phases) : pointers already offset to the row.
struct RowPtrs {
    float2 *Z, *qy, *chi, *chibar;
    const float2 *phi2, *M2, *W2;
    float2 *p_s, *qx_s;   // thread-private shared-memory slots: element m at [m * NT]
};

// ------------------------------------------------------------------------------------------------ q-update
// q_{n+1} = proj_alpha(q_n + sigma M G chibar_n)   (PAPER.md:49 line 2; R4, R7).  Independent of the spectrum.
template <int N, int NT, bool ANISO>
__device__ __forceinline__ void q_update_row(const RowPtrs &r, const ResidentArgs &a, const float2 alpha, const int y,
                                             const int j, const bool want_gap, float2 &gap) {
    constexpr int E = FftCfg<N>::E, T = FftCfg<N>::T;
    const bool has_down = y < N - 1;
    const float2 sig2 = splat(a.sigma);
    const float2 alpha_sq = mul2(alpha, alpha);   // alpha is per lane: every slice runs in its own normalisation (pair_scale)
    float2 c0[E];
#pragma unroll
    for (int m = 0; m < E; ++m) c0[m] = ldcg2(r.chibar + j + T * m);
    // operands are loaded a chunk ahead of the stores: a load cannot be scheduled above an earlier store to a
    // possibly aliasing address, so a load-use-store loop body would expose one L2 latency per element
    constexpr int CH = 8;
    float2 cdv[CH], mmv[CH], qyv[CH];
#pragma unroll
    for (int m = 0; m < E; ++m) {
        const int x = j + T * m;
        if (m % CH == 0) {
#pragma unroll
            for (int k = 0; k < CH; ++k) {
                const int xk = x + T * k;
                cdv[k] = has_down ? ldcg2(r.chibar + N + xk) : c0[m + k];   // Neumann: no row below -> gy = 0
                mmv[k] = ldcg2(r.M2 + xk);
                qyv[k] = ldcg2(r.qy + xk);
            }
        }
        const float2 cd = cdv[m % CH];
        const float2 give = (j == 0 && m + 1 < E) ? c0[m + 1 < E ? m + 1 : m] : c0[m];
        float2 cr = shfl2(give, (j + 1) & (T - 1), T);                   // chibar[y][x+1]
        if (m == E - 1 && j == T - 1) cr = c0[m];                        // Neumann: no column to the right -> gx = 0
        const float2 mm = mmv[m % CH];
        const float2 gx = mul2(mm, sub2(cr, c0[m]));
        const float2 gy = mul2(mm, sub2(cd, c0[m]));
        float2 tx = fma2(sig2, gx, r.qx_s[m * NT]);
        float2 ty = fma2(sig2, gy, qyv[m % CH]);
        if (ANISO) {
            tx.x = fminf(fmaxf(tx.x, -alpha.x), alpha.x);
            tx.y = fminf(fmaxf(tx.y, -alpha.y), alpha.y);
            ty.x = fminf(fmaxf(ty.x, -alpha.x), alpha.x);
            ty.y = fminf(fmaxf(ty.y, -alpha.y), alpha.y);
        } else {
            const float2 n2 = fma2(ty, ty, mul2(tx, tx));
            float2 sc;
            sc.x = proj_factor<kResidentFastProj>(alpha.x, alpha_sq.x, n2.x);  // alpha/|t| where |t| > alpha, else 1 (R13: alpha=0 -> 0)
            sc.y = proj_factor<kResidentFastProj>(alpha.y, alpha_sq.y, n2.y);
            tx = mul2(tx, sc);
            ty = mul2(ty, sc);
        }
        r.qx_s[m * NT] = tx;
        r.qy[x] = ty;
        if (want_gap) {   // alpha*|g| - <g, q_{n+1}>
            float2 gn;
            if (ANISO) {
                gn = make_float2(fabsf(gx.x) + fabsf(gy.x), fabsf(gx.y) + fabsf(gy.y));
            } else {
                const float2 g2 = fma2(gy, gy, mul2(gx, gx));
                gn = make_float2(gap_sqrt<kResidentFastProj>(g2.x), gap_sqrt<kResidentFastProj>(g2.y));
            }
            const float2 dot = fma2(gy, ty, mul2(gx, tx));
            gap = add2(gap, sub2(mul2(alpha, gn), dot));
        }
    }
}

// ------------------------------------------------------------------------------------------------ dual step on Z
// u = K chibar_n (finish) ; p_{n+1} = (p_n + sigma W(u - phi))/(1+sigma) ; start K (W p_{n+1}).  PAPER.md:49 line 1.
template <int N, int NT, int LDR, bool HAS_W, class Tw>
__device__ __forceinline__ void dual_z_row(const RowPtrs &r, const ResidentArgs &a, const int j, float2 *smg,
                                           const Tw &tw, const bool want_gap, float2 &gap) {
    constexpr int E = FftCfg<N>::E, T = FftCfg<N>::T;
    float2 v[E];
#pragma unroll
    for (int m = 0; m < E; ++m) v[m] = ldcg2(r.Z + j + T * m);
    fft_line<N, LDR>(v, smg, j, tw, WarpSync());  // v = (u_a, -u_b)
    const float2 sig2 = splat(a.sigma), inv2 = splat(a.inv_one_plus_sigma), half2 = splat(0.5f);
#pragma unroll
    for (int m = 0; m < E; ++m) {
        const int x = j + T * m;
        float2 res = sub2(v[m], r.phi2[x]);
        float2 w;
        if (HAS_W) { w = r.W2[x]; res = mul2(w, res); }
        const float2 pn = mul2(fma2(sig2, res, r.p_s[m * NT]), inv2);
        if (want_gap) {
            const float2 e = sub2(res, pn);
            gap = fma2(mul2(e, half2), e, gap);
        }
        r.p_s[m * NT] = pn;
        v[m] = HAS_W ? mul2(w, pn) : pn;
    }
    fft_line<N, LDR>(v, smg, j, tw, WarpSync());
#pragma unroll
    for (int m = 0; m < E; ++m) r.Z[j + T * m] = v[m];
}

// ------------------------------------------------------------------------------------------------ divergence term
// d = G^T (M q_{n+1}) = -div(M q)  (PAPER.md:49 line 3; R7).  Independent of the spectrum.
template <int N, int NT>
__device__ __forceinline__ void d_term_row(const RowPtrs &r, const int y, const int j, float2 (&d)[FftCfg<N>::E]) {
    constexpr int E = FftCfg<N>::E, T = FftCfg<N>::T;
    const bool has_up = y > 0;
    float2 mqx_prev = make_float2(0.f, 0.f);
#pragma unroll
    for (int m = 0; m < E; ++m) {
        const int x = j + T * m;
        const float2 mm = r.M2[x];
        const float2 mqx = mul2(mm, r.qx_s[m * NT]);
        const float2 give = (j == T - 1 && m > 0) ? mqx_prev : mqx;
        float2 left = shfl2(give, (j + T - 1) & (T - 1), T);             // (M qx)[y][x-1]
        if (m == 0 && j == 0) left = make_float2(0.f, 0.f);
        const float2 mqy = mul2(mm, r.qy[x]);
        const float2 mqy_up = has_up ? mul2(ldcg2(r.M2 - N + x), ldcg2(r.qy - N + x)) : make_float2(0.f, 0.f);
        // qx is 0 in the last column and qy in the last row (their gradient component is 0 there), so no predicate
        d[m] = add2(sub2(left, mqx), sub2(mqy_up, mqy));
        mqx_prev = mqx;
    }
}

// ------------------------------------------------------------------------------------------------ primal step on Z
// v = K(W p_{n+1}) (finish) ; chi_{n+1} = chi_n - tau v - tau d ; chibar_{n+1} = chi_{n+1} + theta (chi_{n+1} - chi_n) ;
// start K chibar_{n+1}.  PAPER.md:49 lines 3-4.
template <int N, int NT, int LDR, class Tw>
__device__ __forceinline__ void primal_z_row(const RowPtrs &r, const ResidentArgs &a, const int j, float2 *smg,
                                             const Tw &tw, const float2 (&d)[FftCfg<N>::E], float *out_a, float *out_b,
                                             const float2 out_scale, float2 &dn, float2 &cn) {
    constexpr int E = FftCfg<N>::E, T = FftCfg<N>::T;
    float2 v[E];
#pragma unroll
    for (int m = 0; m < E; ++m) v[m] = ldcg2(r.Z + j + T * m);
    fft_line<N, LDR>(v, smg, j, tw, WarpSync());  // v = (v_a, v_b)
    const float2 ntau2 = splat(-a.tau), theta2 = splat(a.theta);
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
        const float2 c_new = fma2(ntau2, d[m], fma2(ntau2, v[m], c_old));
        const float2 dc = sub2(c_new, c_old);
        dn = fma2(dc, dc, dn);
        cn = fma2(c_new, c_new, cn);
        const float2 cbar = fma2(theta2, dc, c_new);
        r.chi[x] = c_new;
        r.chibar[x] = cbar;
        v[m] = cbar;
        if (out_a) out_a[x] = out_scale.x * c_new.x;   // back to the caller's units (exact: a power of two)
        if (out_b) out_b[x] = out_scale.y * c_new.y;
    }
    fft_line<N, LDR>(v, smg, j, tw, WarpSync());
#pragma unroll
    for (int m = 0; m < E; ++m) r.Z[j + T * m] = v[m];
}

// ------------------------------------------------------------------------------------------------ column pass
template <int N, class Tw>
__device__ __forceinline__ void dipole_col(float2 *zc, const float *__restrict__ dcol, const int j, float2 *smg,
                                           const Tw &tw) {
    constexpr int E = FftCfg<N>::E, T = FftCfg<N>::T;
    float2 v[E];
#pragma unroll
    for (int m = 0; m < E; ++m) v[m] = ldcg2(zc + (j + T * m) * N);
    float dv[E];
#pragma unroll
    for (int m = 0; m < E; ++m) dv[m] = __ldg(dcol + (j + T * m) * N);
    fft_line<N, T>(v, smg, j, tw, BlockSync());
#pragma unroll
    for (int m = 0; m < E; ++m) v[m] = make_float2(v[m].x * dv[m], v[m].y * -dv[m]);  // conj(D z^): next FFT = conj(inverse)
    fft_line<N, T>(v, smg, j, tw, BlockSync());
#pragma unroll
    for (int m = 0; m < E; ++m) zc[(j + T * m) * N] = v[m];
}

// ------------------------------------------------------------------------------------------------ the kernel
template <int N, int C, int NT, int MINB, bool HAS_W, bool ANISO>
__global__ void __launch_bounds__(NT, MINB)
resident_kernel(const ResidentArgs a) {
    using Cfg = ResCfg<N, C, NT>;
    constexpr int E = Cfg::E, T = Cfg::T, RPC = Cfg::RPC, P = N * N;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *exch = reinterpret_cast<float2 *>(smem_raw);
    float2 *tws = exch + Cfg::EXCH;
    float2 *p_sm = tws + E * T;
    float2 *qx_sm = p_sm + Cfg::PRIV;
    float *red = reinterpret_cast<float *>(qx_sm + Cfg::PRIV);
    float *dec = red + Cfg::NWARPS * 8;  // [0..3]: P0a, P0b, gap_a, gap_b broadcast

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
    const int kx = row0 + cgi * Cfg::COLS + cc;
    float2 *smg_col = exch + (cgi * Cfg::COLS + cc) * Cfg::CS;
    TwiddlesSmem<N> tw_col;
    tw_col.w = tws + cj;

    const long long soff = (long long)cid * P;
    RowPtrs r;
    r.Z = a.Z + soff + y * N; r.qy = a.qy + soff + y * N; r.chi = a.chi + soff + y * N;
    r.chibar = a.chibar + soff + y * N; r.phi2 = a.phi2 + soff + y * N; r.M2 = a.M2 + soff + y * N;
    r.W2 = HAS_W ? a.W2 + soff + y * N : nullptr;
    r.p_s = p_sm + tid; r.qx_s = qx_sm + tid;
    float2 *zcol = a.Z + soff + kx;
    const float *dcol = a.Dtab + kx;
    float *part = a.part + (long long)cid * C * 8;

    for (int pair = cid; pair < a.npairs; pair += ncl) {
        const int s0 = 2 * pair, s1 = s0 + 1;
        const bool has_b = s1 < a.batch;

        // ---- S7 load: field, mask (, W) of my rows -> interleaved scratch; zero state; partial sums of 1/2||W phi||^2
        {
            const float *fa = a.field + (long long)s0 * P + row0 * N;
            const float *fb = a.field + (long long)s1 * P + row0 * N;
            const float *ma = a.mask ? a.mask + s0 * a.mask_bstride + row0 * N : nullptr;
            const float *mb = a.mask ? a.mask + s1 * a.mask_bstride + row0 * N : nullptr;
            const float *wa = HAS_W ? a.weight + (long long)s0 * P + row0 * N : nullptr;
            const float *wb = HAS_W ? a.weight + (long long)s1 * P + row0 * N : nullptr;
            float acc[2] = {0.f, 0.f};
            const float2 zero = make_float2(0.f, 0.f);
            float2 *Zs = a.Z + soff, *qys = a.qy + soff, *chis = a.chi + soff, *cbs = a.chibar + soff;
            float2 *phs = a.phi2 + soff, *Ms = a.M2 + soff;
            for (int i = tid; i < RPC * N; i += NT) {
                const int o = row0 * N + i;
                const float va = fa[i], vb = has_b ? fb[i] : 0.f;
                float w0 = 1.f, w1 = 1.f;
                if (HAS_W) { w0 = wa[i]; w1 = has_b ? wb[i] : 0.f; (a.W2 + soff)[o] = make_float2(w0, w1); }
                phs[o] = make_float2(va, -vb);
                Ms[o] = make_float2(ma ? ma[i] : 1.f, has_b ? (mb ? mb[i] : 1.f) : 0.f);
                qys[o] = zero; chis[o] = zero; cbs[o] = zero; Zs[o] = zero;
                acc[0] = fmaf(w0 * va, w0 * va, acc[0]);
                acc[1] = fmaf(w1 * vb, w1 * vb, acc[1]);
            }
#pragma unroll
            for (int m = 0; m < E; ++m) { r.p_s[m * NT] = zero; r.qx_s[m * NT] = zero; }
            const float t = block_sum<NT, 2>(acc, red);
            if (tid < 2) part[rank * 8 + tid] = t;
        }
        cluster_sync_all<C>();
        if (tid < 2) {
            float t = 0.f;
            for (int q = 0; q < C; ++q) t += __ldcg(part + q * 8 + tid);
            dec[tid] = 0.5f * t;
        }
        __syncthreads();
        // normalisation of the two slices (pair_scale): phi (stored unscaled above) and P0 are rescaled, alpha per lane
        const float ca = pair_scale(2.f * dec[0], (float)P), cb = pair_scale(2.f * dec[1], (float)P);
        if (ca != 1.f || cb != 1.f) {
            float2 *phs = a.phi2 + soff;
            const float2 c2 = make_float2(ca, cb);
            for (int i = tid; i < RPC * N; i += NT) phs[row0 * N + i] = mul2(c2, phs[row0 * N + i]);   // own writes, own reads
        }
        const float P0a = dec[0] * ca * ca, P0b = dec[1] * cb * cb;
        const float2 alpha2 = make_float2(a.alpha * ca, a.alpha * cb);
        const float inv_ca = 1.f / ca, inv_cb = 1.f / cb;
        // R13b: an all-zero slice is never scheduled (every iteration would be a no-op)
        int stop_a = (P0a == 0.f) ? 0 : a.max_iters;
        int stop_b = (!has_b || P0b == 0.f) ? 0 : a.max_iters;
        float gap_a = 0.f, gap_b = 0.f;
        if (stop_a == 0) for (int i = tid; i < RPC * N; i += NT) a.chi_out[(long long)s0 * P + row0 * N + i] = 0.f;
        if (has_b && stop_b == 0) for (int i = tid; i < RPC * N; i += NT) a.chi_out[(long long)s1 * P + row0 * N + i] = 0.f;

        for (int n = 0; n < a.max_iters; ++n) {
            const bool act_a = n < stop_a, act_b = n < stop_b;
            if (!act_a && !act_b) break;
            const bool last = (n + 1 == a.max_iters);
            const bool check = a.tol > 0.f && ((n + 1) % a.check_every) == 0;
            const bool want_gap = check || last;

            // (1) q-update: needs only chibar_n and q_n, both complete since the barrier after the last primal step
            float2 gap = make_float2(0.f, 0.f);
            q_update_row<N, NT, ANISO>(r, a, alpha2, y, j, want_gap, gap);
            if (n > 0) cluster_wait<C>();            // K1 column pass of all CTAs is complete
            // (2) dual step on the spectrum rows
            dual_z_row<N, NT, Cfg::LDR, HAS_W>(r, a, j, smg_row, tw_row, want_gap, gap);
            if (want_gap) {
                float acc[2] = {gap.x, gap.y};
                const float t = block_sum<NT, 2>(acc, red);
                if (tid < 2) part[rank * 8 + 2 + tid] = t;
            }
            cluster_sync_all<C>();
            // (3) K2 column pass; every CTA reduces the same gap partials in the same order (same decision everywhere)
            if (want_gap && tid < 2) {
                float t = 0.f;
                for (int q = 0; q < C; ++q) t += __ldcg(part + q * 8 + 2 + tid);
                dec[2 + tid] = t;
            }
            dipole_col<N>(zcol, dcol, cj, smg_col, tw_col);
            if (want_gap) {   // dec[] was written before the __syncthreads inside dipole_col
                if (act_a) { gap_a = dec[2] / P0a; if (check && gap_a < a.tol) stop_a = n + 1; }
                if (act_b) { gap_b = dec[3] / P0b; if (check && gap_b < a.tol) stop_b = n + 1; }
            }
            cluster_arrive<C>();
            // (4) divergence of M q_{n+1}: independent of the spectrum, overlaps the barrier
            float2 d[E];
            d_term_row<N, NT>(r, y, j, d);
            cluster_wait<C>();
            // (5) primal step on the spectrum rows; a slice finishing now also writes chi to the caller's buffer
            {
                float *out_a = (act_a && n + 1 >= stop_a) ? a.chi_out + (long long)s0 * P + y * N : nullptr;
                float *out_b = (act_b && n + 1 >= stop_b) ? a.chi_out + (long long)s1 * P + y * N : nullptr;
                float2 dn = make_float2(0.f, 0.f), cn = make_float2(0.f, 0.f);
                primal_z_row<N, NT, Cfg::LDR>(r, a, j, smg_row, tw_row, d, out_a, out_b, make_float2(inv_ca, inv_cb), dn, cn);
                if (out_a || out_b) {   // residual of the final iterate (reported, not used for stopping)
                    float acc[4] = {dn.x, cn.x, dn.y, cn.y};
                    const float t = block_sum<NT, 4>(acc, red);
                    if (tid < 4 && ((tid < 2) ? out_a != nullptr : out_b != nullptr)) part[rank * 8 + 4 + tid] = t;
                }
            }
            cluster_sync_all<C>();
            // (6) K1 column pass of the next iteration, if any slice of the pair goes on
            if (n + 1 < a.max_iters && (n + 1 < stop_a || n + 1 < stop_b)) {
                dipole_col<N>(zcol, dcol, cj, smg_col, tw_col);
                cluster_arrive<C>();                // waited for after the next q-update
            }
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
