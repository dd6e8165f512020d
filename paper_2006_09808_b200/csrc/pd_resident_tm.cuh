// pd_resident_tm.cuh -- resident variant, W = identity: the whole primal, dual and k-space state of a slice pair stays
// ON CHIP for all iterations of the solve (BASELINE.json north_star (c); "all intermediates stay on the
// device", taken one level further down the memory hierarchy).
//
// One thread-block cluster of C CTAs owns one slice pair (two real slices ride one complex transform) for
// all its iterations; CTA r owns rows [32 r, 32 r + 32) in the row phases and 32 columns (16 + their mirror images) in
// the column phases.  Where every array lives:
//
//   tensor memory (TMEM, 256 KB/SM)  p^ and phi^ (column role), qx and chi (row role): the four arrays that only their
//                                    owning thread ever touches -- a private window of 8E columns per thread, moved
//                                    with one tcgen05.ld/st per 8 or 16 complex values (tmem.cuh)
//   shared memory                    chibar and qy, in the owning thread's order [m][tid]; the rows above and below
//                                    are the neighbouring thread groups' slots (tid -+ T), and across the CTA boundary
//                                    the neighbouring CTA's shared memory, read through DISTRIBUTED SHARED MEMORY
//                                    (mapa + ld.shared::cluster), one halo row per CTA, phase and direction
//   registers                        the mask M as one bit per pixel and lane (own row and the row above), when every
//                                    mask value of the pair is 0 or 1 (otherwise M is read from an L2 scratch plane)
//   L2 (never HBM)                   the spectrum Z in transit between row and column ownership (the transposes:
//                                    4 x 8 B per pixel pair and iteration), and D (4 B)
//
// HBM is touched when a pair is loaded (field, mask) and when chi_N is stored.  Same algebra as the Fourier-domain
// dual of DESIGN.md 5.0 (PAPER.md:49 line 1 commutes with the FFT when W = I):
//     p^_{n+1} = (p^_n + sigma (D X^_n - phi^)) / (1 + sigma),   X^_n = F chibar_n,   K p_{n+1} = F^-1 (D p^_{n+1}).
// Per pair and iteration n, phases separated by ONE cluster barrier each:
//   column phase n : X^_n = column FFT of Z ; p^ update ; Z <- column FFT of conj(D/N^2 p^_{n+1})
//   q-update n     : q_{n+1} = proj_alpha(q_n + sigma M G chibar_n)                       (PAPER.md:49 line 2)
//   -- cluster barrier, stop decision (same in every CTA) --
//   row phase n    : d = G^T M q_{n+1} ; v = conj(row FFT of Z) = K p_{n+1} ; chi_{n+1} = chi_n - tau (v + d) ;
//                    chibar_{n+1} ; Z <- row FFT of chibar_{n+1}                          (PAPER.md:49 lines 3-4)
//   -- cluster barrier --
// The data term of the gap (R9) is taken in the Fourier domain by Parseval over mirror-paired columns:
// with z = a + i b, A(k) = (Z(k) + conj Z(-k))/2 and B(k) = (Z(k) - conj Z(-k))/(2i) are accumulated per lane
// directly (no difference of two large sums, so a weak slice does not lose digits to a strong partner).
#pragma once
#include "pd_resident.cuh"
#include "tmem.cuh"

namespace pdk {

// regulariser / projection of the kernel instance: the paper's TV term with the isotropic or anisotropic reading of |.|
// (R4), or l1 on chi with a shrinkage prox (PD_REG_L1: no q-update, no divergence term)
constexpr int kModeIso = 0, kModeAniso = 1, kModeL1 = 2;

struct ResidentTmArgs {
    int batch, npairs, max_iters, check_every;
    float alpha, sigma, tau, theta, inv_one_plus_sigma, tol;
    const float *field, *mask;
    long long mask_bstride;
    float *chi_out;
    float2 *Z, *M2;        // per-cluster L2 scratch, each [nclusters][N*N]: spectrum in transit; mask planes (general masks)
    const float *Dpriv;    // D/(N*N) in the column phase's thread-private order: [C][E][NT]
    const float2 *tw_tab;  // exp(-2 pi i n / N)
    float *part;           // [nclusters][C][8] per-CTA partial sums
    int *iters_done;
    float *relgap, *relres;
};

// Column kx owned by (cluster rank, column group cgi in {0,1}, slot cc in 0..15): the low half [16 rank, 16 rank + 16)
// and its mirror images N - kx; the two self-mirrored columns 0 and N/2 both sit in rank 0, slot 0.
// The host builds Dpriv with the same function (pd_api.cu).
__host__ __device__ constexpr int fd_column_of(int N, int rank, int cgi, int cc) {
    const int lo = 16 * rank + cc;
    return cgi == 0 ? lo : (lo == 0 ? N / 2 : N - lo);
}

// ---- distributed shared memory: the same shared-memory offset in another CTA of the cluster
__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t dsmem_addr(const void *p, const unsigned rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_addr(p)), "r"(rank));
    return r;
}
__device__ __forceinline__ float2 ld_dsmem2(const uint32_t addr) {
    float2 v;
    asm volatile("ld.shared::cluster.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr) : "memory");
    return v;
}

// (M_a, M_b) of element m from the per-thread bit mask (bit 2m: lane a, bit 2m+1: lane b)
__device__ __forceinline__ float2 mask_from_bits(const unsigned bits, const int m) {
    return make_float2((bits >> (2 * m)) & 1u ? 1.f : 0.f, (bits >> (2 * m + 1)) & 1u ? 1.f : 0.f);
}

// Everything a thread needs in its row role
template <int N, int NT>
struct TmRow {
    static constexpr int E = FftCfg<N>::E, T = FftCfg<N>::T;
    float2 *cb_t, *qy_t;          // this thread's chibar / qy slots in shared memory: element m at [m * NT]
    uint32_t tm_qx, tm_chi;       // this thread's TMEM windows
    float2 *Z;                    // row y of the spectrum scratch (L2)
    const float2 *M2;             // row y of the mask scratch (L2; general masks only)
    // shared::cluster addresses (element m at + m*NT*8) of the row below in chibar and of the row above in qy: the
    // neighbouring thread group's slots in this CTA, or the neighbouring CTA's first / last row (DISTRIBUTED SHARED
    // MEMORY), or -- at the image border -- the thread's own row (gy = 0) / nothing (has_above false)
    uint32_t cb_below, qy_above;
    bool has_above;
    unsigned mbits;               // the mask of this thread's elements, one bit per pixel and lane (binary masks)
    bool mbin;                    // every mask value of the pair is 0 or 1
};

// ------------------------------------------------------------------------------------------------ column phase
// Thread (column kx, slot j) holds ky = j + T m.  zc = &Z[kx]; dpriv already offset by the thread id.
//   X^ = column FFT of Z (zero when `first`: chibar_0 = 0)
//   p^_{n+1} = (p^_n + sigma (D X^ - phi^)) / (1 + sigma)                 [PAPER.md:49 line 1 in the Fourier domain]
//   Z <- column FFT of conj(D/N^2 p^_{n+1})   (= conjugate of the inverse transform, finished by the row phase)
// With want_gap: Sa += sum |dp(k) + conj dp(-k)|^2, Sb += sum |dp(k) - conj dp(-k)|^2, dp = p^_{n+1} - p^_n (the
// mirror column's dp is in smg_mirror).
template <int N, int NT, class Tw, class Sync>
__device__ __forceinline__ void dual_tm_col(float2 *zc, const float *__restrict__ dpriv, const uint32_t tm_ph,
                                            const uint32_t tm_fh, const int j, float2 *smg, const float2 *smg_mirror,
                                            const Tw &tw, const Sync colsync, const ResidentTmArgs &a, const bool first,
                                            const bool want_gap, float &Sa, float &Sb) {
    constexpr int E = FftCfg<N>::E, T = FftCfg<N>::T, CH = 8;
    float2 v[E];
    float dv[E];
#pragma unroll
    for (int m = 0; m < E; ++m) dv[m] = __ldg(dpriv + m * NT);
    if (!first) {
#pragma unroll
        for (int m = 0; m < E; ++m) v[m] = ldcg2(zc + (j + T * m) * N);
        fft_line<N, T>(v, smg, j, tw, colsync);
    } else {
#pragma unroll
        for (int m = 0; m < E; ++m) v[m] = make_float2(0.f, 0.f);
    }
    const float2 sig2 = splat(a.sigma), inv2 = splat(a.inv_one_plus_sigma);
    constexpr float NN = (float)N * (float)N;
    if (want_gap) __syncthreads();   // the exchange region is free (readers of the FFT above are done)
#pragma unroll
    for (int c = 0; c < E / CH; ++c) {
        float2 ph[CH], fh[CH];
        tm_ld(tm_ph + 2 * CH * c, ph);
        tm_ld(tm_fh + 2 * CH * c, fh);
#pragma unroll
        for (int k = 0; k < CH; ++k) {
            const int m = c * CH + k;
            const float d = dv[m];
            const float2 res = sub2(mul2(splat(d * NN), v[m]), fh[k]);
            const float2 pn = mul2(fma2(sig2, res, ph[k]), inv2);
            if (want_gap) smg[j + T * m] = sub2(pn, ph[k]);
            ph[k] = pn;
            v[m] = make_float2(d * pn.x, -d * pn.y);
        }
        tm_st(tm_ph + 2 * CH * c, ph);
    }
    if (want_gap) {
        __syncthreads();
#pragma unroll
        for (int m = 0; m < E; ++m) {
            const int ky = j + T * m;
            const float2 dp = smg[ky];
            const float2 dm = smg_mirror[(N - ky) & (N - 1)];
            const float ax = dp.x + dm.x, ay = dp.y - dm.y, bx = dp.x - dm.x, by = dp.y + dm.y;
            Sa = fmaf(ax, ax, fmaf(ay, ay, Sa));
            Sb = fmaf(bx, bx, fmaf(by, by, Sb));
        }
    }
    fft_line<N, T>(v, smg, j, tw, colsync);
#pragma unroll
    for (int m = 0; m < E; ++m) zc[(j + T * m) * N] = v[m];
    tm_st_wait();
}

// ------------------------------------------------------------------------------------------------ q-update
// q_{n+1} = proj_alpha(q_n + sigma M G chibar_n)   (PAPER.md:49 line 2; R4, R7).  Independent of the spectrum.
// The scale of the isotropic projection is min(1, alpha / |t|) (proj_scale: hardware reciprocal square root by default
// in the resident kernels, R17 gives the measured cost of the IEEE sqrt + division it replaces); |t| = 0 gives
// min(1, inf) = 1, and alpha = 0 gives 0 (or min(1, NaN) = 1 on a zero vector), so R13 holds without a branch.
template <int N, int NT, bool ANISO>
__device__ __forceinline__ void q_update_tm(const TmRow<N, NT> &r, const ResidentTmArgs &a, const float2 alpha, const int j,
                                            const bool want_gap, float2 &gap) {
    constexpr int E = FftCfg<N>::E, T = FftCfg<N>::T, CH = 8;
    const float sigma = a.sigma;   // alpha is per lane: every slice runs in its own normalisation (pair_scale)
    // chibar[y][x+1] is the next thread's slot of the same element, or (last thread of the row) the first thread's
    // slot of the next element: the same immediate offsets from a per-thread index
    const int cr_off = (j == T - 1) ? NT - T + 1 : 1;
    unsigned mbits = r.mbits;
    asm volatile("" : "+r"(mbits));   // keep the bit tests next to their use (hoisted out of the iteration loop they spill)
#pragma unroll
    for (int c = 0; c < E / CH; ++c) {
        float2 c0v[CH], crv[CH], cdv[CH], qxv[CH], qyv[CH], mmv[CH];
#pragma unroll
        for (int k = 0; k < CH; ++k) c0v[k] = r.cb_t[(c * CH + k) * NT];
#pragma unroll
        for (int k = 0; k < CH; ++k) {
            const int m = c * CH + k;
            crv[k] = r.cb_t[m * NT + cr_off];
            if (m == E - 1 && j == T - 1) crv[k] = c0v[k];   // Neumann in the last column: gx = 0
        }
        // the row below: the next thread group's slots, the next CTA's first row, or the own row (Neumann: gy = 0)
#pragma unroll
        for (int k = 0; k < CH; ++k) cdv[k] = ld_dsmem2(r.cb_below + (uint32_t)((c * CH + k) * NT * 8));
        tm_ld(r.tm_qx + 2 * CH * c, qxv);
#pragma unroll
        for (int k = 0; k < CH; ++k) qyv[k] = r.qy_t[(c * CH + k) * NT];
        if (!r.mbin) {
#pragma unroll
            for (int k = 0; k < CH; ++k) mmv[k] = ldcg2(r.M2 + j + T * (c * CH + k));
        }
#pragma unroll
        for (int k = 0; k < CH; ++k) {
            const int m = c * CH + k;
            float2 sm2;   // sigma * M
            if (r.mbin) sm2 = make_float2((mbits >> (2 * m)) & 1u ? sigma : 0.f, (mbits >> (2 * m + 1)) & 1u ? sigma : 0.f);
            else sm2 = mul2(splat(sigma), mmv[k]);
            const float2 dx = sub2(crv[k], c0v[k]), dy = sub2(cdv[k], c0v[k]);
            float2 tx = fma2(sm2, dx, qxv[k]);
            float2 ty = fma2(sm2, dy, qyv[k]);
            if (ANISO) {
                tx.x = fminf(fmaxf(tx.x, -alpha.x), alpha.x);
                tx.y = fminf(fmaxf(tx.y, -alpha.y), alpha.y);
                ty.x = fminf(fmaxf(ty.x, -alpha.x), alpha.x);
                ty.y = fminf(fmaxf(ty.y, -alpha.y), alpha.y);
            } else {
                const float2 n2 = fma2(ty, ty, mul2(tx, tx));
                const float2 sc = make_float2(proj_factor<kResidentFastProj>(alpha.x, alpha.x * alpha.x, n2.x),
                                              proj_factor<kResidentFastProj>(alpha.y, alpha.y * alpha.y, n2.y));
                tx = mul2(tx, sc);
                ty = mul2(ty, sc);
            }
            qxv[k] = tx;
            r.qy_t[m * NT] = ty;
            if (want_gap) {   // alpha*|g| - <g, q_{n+1}>, g = M G chibar_n
                const float2 mm = r.mbin ? mask_from_bits(mbits, m) : mmv[k];
                const float2 gx = mul2(mm, dx), gy = mul2(mm, dy);
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
        tm_st(r.tm_qx + 2 * CH * c, qxv);
    }
    tm_st_wait();
}

// ------------------------------------------------------------------------------------------------ divergence term
// d = G^T (M q_{n+1}) = -div(M q)  (PAPER.md:49 line 3; R7).  Independent of the spectrum.  With a 0/1 mask M q = q
// (q stays zero wherever M is zero: q_0 = 0 and the update adds sigma M g), so no mask is applied.
template <int N, int NT>
__device__ __forceinline__ void d_term_tm(const TmRow<N, NT> &r, const int j, float2 (&d)[FftCfg<N>::E]) {
    constexpr int E = FftCfg<N>::E, T = FftCfg<N>::T, CH = 8;
    const float2 zero = make_float2(0.f, 0.f);
    float2 mqx_prev = zero;
#pragma unroll
    for (int c = 0; c < E / CH; ++c) {
        float2 qxv[CH], upv[CH];
        tm_ld(r.tm_qx + 2 * CH * c, qxv);
        // (M qy) of the row above: the previous thread group's slots, the previous CTA's last row, or none
#pragma unroll
        for (int k = 0; k < CH; ++k) {
            const float2 u = ld_dsmem2(r.qy_above + (uint32_t)((c * CH + k) * NT * 8));
            upv[k] = r.has_above ? u : zero;
        }
        if (!r.mbin && r.has_above) {
#pragma unroll
            for (int k = 0; k < CH; ++k) upv[k] = mul2(ldcg2(r.M2 - N + j + T * (c * CH + k)), upv[k]);
        }
#pragma unroll
        for (int k = 0; k < CH; ++k) {
            const int m = c * CH + k;
            float2 mqx = qxv[k], mqy = r.qy_t[m * NT];
            if (!r.mbin) {
                const float2 mm = ldcg2(r.M2 + j + T * m);
                mqx = mul2(mm, mqx);
                mqy = mul2(mm, mqy);
            }
            const float2 give = (j == T - 1 && m > 0) ? mqx_prev : mqx;
            float2 left = shfl2(give, (j + T - 1) & (T - 1), T);             // (M qx)[y][x-1]
            if (m == 0 && j == 0) left = zero;
            // qx is 0 in the last column and qy in the last row (their gradient component is 0 there), so no predicate
            d[m] = add2(sub2(left, mqx), sub2(upv[k], mqy));
            mqx_prev = mqx;
        }
    }
}

// ------------------------------------------------------------------------------------------------ row phase
// v = K p_{n+1}: the row FFT of Z gives conj(v_a + i v_b) = (v_a, -v_b).
// chi_{n+1} = chi_n - tau v - tau d ; chibar_{n+1} = chi_{n+1} + theta (chi_{n+1} - chi_n) ; Z <- row FFT of chibar_{n+1}.
// L1 (PD_REG_L1): d = 0 and chi_{n+1} = shrink(chi_n - tau v, thr0 M), thr0 = tau alpha per lane (soft shrinkage, the
// prox of the l1 norm; BASELINE.json north_star).
template <int N, int NT, int LDR, bool L1, class Tw>
__device__ __forceinline__ void primal_tm_row(const TmRow<N, NT> &r, const ResidentTmArgs &a, const int j, float2 *smg,
                                              const Tw &tw, const float2 (&d)[FftCfg<N>::E], float *out_a,
                                              float *out_b, const float2 out_scale, const float2 thr0, float2 &dn,
                                              float2 &cn, const bool need_next) {
    constexpr int E = FftCfg<N>::E, T = FftCfg<N>::T, CH = 8;
    float2 v[E];
#pragma unroll
    for (int m = 0; m < E; ++m) v[m] = ldcg2(r.Z + j + T * m);
    fft_line<N, LDR>(v, smg, j, tw, WarpSync());
    const float2 ntau2 = splat(-a.tau), ntau_v = make_float2(-a.tau, a.tau), theta2 = splat(a.theta);
#pragma unroll
    for (int c = 0; c < E / CH; ++c) {
        float2 cov[CH];
        tm_ld(r.tm_chi + 2 * CH * c, cov);
#pragma unroll
        for (int k = 0; k < CH; ++k) {
            const int m = c * CH + k, x = j + T * m;
            const float2 c_old = cov[k];
            float2 c_new;
            if constexpr (L1) {
                const float2 mm = r.mbin ? mask_from_bits(r.mbits, m) : ldcg2(r.M2 + j + T * m);
                const float2 thr = mul2(thr0, mm), cand = fma2(ntau_v, v[m], c_old);
                c_new = make_float2(copysignf(fmaxf(fabsf(cand.x) - thr.x, 0.f), cand.x),
                                    copysignf(fmaxf(fabsf(cand.y) - thr.y, 0.f), cand.y));
            } else {
                c_new = fma2(ntau2, d[m], fma2(ntau_v, v[m], c_old));
            }
            const float2 dc = sub2(c_new, c_old);
            dn = fma2(dc, dc, dn);
            cn = fma2(c_new, c_new, cn);
            const float2 cbar = fma2(theta2, dc, c_new);
            cov[k] = c_new;
            r.cb_t[m * NT] = cbar;
            v[m] = cbar;
            if (out_a) out_a[x] = out_scale.x * c_new.x;   // back to the caller's units (exact: a power of two)
            if (out_b) out_b[x] = out_scale.y * c_new.y;
        }
        tm_st(r.tm_chi + 2 * CH * c, cov);
    }
    if (need_next) {
        fft_line<N, LDR>(v, smg, j, tw, WarpSync());
#pragma unroll
        for (int m = 0; m < E; ++m) r.Z[j + T * m] = v[m];
    }
    tm_st_wait();
}

template <int N, int C, int NT>
struct ResTmCfg {
    using Base = ResCfg<N, C, NT>;
    static constexpr int E = Base::E, T = Base::T;
    static constexpr int COLS_PER_THREAD = 8 * E;                     // 4 arrays of E float2
    static constexpr int TMEM_COLS = (NT / 128) * COLS_PER_THREAD;    // warps of one lane quarter split the columns
    static constexpr int SMEM_BYTES = (Base::EXCH + E * T + 2 * Base::PRIV) * 8 + Base::NWARPS * 8 * 4 + 128;
    static_assert(NT % 128 == 0, "every lane quarter of the tensor memory needs the same number of warps");
    static_assert(TMEM_COLS >= 32 && TMEM_COLS <= 512 && (TMEM_COLS & (TMEM_COLS - 1)) == 0, "TMEM allocation: power of two in [32, 512]");
};

// ------------------------------------------------------------------------------------------------ the kernel
template <int N, int C, int NT, int MODE>
__global__ void __launch_bounds__(NT, 1)
resident_tm_kernel(const ResidentTmArgs a) {
    constexpr bool ANISO = MODE == kModeAniso, L1 = MODE == kModeL1;
    using Cfg = ResCfg<N, C, NT>;
    using TCfg = ResTmCfg<N, C, NT>;
    constexpr int E = Cfg::E, T = Cfg::T, RPC = Cfg::RPC, P = N * N, CH = 8;
    static_assert(RPC == 32 && Cfg::NCG == 2 && Cfg::COLS == 16, "mirror-pair column ownership needs 2 groups of 16 columns");
    static_assert(E % CH == 0, "elements are moved in chunks of 8");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *exch = reinterpret_cast<float2 *>(smem_raw);
    float2 *tws = exch + Cfg::EXCH;
    float2 *cb_sm = tws + E * T;          // chibar, [m][tid] in the row role's order
    float2 *qy_sm = cb_sm + Cfg::PRIV;    // qy, same order
    float *red = reinterpret_cast<float *>(qy_sm + Cfg::PRIV);
    float *dec = red + Cfg::NWARPS * 8;   // [0..1] P0 ; [2..3] gap ; [4..7] scratch of the gap combination ; [8] mask flag
    uint32_t *tm_slot = reinterpret_cast<uint32_t *>(dec + 12);

    const int tid = threadIdx.x;
    const int rank = (C == 1) ? 0 : (int)cluster_ctarank();
    const int cid = (C == 1) ? (int)blockIdx.x : (int)cluster_id_x();
    const int ncl = (C == 1) ? (int)gridDim.x : (int)num_clusters_x();

    TwiddlesSmem<N>::fill(tws, a.tw_tab, tid, NT);
    const uint32_t tm_base = tmem_alloc(tm_slot, TCfg::TMEM_COLS);   // contains the __syncthreads that publishes tws
    const uint32_t tm = tmem_thread_window(tm_base, TCfg::COLS_PER_THREAD);
    const uint32_t tm_ph = tm, tm_fh = tm + 2 * E;                   // column role: p^, phi^

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
    // the T threads of a column all sit in one column group (warps [cgi NT/64, (cgi+1) NT/64)): the two groups
    // exchange through separate hardware barriers and drift apart (one in FFT arithmetic, the other in loads)
    const NamedSync colsync{1 + cgi, NT / 2};

    const long long soff = (long long)cid * P;
    TmRow<N, NT> r;
    r.cb_t = cb_sm + tid; r.qy_t = qy_sm + tid;
    r.tm_qx = tm + 4 * E; r.tm_chi = tm + 6 * E;
    r.Z = a.Z + soff + y * N; r.M2 = a.M2 + soff + y * N;
    r.cb_below = (g < RPC - 1) ? dsmem_addr(cb_sm + tid + T, (unsigned)rank)
               : (rank < C - 1) ? dsmem_addr(cb_sm + j, (unsigned)(rank + 1))                         // row 0 of CTA rank+1
                                : dsmem_addr(cb_sm + tid, (unsigned)rank);                            // image border
    r.has_above = y > 0;
    r.qy_above = (g > 0) ? dsmem_addr(qy_sm + tid - T, (unsigned)rank)
               : dsmem_addr(qy_sm + (RPC - 1) * T + j, (unsigned)(rank > 0 ? rank - 1 : 0));          // row 31 of CTA rank-1
    r.mbits = 0u; r.mbin = true;
    float2 *zcol = a.Z + soff + kx;
    const float *dpriv = a.Dpriv + rank * (RPC * N) + tid;
    float *part = a.part + (long long)cid * C * 8;
    // 1/2 sum_x e^2 = sum_k |E(k)|^2 / (2 N^2), E = (dp(k) +- conj dp(-k)) / (2 sigma)   (Parseval, header comment)
    const float gap_scale = 0.125f / ((float)N * (float)N * a.sigma * a.sigma);

    for (int pair = cid; pair < a.npairs; pair += ncl) {
        const int s0 = 2 * pair, s1 = s0 + 1;
        const bool has_b = s1 < a.batch;
        const float2 zero = make_float2(0.f, 0.f);

        // ---- S7 load: my row of field and mask; zero state; P0 partial sums; mask bits; then (the slices' norms are
        // known after one cluster barrier) normalisation (pair_scale) and row FFT of phi
        float2 v[E];
        {
            const float *fa = a.field + (long long)s0 * P + y * N;
            const float *fb = a.field + (long long)s1 * P + y * N;
            const float *ma = a.mask ? a.mask + s0 * a.mask_bstride + y * N : nullptr;
            const float *mb = a.mask ? a.mask + s1 * a.mask_bstride + y * N : nullptr;
            float acc[2] = {0.f, 0.f};
            unsigned bits = 0u;
            int general = 0;
#pragma unroll
            for (int m = 0; m < E; ++m) {
                const int x = j + T * m;
                const float va = fa[x], vb = has_b ? fb[x] : 0.f;
                v[m] = make_float2(va, vb);
                const float wa = ma ? ma[x] : 1.f, wb = has_b ? (mb ? mb[x] : 1.f) : 0.f;
                (a.M2 + soff + y * N)[x] = make_float2(wa, wb);
                general |= (wa != 0.f && wa != 1.f) || (wb != 0.f && wb != 1.f);
                bits |= (wa != 0.f ? 1u : 0u) << (2 * m) | (wb != 0.f ? 1u : 0u) << (2 * m + 1);
                acc[0] = fmaf(va, va, acc[0]);
                acc[1] = fmaf(vb, vb, acc[1]);
                r.cb_t[m * NT] = zero; r.qy_t[m * NT] = zero;
            }
            r.mbits = bits;
#pragma unroll
            for (int c = 0; c < E / CH; ++c) {
                float2 z8[CH];
#pragma unroll
                for (int k = 0; k < CH; ++k) z8[k] = zero;
                tm_st(tm_ph + 2 * CH * c, z8);
                tm_st(r.tm_qx + 2 * CH * c, z8);
                tm_st(r.tm_chi + 2 * CH * c, z8);
            }
            general = __syncthreads_or(general);
            const float t = block_sum<NT, 2>(acc, red);
            if (tid < 2) part[rank * 8 + tid] = t;
            if (tid == 2) part[rank * 8 + 6] = general ? 1.f : 0.f;
            tm_st_wait();
        }
        cluster_sync_all<C>();
        if (tid < 3) {
            float t = 0.f;
            const int o = tid < 2 ? tid : 6;
            for (int q = 0; q < C; ++q) t += __ldcg(part + q * 8 + o);
            dec[tid < 2 ? tid : 8] = tid < 2 ? 0.5f * t : t;
        }
        __syncthreads();
        const float ca = pair_scale(2.f * dec[0], (float)P), cb = pair_scale(2.f * dec[1], (float)P);
        {
            const float2 c2 = make_float2(ca, cb);
#pragma unroll
            for (int m = 0; m < E; ++m) v[m] = mul2(c2, v[m]);
            fft_line<N, Cfg::LDR>(v, smg_row, j, tw_row, WarpSync());
#pragma unroll
            for (int m = 0; m < E; ++m) r.Z[j + T * m] = v[m];
        }
        cluster_sync_all<C>();
        // ---- phi^ = column FFT of the row-transformed field, kept in the column role's private window
        {
#pragma unroll
            for (int m = 0; m < E; ++m) v[m] = ldcg2(zcol + (cj + T * m) * N);
            fft_line<N, T>(v, smg_col, cj, tw_col, BlockSync());   // its __syncthreads also publish dec[]
#pragma unroll
            for (int c = 0; c < E / CH; ++c) {
                float2 f8[CH];
#pragma unroll
                for (int k = 0; k < CH; ++k) f8[k] = v[c * CH + k];
                tm_st(tm_fh + 2 * CH * c, f8);
            }
            tm_st_wait();
        }
        const float P0a = dec[0] * ca * ca, P0b = dec[1] * cb * cb;
        const float2 alpha2 = make_float2(a.alpha * ca, a.alpha * cb), out_scale = make_float2(1.f / ca, 1.f / cb);
        r.mbin = dec[8] == 0.f;   // every CTA of the cluster takes the same path
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

            // (1) column phase: p^_{n+1} and the spectrum of K p_{n+1}
            float Sa = 0.f, Sb = 0.f;
            dual_tm_col<N, NT>(zcol, dpriv, tm_ph, tm_fh, cj, smg_col, smg_mir, tw_col, colsync, a, n == 0, want_gap, Sa, Sb);
            // (2) q-update from chibar_n (chibar_0 = 0 and q_0 = 0: nothing to do in the first iteration)
            float2 gap = zero;
            if (!L1 && n > 0) q_update_tm<N, NT, ANISO>(r, a, alpha2, j, want_gap, gap);
            if (want_gap) {
                float acc[4] = {Sa, Sb, gap.x, gap.y};
                const float t = block_sum<NT, 4>(acc, red);
                if (tid < 4) dec[4 + tid] = t;
                __syncthreads();
                if (tid < 2) part[rank * 8 + 2 + tid] = gap_scale * dec[4 + tid] + dec[6 + tid];
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
                if constexpr (!L1) d_term_tm<N, NT>(r, j, d);
                float *out_a = (act_a && n + 1 >= stop_a) ? a.chi_out + (long long)s0 * P + y * N : nullptr;
                float *out_b = (act_b && n + 1 >= stop_b) ? a.chi_out + (long long)s1 * P + y * N : nullptr;
                const bool need_next = (n + 1 < a.max_iters) && (n + 1 < stop_a || n + 1 < stop_b);
                float2 dn = zero, cn = zero;
                primal_tm_row<N, NT, Cfg::LDR, L1>(r, a, j, smg_row, tw_row, d, out_a, out_b, out_scale, mul2(splat(a.tau), alpha2), dn, cn, need_next);
                if (out_a || out_b) {   // residual of the final iterate (reported, not used for stopping)
                    float acc[4] = {dn.x, cn.x, dn.y, cn.y};
                    const float t = block_sum<NT, 4>(acc, red);
                    if (tid < 4 && ((tid < 2) ? out_a != nullptr : out_b != nullptr)) part[rank * 8 + 4 + tid] = t;
                }
            }
            cluster_sync_all<C>();
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
        cluster_sync_all<C>();   // shared memory, scratch and partials are reused by the next pair
    }
    tmem_free(tm_base, TCfg::TMEM_COLS);
}

}  // namespace pdk
