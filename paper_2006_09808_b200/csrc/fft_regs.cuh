// fft_regs.cuh -- register-resident complex FFT building blocks for sm_100a.
//
// A length-N line (N in {64,128,256}) is transformed by T = N/E cooperating threads that each
// hold E points in registers: one in-register DFT of size E, a twiddle multiply, ONE exchange
// through shared memory, and E/T in-register DFTs of size T.  Input and output use the same
// thread<->index map (thread j holds the points j + T*m, m = 0..E-1), so a forward and an inverse
// transform chain without any extra shuffle (used for F^-1 D F).
// N = 512 keeps 16 points per thread (a whole warp per line, T = 32) and runs THREE stages of in-register
// 8-point DFTs with two exchanges (fft_line3): 32 points per thread cost 64 registers for the line alone, which
// held the 512-wide streaming kernels at 96-128 registers and 16-20 warps per SM.
//
// Only the forward (exp(-i...)) transform exists; the inverse is obtained by swapping re/im before
// and after, which is a register renaming.
#pragma once
#include <cuda_runtime.h>

// Blackwell packed fp32x2 arithmetic (FADD2/FFMA2) for the complex butterflies; undefine to fall back to scalar.
#ifndef PDK_SCALAR_BUTTERFLY
#define PDK_PACKED_F32X2 1
#endif

namespace pdk {

// E points per thread, T threads per line; TW: float2 entries of the shared-memory twiddle table (TwiddlesSmem);
// REGION: float2 entries the exchange region of one line needs at least (two-stage lines: E rows of the caller's LD)
// COL: the configuration of the COLUMN kernels, whose T threads of a line sit in different warps and exchange through
// CTA-wide barriers: there the two-stage 512-point line (32 points per thread, two barriers per transform) measured
// faster than the three-stage one (four barriers; 64-register cap at 512 threads per CTA): C4 columns 34.3 vs 38.3 ms.
template <int N, bool COL = false> struct FftCfg;
template <bool COL> struct FftCfg<64, COL>  { static constexpr int E = 8,  T = 8,  TW = E * T, REGION = 0; };
template <bool COL> struct FftCfg<128, COL> { static constexpr int E = 16, T = 8,  TW = E * T, REGION = 0; };
template <bool COL> struct FftCfg<256, COL> { static constexpr int E = 16, T = 16, TW = E * T, REGION = 0; };
template <> struct FftCfg<512, false> { static constexpr int E = 16, T = 32, TW = 2 * E * T, REGION = 544; };
template <> struct FftCfg<512, true>  { static constexpr int E = 32, T = 16, TW = E * T, REGION = 0; };

// cos(2*pi*i/32), sin(2*pi*i/32), i = 0..15, as literals so that they fold after unrolling.
__device__ __forceinline__ float cos32(int i) {
    switch (i) {
        case 0: return 1.0f;
        case 1: return 0.98078528040323044913f;
        case 2: return 0.92387953251128675613f;
        case 3: return 0.83146961230254523708f;
        case 4: return 0.70710678118654752440f;
        case 5: return 0.55557023301960222474f;
        case 6: return 0.38268343236508977173f;
        case 7: return 0.19509032201612826785f;
        case 8: return 0.0f;
        case 9: return -0.19509032201612826785f;
        case 10: return -0.38268343236508977173f;
        case 11: return -0.55557023301960222474f;
        case 12: return -0.70710678118654752440f;
        case 13: return -0.83146961230254523708f;
        case 14: return -0.92387953251128675613f;
        default: return -0.98078528040323044913f;
    }
}
__device__ __forceinline__ float sin32(int i) { return cos32(i < 8 ? 8 - i : i - 8); }  // sin(t) = cos(pi/2 - t)

// d * exp(-2*pi*i*k/R), 0 <= k < R/2, k known after unrolling.
template <int R>
__device__ __forceinline__ float2 twiddle_mul(float2 d, int k) {
    constexpr float C8 = 0.70710678118654752440f;
    if (k == 0) return d;
    if (4 * k == R) return make_float2(d.y, -d.x);
#ifdef PDK_PACKED_F32X2
    // Blackwell's packed FFMA2 takes its operands with the halves swapped and with a sign per half (SASS: R.F32x2.LO_HI.NP)
    // and a scalar broadcast (R.F32), so a complex multiplication is TWO instructions, FMUL2 + FFMA2, instead of four
    // scalar ones: (d.x c + d.y s, d.y c - d.x s) = d (c, c) + (d.y, d.x) (s, -s)
    const float2 dsw = make_float2(d.y, d.x);
    if (8 * k == R) return __fmul2_rn(__ffma2_rn(dsw, make_float2(1.f, -1.f), d), make_float2(C8, C8));          // C8 (d.x + d.y, d.y - d.x)
    if (8 * k == 3 * R) return __fmul2_rn(__ffma2_rn(dsw, make_float2(1.f, -1.f), make_float2(-d.x, -d.y)), make_float2(C8, C8));   // C8 (d.y - d.x, -d.x - d.y)
    const int i = k * (32 / R);  // angle index on the 32-point circle, in (0,16)
    const float c = cos32(i), s = sin32(i);
    return __ffma2_rn(dsw, make_float2(s, -s), __fmul2_rn(d, make_float2(c, c)));
#else
    if (8 * k == R) return make_float2(C8 * (d.x + d.y), C8 * (d.y - d.x));
    if (8 * k == 3 * R) return make_float2(C8 * (d.y - d.x), -C8 * (d.x + d.y));
    const int i = k * (32 / R);  // angle index on the 32-point circle, in (0,16)
    const float c = cos32(i), s = sin32(i);
    return make_float2(fmaf(d.y, s, d.x * c), fmaf(-d.x, s, d.y * c));
#endif
}

// Radix-2 decimation-in-frequency on v[OFF..OFF+R): leaves X[k] at bit-reversed position.
template <int R, int OFF>
struct Dif {
    template <int E>
    static __device__ __forceinline__ void run(float2 (&v)[E]) {
        constexpr int H = R / 2;
#pragma unroll
        for (int k = 0; k < H; ++k) {
            const float2 a = v[OFF + k], b = v[OFF + k + H];
#ifdef PDK_PACKED_F32X2
            // Blackwell packed fp32x2: one FADD2 / FFMA2 per complex add / subtract
            v[OFF + k] = __fadd2_rn(a, b);
            v[OFF + k + H] = twiddle_mul<R>(__ffma2_rn(b, make_float2(-1.f, -1.f), a), k);
#else
            v[OFF + k] = make_float2(a.x + b.x, a.y + b.y);
            v[OFF + k + H] = twiddle_mul<R>(make_float2(a.x - b.x, a.y - b.y), k);
#endif
        }
        Dif<H, OFF>::run(v);
        Dif<H, OFF + H>::run(v);
    }
};
template <int OFF>
struct Dif<1, OFF> {
    template <int E>
    static __device__ __forceinline__ void run(float2 (&)[E]) {}
};

__host__ __device__ constexpr int bit_reverse(int k, int R) {
    int r = 0;
    for (int b = 1; b < R; b <<= 1) {
        r = (r << 1) | (k & 1);
        k >>= 1;
    }
    return r;
}

// In-register forward DFT of size R, natural order in and out (the permutation is register renaming).
template <int R>
__device__ __forceinline__ void dft_reg(float2 (&v)[R]) {
    Dif<R, 0>::run(v);
    float2 t[R];
#pragma unroll
    for (int k = 0; k < R; ++k) t[k] = v[bit_reverse(k, R)];
#pragma unroll
    for (int k = 0; k < R; ++k) v[k] = t[k];
}

// sum over the T threads of one line (T a power of two <= 32, the group is aligned inside its warp)
template <int T>
__device__ __forceinline__ float group_sum(float v) {
#pragma unroll
    for (int o = T / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__device__ __forceinline__ float2 cmul(float2 a, float2 w) {
#ifdef PDK_PACKED_F32X2
    // (a.x w.x - a.y w.y, a.x w.y + a.y w.x) = a (w.x, w.x) + (a.y, a.x) (-w.y, w.y): FMUL2 + FFMA2 (see twiddle_mul)
    return __ffma2_rn(make_float2(a.y, a.x), make_float2(-w.y, w.y), __fmul2_rn(a, make_float2(w.x, w.x)));
#else
    return make_float2(fmaf(-a.y, w.y, a.x * w.x), fmaf(a.x, w.y, a.y * w.x));
#endif
}

struct WarpSync {   // the T threads of a line sit in one warp
    __device__ __forceinline__ void operator()() const { __syncwarp(); }
};
struct BlockSync {  // the T threads of a line are spread over the warps of the CTA
    __device__ __forceinline__ void operator()() const { __syncthreads(); }
};
struct NamedSync {  // ... over `count` threads (whole warps) that all use hardware barrier `id` (1..15)
    int id, count;
    __device__ __forceinline__ void operator()() const { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory"); }
};

// Per-thread inter-stage twiddles W_N^(j*k2), k2 = 1..E-1 (index 0 unused), from the plan's double-precision table.
template <int N>
struct Twiddles {
    static constexpr int E = FftCfg<N>::E, T = FftCfg<N>::T;
    static constexpr bool kThree = false;
    float2 w[E];
    __device__ __forceinline__ void load(const float2 *__restrict__ table, int j) {
#pragma unroll
        for (int k = 1; k < E; ++k) w[k] = __ldg(table + ((j * k) & (N - 1)));
        w[0] = make_float2(1.f, 0.f);
    }
};

// Same twiddles kept in shared memory as a table tws[k2*T + j] = W_N^(j*k2) (conflict-free: consecutive j), read when
// needed instead of living in E registers for the whole kernel.
template <int N, bool COL = false>
struct TwiddlesSmem {
    static constexpr int E = FftCfg<N, COL>::E, T = FftCfg<N, COL>::T;
    static constexpr bool kThree = false;
    const float2 *w;  // &tws[j]
    __device__ __forceinline__ float2 get(int k) const { return w[k * T]; }
    // fill a table of E*T float2 from the plan's W_N^n table (all threads of the CTA cooperate; caller synchronises)
    static __device__ __forceinline__ void fill(float2 *tws, const float2 *__restrict__ table, int tid, int nthreads) {
        for (int i = tid; i < E * T; i += nthreads) tws[i] = __ldg(table + (((i % T) * (i / T)) & (N - 1)));
    }
};
// N = 512, three stages (fft_line3): two tables of 16 entries per thread, [idx][j]:
//   table 1, idx = 8 b + k3 : W_64^(n2 k3),            n2 = (j >> 3) + 4 b
//   table 2, idx = 8 c + k2 : W_512^(n1 (k3 + 8 k2)),  n1 = j & 7, k3 = 2 (j >> 3) + c
template <>
struct TwiddlesSmem<512, false> {
    static constexpr int E = 16, T = 32;
    static constexpr bool kThree = true;
    const float2 *w;  // &tws[j]
    __device__ __forceinline__ float2 get1(int idx) const { return w[idx * T]; }
    __device__ __forceinline__ float2 get2(int idx) const { return w[(16 + idx) * T]; }
    static __device__ __forceinline__ void fill(float2 *tws, const float2 *__restrict__ table, int tid, int nthreads) {
        for (int i = tid; i < 2 * E * T; i += nthreads) {
            const int j = i % T, idx = (i / T) % 16, hi = idx >> 3, lo = idx & 7;
            const int e = (i < E * T) ? 8 * ((j >> 3) + 4 * hi) * lo                     // 8 n2 k3
                                      : (j & 7) * ((2 * (j >> 3) + hi) + 8 * lo);        // n1 (k3 + 8 k2)
            tws[i] = __ldg(table + (e & 511));
        }
    }
};
template <int N>
__device__ __forceinline__ float2 tw_get(const Twiddles<N> &tw, int k) { return tw.w[k]; }
template <int N, bool COL>
__device__ __forceinline__ float2 tw_get(const TwiddlesSmem<N, COL> &tw, int k) { return tw.get(k); }

// N = 512 = 8 x 8 x 8 with n = n1 + 8 n2 + 64 n3 and k = k3 + 8 k2 + 64 k1 (thread j of the warp holds n = j + 32 m:
// n1 = j & 7, n2 = (j >> 3) + 4 (m & 1), n3 = m >> 1):
//   A[n1,n2,k3] = sum_n3 x[n] W_8^(n3 k3)          ; A *= W_64^(n2 k3)            ; exchange 1 (over n2)
//   B[n1,k3,k2] = sum_n2 A[n1,n2,k3] W_8^(n2 k2)   ; B *= W_512^(n1 (k3 + 8 k2))  ; exchange 2 (over n1)
//   X[k3 + 8 k2 + 64 k1] = sum_n1 B[n1,k3,k2] W_8^(n1 k1)
// Every stage is two in-register 8-point DFTs over the elements of equal parity of m; the output lands in the input's
// map (k = j + 32 m with k3 = j & 7, k2 = (j >> 3) + 4 (m & 1), k1 = m >> 1).  sm: >= FftCfg<512>::REGION float2.
// Exchange 1 is bank-conflict free both ways; the writes of exchange 2 are two-way conflicted, its reads free.
template <class Sync>
__device__ __forceinline__ void fft_line3(float2 (&v)[16], float2 *sm, const int j, const TwiddlesSmem<512, false> &tw, Sync sync) {
    const int r = j & 7, q = j >> 3;
    float2 w[8];
#pragma unroll
    for (int b = 0; b < 2; ++b) {   // stage A
#pragma unroll
        for (int i = 0; i < 8; ++i) w[i] = v[b + 2 * i];
        dft_reg<8>(w);
#pragma unroll
        for (int k = 0; k < 8; ++k) v[b + 2 * k] = (k == 0) ? w[0] : cmul(w[k], tw.get1(8 * b + k));
    }
    sync();  // earlier readers of sm are done
#pragma unroll
    for (int b = 0; b < 2; ++b)
#pragma unroll
        for (int k3 = 0; k3 < 8; ++k3) sm[(k3 >> 1) * 136 + (k3 & 1) * 64 + b * 32 + j] = v[b + 2 * k3];   // (k3, n2 = q + 4b, n1 = r)
    sync();
#pragma unroll
    for (int c = 0; c < 2; ++c) {   // stage B: k3 = 2q + c
#pragma unroll
        for (int n2 = 0; n2 < 8; ++n2) w[n2] = sm[q * 136 + c * 64 + n2 * 8 + r];
        dft_reg<8>(w);
#pragma unroll
        for (int k = 0; k < 8; ++k) v[c + 2 * k] = cmul(w[k], tw.get2(8 * c + k));
    }
    sync();  // exchange 1 has been read
#pragma unroll
    for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int k2 = 0; k2 < 8; ++k2) sm[r * 65 + k2 * 8 + 2 * q + c] = v[c + 2 * k2];   // (n1 = r, k2, k3 = 2q + c)
    sync();
#pragma unroll
    for (int b = 0; b < 2; ++b) {   // stage C: k3 = r, k2 = q + 4b
#pragma unroll
        for (int n1 = 0; n1 < 8; ++n1) w[n1] = sm[n1 * 65 + (q + 4 * b) * 8 + r];
        dft_reg<8>(w);
#pragma unroll
        for (int k1 = 0; k1 < 8; ++k1) v[b + 2 * k1] = w[k1];
    }
}

// Cooperative forward FFT of one length-N line held by T threads (thread j: points j + T*m).
//   sm : this line's exchange region, E rows of LD float2 (row k2, column j)
//   SYNC: functor that synchronises the T threads of the line (and orders their shared-memory accesses)
template <int N, int LD, class Tw, class Sync>
__device__ __forceinline__ void fft_line(float2 (&v)[Tw::E], float2 *sm, int j, const Tw &tw,
                                         Sync sync) {
    if constexpr (Tw::kThree) {
        fft_line3(v, sm, j, tw, sync);
        return;
    } else {
    constexpr int E = Tw::E, T = Tw::T, C = E / T;
    dft_reg<E>(v);  // over n2: Y[j][k2]
#pragma unroll
    for (int k = 1; k < E; ++k) v[k] = cmul(v[k], tw_get(tw, k));
    sync();  // earlier readers of sm are done
#pragma unroll
    for (int k = 0; k < E; ++k) sm[k * LD + j] = v[k];
    sync();
#pragma unroll
    for (int c = 0; c < C; ++c) {
        float2 w[T];
#pragma unroll
        for (int n = 0; n < T; ++n) w[n] = sm[(j + T * c) * LD + n];
        dft_reg<T>(w);  // over n1: X[E*k1 + (j + T*c)] = X[j + T*(C*k1 + c)]
#pragma unroll
        for (int k1 = 0; k1 < T; ++k1) v[C * k1 + c] = w[k1];
    }
    }
}

}  // namespace pdk
