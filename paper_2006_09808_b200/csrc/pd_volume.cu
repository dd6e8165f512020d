// pd_volume.cu -- the true 3-D variant: Eq.(1) as the paper literally states it, "G is the
// gradient operator in all three dimensions", with the 3-D dipole kernel, one problem per VOLUME
// [nz][ny][nx] (slices are coupled: no per-slice stop, the iteration count is the caller's; R23, 5.7).
//
// A streaming implementation: W = identity (else the literal path below), so the dual p lives in the Fourier domain as in DESIGN.md 5.0 -- ONE 3-D FFT
// round trip per iteration -- and two real volumes (coils) ride one complex transform, z = a + i b (D3 is real and even,
// so F^-1 D3 F z = K a + i K b, and the p-update is linear: it acts on the packed spectrum as it stands):
//   x lines (chi_bar real -> complex) ; y lines ; z lines + [ p^ <- (p^ + sigma (D Z - phi^))/(1+sigma) ; Z <- D p^ ] + z lines
//   back ; y lines back ; x lines back (-> K p, real) ; q-update (3 components) ; chi-update with the 3-D divergence.
// Line transforms: radix-2 in shared memory, 16 lines per CTA; strided axes (y, z) are read as tiles of 16 adjacent x so
// that every access is a full 128-byte line.  Twiddles and D come from double-precision host tables (R17).  No cuFFT.
#include "../../include/pd.h"
#include "fft_regs.cuh"

#include <cuda_runtime.h>

#include <cmath>
#include <cstring>
#include <new>
#include <vector>

int pd_cuda_fail_(int cuda_error, const char *where);   // pd_api.cu: records the text behind PD_ECUDA

namespace {

constexpr int kTL = 16;         // lines per CTA
constexpr int kThreads = 256;

enum { kModePlain = 0, kModeInReal = 1, kModeOutReal = 2, kModeStoreSpectrum = 3, kModeDual = 4, kModeInRealScaled = 5, kModeMulD = 6 };

struct FftArgs {
    const float *in_real;     // kModeInReal
    float2 *z;                // complex work volume (in place)
    float *out_real;          // kModeOutReal
    float2 *phihat, *phat;    // kModeStoreSpectrum / kModeDual
    const float *D;           // [nz][ny][nx], unscaled
    const float2 *tw;         // exp(-2 pi i k / N), k < N
    long long nlines;         // x pass: number of lines (of the PAIRED volumes)
    long long V;              // voxels of one volume
    int lines_per_vol;        // nz * ny
    const float *cscale;      // kModeInReal: per-volume factor applied on load (NULL: none)
    int nvol;                 // real volumes: the pair pv holds volume 2 pv in its real part and 2 pv + 1 (if any) in its imaginary part
    long long S;              // strided pass: distance between consecutive points of a line (nx, or nx*ny)
    float sigma, inv1ps, out_scale;
    int inverse;
};

template <int N> struct Log2 { static constexpr int v = 1 + Log2<N / 2>::v; };
template <> struct Log2<1> { static constexpr int v = 0; };

template <int N>
__device__ __forceinline__ int brev(int k) { return (int)(__brev((unsigned)k) >> (32 - Log2<N>::v)); }

// radix-2 decimation in time over the kTL lines of the tile; input in bit-reversed order, output in natural order
template <int N>
__device__ __forceinline__ void fft_tile(float2 *buf, const float2 *tws, bool inverse) {
    constexpr int LOGN = Log2<N>::v, LD = N + 1;
#pragma unroll 1
    for (int s = 0; s < LOGN; ++s) {
        const int half = 1 << s;
        for (int idx = threadIdx.x; idx < kTL * (N / 2); idx += kThreads) {
            const int l = idx / (N / 2), b = idx % (N / 2);
            const int j = b & (half - 1), i0 = ((b >> s) << (s + 1)) + j, i1 = i0 + half;
            float2 w = tws[j << (LOGN - 1 - s)];
            if (inverse) w.y = -w.y;
            const float2 a = buf[l * LD + i0], c = buf[l * LD + i1];
            const float2 t = make_float2(c.x * w.x - c.y * w.y, c.x * w.y + c.y * w.x);
            buf[l * LD + i0] = make_float2(a.x + t.x, a.y + t.y);
            buf[l * LD + i1] = make_float2(a.x - t.x, a.y - t.y);
        }
        __syncthreads();
    }
}

// STRIDED = false: lines along x (contiguous), the tile is 16 consecutive lines.
// STRIDED = true : point k of line (o, j) sits at (o*N + k)*S + j; the tile is 16 consecutive j (blockIdx.x), o = blockIdx.y.
template <int N, bool STRIDED>
__global__ void __launch_bounds__(kThreads) fft_lines_kernel(const FftArgs a, const int mode) {
    constexpr int LD = N + 1;
    __shared__ float2 buf[kTL * LD];
    __shared__ float2 tws[N / 2 > 0 ? N / 2 : 1];
    for (int k = threadIdx.x; k < N / 2; k += kThreads) tws[k] = a.tw[k];
    const long long L0 = (long long)blockIdx.x * kTL;                                    // first line (x) / first j (strided)
    const long long base = STRIDED ? (long long)blockIdx.y * N * a.S + L0 : L0 * N;
    // ---- load (bit-reversed positions)
    for (int idx = threadIdx.x; idx < kTL * N; idx += kThreads) {
        int l, k;
        long long g;
        if (STRIDED) { l = idx % kTL; k = idx / kTL; g = base + (long long)k * a.S + l; }
        else { l = idx / N; k = idx % N; g = base + (long long)l * N + k; }
        float2 v = make_float2(0.f, 0.f);
        if (STRIDED || L0 + l < a.nlines) {
            if (mode == kModeInReal || mode == kModeInRealScaled) {
                const long long pv = (L0 + l) / a.lines_per_vol, r = g + pv * a.V;       // volume 2 pv, same line and point
                v = make_float2(a.in_real[r], 2 * pv + 1 < a.nvol ? a.in_real[r + a.V] : 0.f);
                if (mode == kModeInRealScaled) { v.x *= a.cscale[2 * pv]; if (2 * pv + 1 < a.nvol) v.y *= a.cscale[2 * pv + 1]; }
            } else {
                v = a.z[g];
            }
        }
        buf[l * LD + brev<N>(k)] = v;
    }
    __syncthreads();
    fft_tile<N>(buf, tws, a.inverse != 0);
    if (mode == kModeStoreSpectrum || mode == kModeDual || mode == kModeMulD) {
        // the last forward axis: every coordinate is a frequency now (PAPER.md:49 line 1 in the Fourier domain, W = I)
        for (int idx = threadIdx.x; idx < kTL * N; idx += kThreads) {
            const int l = idx % kTL, k = idx / kTL;
            const long long g = base + (long long)k * a.S + l;
            const float2 z = buf[l * LD + k];
            if (mode == kModeStoreSpectrum) { a.phihat[g] = z; continue; }
            const float d = a.D[g - (long long)blockIdx.y * N * a.S];
            if (mode == kModeMulD) { buf[l * LD + k] = make_float2(d * z.x, d * z.y); continue; }   // literal path: K alone
            const float2 f = a.phihat[g];
            float2 p = a.phat[g];
            p.x = (p.x + a.sigma * (d * z.x - f.x)) * a.inv1ps;
            p.y = (p.y + a.sigma * (d * z.y - f.y)) * a.inv1ps;
            a.phat[g] = p;
            buf[l * LD + k] = make_float2(d * p.x, d * p.y);                             // spectrum of K p (unnormalised)
        }
        if (mode == kModeStoreSpectrum) return;
        __syncthreads();
        for (int idx = threadIdx.x; idx < kTL * N; idx += kThreads) {                    // natural -> bit-reversed, in place
            const int l = idx % kTL, k = idx / kTL, r = brev<N>(k);
            if (k < r) { const float2 t = buf[l * LD + k]; buf[l * LD + k] = buf[l * LD + r]; buf[l * LD + r] = t; }
        }
        __syncthreads();
        fft_tile<N>(buf, tws, true);
    }
    // ---- store
    for (int idx = threadIdx.x; idx < kTL * N; idx += kThreads) {
        int l, k;
        long long g;
        if (STRIDED) { l = idx % kTL; k = idx / kTL; g = base + (long long)k * a.S + l; }
        else { l = idx / N; k = idx % N; g = base + (long long)l * N + k; }
        if (!STRIDED && L0 + l >= a.nlines) continue;
        const float2 v = buf[l * LD + k];
        if (mode == kModeOutReal) {
            const long long pv = (L0 + l) / a.lines_per_vol, r = g + pv * a.V;
            a.out_real[r] = v.x * a.out_scale;
            if (2 * pv + 1 < a.nvol) a.out_real[r + a.V] = v.y * a.out_scale;
        } else {
            a.z[g] = v;
        }
    }
}

// Lines of 64, 128 or 256 points: the register transform of fft_regs.cuh (T threads per line hold E points each, one
// exchange through shared memory, packed FFMA2 butterflies); input and output share the thread map k = j + T m, so the
// forward transform, the p-update and the inverse transform of the z pass chain in registers.  Same tiles as above.
template <int N, bool STRIDED, int mode>
__global__ void __launch_bounds__(kTL * pdk::FftCfg<N>::T, (mode == kModeDual ? 512 : 768) / (kTL * pdk::FftCfg<N>::T)) fft_lines_reg_kernel(const FftArgs a) {
    using Cfg = pdk::FftCfg<N>;
    constexpr int E = Cfg::E, T = Cfg::T, LD = T + 1, NT = kTL * T;
    // exchange region of one line: E rows of LD, plus one entry so that the regions of the 16 lines of a tile start in
    // different banks (E*LD float2 is a multiple of 32 words: sixteen lines on one bank, a 16-way conflict, measured)
    constexpr int REG = E * LD + 1;
    __shared__ float2 tws[E * T];
    __shared__ float2 ex[kTL * REG];
    pdk::TwiddlesSmem<N>::fill(tws, a.tw, threadIdx.x, NT);
    const int l = STRIDED ? threadIdx.x % kTL : threadIdx.x / T;     // line of the tile
    const int j = STRIDED ? threadIdx.x / kTL : threadIdx.x % T;     // thread of the line
    pdk::TwiddlesSmem<N> tw;
    tw.w = tws + j;
    float2 *sm = ex + l * REG;
    const long long L0 = (long long)blockIdx.x * kTL;
    const long long vol = STRIDED ? (long long)blockIdx.y * N * a.S : 0;                 // first point of my (outer) block
    const long long base = STRIDED ? vol + L0 + l : (L0 + l) * N;                        // first point of my line
    const int step = STRIDED ? (int)a.S : 1;                                             // distance between its points
    const bool live = STRIDED || L0 + l < a.nlines;
    float2 *const zl = a.z + base;
    // real volumes behind the pair (x passes only): volume 2 pv at rbase, volume 2 pv + 1 one volume further
    const long long pv = STRIDED ? 0 : (L0 + l) / a.lines_per_vol, rbase = base + pv * a.V;
    const bool has_b = !STRIDED && 2 * pv + 1 < a.nvol;
    constexpr bool IN_REAL = mode == kModeInReal || mode == kModeInRealScaled;
    float ca = 1.f, cb = 1.f;   // per-volume power-of-two normalisation of the field (exact), see vol_scale_kernel
    if (mode == kModeInRealScaled) { ca = a.cscale[2 * pv]; if (has_b) cb = a.cscale[2 * pv + 1]; }
    float2 v[E];
#pragma unroll
    for (int m = 0; m < E; ++m) {
        const int o = (j + T * m) * step;
        if (!live) v[m] = make_float2(0.f, 0.f);
        else if (IN_REAL) v[m] = make_float2(__ldg(a.in_real + rbase + o), has_b ? __ldg(a.in_real + rbase + a.V + o) : 0.f);
        else v[m] = zl[o];
    }
    if (mode == kModeInRealScaled) {   // after all loads have been issued
#pragma unroll
        for (int m = 0; m < E; ++m) v[m] = make_float2(ca * v[m].x, cb * v[m].y);
    }
    __syncthreads();   // twiddle table filled
    auto transform = [&](bool inverse) {   // the inverse is the forward transform of the swapped halves (fft_regs.cuh)
        if (inverse) {
#pragma unroll
            for (int m = 0; m < E; ++m) v[m] = make_float2(v[m].y, v[m].x);
        }
        if (STRIDED) pdk::fft_line<N, LD>(v, sm, j, tw, pdk::BlockSync());
        else pdk::fft_line<N, LD>(v, sm, j, tw, pdk::WarpSync());
        if (inverse) {
#pragma unroll
            for (int m = 0; m < E; ++m) v[m] = make_float2(v[m].y, v[m].x);
        }
    };
    // z pass of the iteration: with 8 points per thread the operands of the p-update are requested BEFORE the forward
    // transform, so that a CTA has one memory phase instead of two dependent ones (40 registers; not at 16 points)
    constexpr bool PRE = (mode == kModeDual) && E <= 8;
    float2 pf[PRE ? E : 1], pp[PRE ? E : 1];
    float pd[PRE ? E : 1];
    if (PRE) {
#pragma unroll
        for (int m = 0; m < E; ++m) {
            const int o = (j + T * m) * step;
            pd[m] = __ldg(a.D + (base - vol) + o);
            pf[m] = a.phihat[base + o];
            pp[m] = a.phat[base + o];
        }
    }
    transform(a.inverse != 0);
    if (mode == kModeStoreSpectrum) {
        float2 *const fl = a.phihat + base;
#pragma unroll
        for (int m = 0; m < E; ++m) fl[(j + T * m) * step] = v[m];
        return;
    }
    if (mode == kModeMulD) {   // literal path (W set): K = F^-1 D3 F alone
        const float *const dl = a.D + (base - vol);
#pragma unroll
        for (int m = 0; m < E; ++m) {
            const float d = __ldg(dl + (j + T * m) * step);
            v[m] = make_float2(d * v[m].x, d * v[m].y);
        }
        transform(true);
    }
    if (mode == kModeDual) {   // PAPER.md:49 line 1 in the Fourier domain (W = I), then the spectrum of K p
        const float2 *const fl = a.phihat + base;
        float2 *const pl = a.phat + base;
        const float *const dl = a.D + (base - vol);
#pragma unroll
        for (int m = 0; m < E; ++m) {
            const int o = (j + T * m) * step;
            const float d = PRE ? pd[m] : __ldg(dl + o);
            const float2 f = PRE ? pf[m] : fl[o];
            float2 p = PRE ? pp[m] : pl[o];
            p.x = (p.x + a.sigma * (d * v[m].x - f.x)) * a.inv1ps;
            p.y = (p.y + a.sigma * (d * v[m].y - f.y)) * a.inv1ps;
            pl[o] = p;
            v[m] = make_float2(d * p.x, d * p.y);
        }
        transform(true);
    }
    if (!live) return;
#pragma unroll
    for (int m = 0; m < E; ++m) {
        const int o = (j + T * m) * step;
        if (mode == kModeOutReal) {
            a.out_real[rbase + o] = v[m].x * a.out_scale;
            if (has_b) a.out_real[rbase + a.V + o] = v[m].y * a.out_scale;
        } else {
            zl[o] = v[m];
        }
    }
}

// z lines of ANY length up to 64 (the paper's volumes have 25, 12 and 42 slices): a dense DFT per line in
// shared memory, O(nz^2) -- 2 x 42 complex multiply-adds per voxel pair for nz = 42, still cheaper than the pass's memory
// traffic is long.  Same tiles (16 adjacent x) and the same modes as the strided kernels above.
constexpr int kDenseMax = 64;
__global__ void __launch_bounds__(kThreads) dft_lines_dense_kernel(const FftArgs a, const int mode, const int N) {
    __shared__ float2 buf[2][kTL * (kDenseMax + 1)];
    __shared__ float2 tws[kDenseMax];
    const int LD = N + 1;
    for (int k = threadIdx.x; k < N; k += kThreads) tws[k] = a.tw[k];
    const long long vol = (long long)blockIdx.y * N * a.S, base = vol + (long long)blockIdx.x * kTL;
    for (int idx = threadIdx.x; idx < kTL * N; idx += kThreads) {
        const int l = idx % kTL, k = idx / kTL;
        buf[0][l * LD + k] = a.z[base + (long long)k * a.S + l];
    }
    __syncthreads();
    auto dft = [&](const float2 *in, float2 *out, bool inverse) {   // out[k] = sum_n in[n] W^(+-nk)
        for (int idx = threadIdx.x; idx < kTL * N; idx += kThreads) {
            const int l = idx % kTL, k = idx / kTL;
            float2 acc = make_float2(0.f, 0.f);
            int e = 0;
            for (int n = 0; n < N; ++n) {
                float2 w = tws[e];
                if (inverse) w.y = -w.y;
                const float2 c = in[l * LD + n];
                acc.x = fmaf(c.x, w.x, fmaf(-c.y, w.y, acc.x));
                acc.y = fmaf(c.x, w.y, fmaf(c.y, w.x, acc.y));
                e += k;
                if (e >= N) e -= N;
            }
            out[l * LD + k] = acc;
        }
        __syncthreads();
    };
    dft(buf[0], buf[1], a.inverse != 0);
    float2 *res = buf[1];
    if (mode == kModeStoreSpectrum || mode == kModeDual || mode == kModeMulD) {
        for (int idx = threadIdx.x; idx < kTL * N; idx += kThreads) {
            const int l = idx % kTL, k = idx / kTL;
            const long long g = base + (long long)k * a.S + l;
            const float2 z = buf[1][l * LD + k];
            if (mode == kModeStoreSpectrum) { a.phihat[g] = z; continue; }
            const float d = a.D[g - vol];
            if (mode == kModeMulD) { buf[1][l * LD + k] = make_float2(d * z.x, d * z.y); continue; }
            const float2 f = a.phihat[g];
            float2 p = a.phat[g];
            p.x = (p.x + a.sigma * (d * z.x - f.x)) * a.inv1ps;
            p.y = (p.y + a.sigma * (d * z.y - f.y)) * a.inv1ps;
            a.phat[g] = p;
            buf[1][l * LD + k] = make_float2(d * p.x, d * p.y);
        }
        if (mode == kModeStoreSpectrum) return;
        __syncthreads();
        dft(buf[1], buf[0], true);
        res = buf[0];
    }
    for (int idx = threadIdx.x; idx < kTL * N; idx += kThreads) {
        const int l = idx % kTL, k = idx / kTL;
        a.z[base + (long long)k * a.S + l] = res[l * LD + k];
    }
}

struct VoxArgs {
    int nx, ny, nz;           // powers of two; nx a multiple of 4
    int lx, ly, lv, lz;       // log2 nx, log2 ny, log2 (nx ny nz) (unused), log2 nz or -1 when nz is not a power of two
    const float *cscale;      // [nvol] normalisation of every volume: the ball of volume v has radius alpha * cscale[v]
    const float *weight, *field;   // literal path (W set): W, and the caller's phi (normalised on the fly)
    float *p, *wp;                 // literal path: the dual p in the image domain, and W p (input of the second K)
    float inv1ps;
    long long nvox;           // nvol * nz * ny * nx
    const float *mask;        // or NULL (ones)
    float *chi, *chibar, *qx, *qy, *qz;
    const float *kp;
    float sigma, tau, theta, alpha;
};

__device__ __forceinline__ float4 ld4(const float *p) { return *reinterpret_cast<const float4 *>(p); }
__device__ __forceinline__ void st4(float *p, float4 v) { *reinterpret_cast<float4 *>(p) = v; }
__device__ __forceinline__ float4 sub4(float4 a, float4 b) { return make_float4(a.x - b.x, a.y - b.y, a.z - b.z, a.w - b.w); }

// q <- proj_alpha(q + sigma M G chi_bar): forward differences, Neumann, pointwise Euclidean norm over the three components
// (PAPER.md:49 line 2; R4, R7, R13 carried to 3-D by R23).  Four voxels along x per thread and trip.
__global__ void __launch_bounds__(kThreads, 4) q_update3_kernel(const VoxArgs a) {
    const long long sy = a.nx, sz = (long long)a.nx << a.ly, nquad = a.nvox >> 2;
    const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f), one = make_float4(1.f, 1.f, 1.f, 1.f);
    for (long long i4 = (long long)blockIdx.x * kThreads + threadIdx.x; i4 < nquad; i4 += (long long)gridDim.x * kThreads) {
        const long long i = i4 << 2;
        const int plane = (int)(i >> (a.lx + a.ly)), vol = a.lz >= 0 ? plane >> a.lz : plane / a.nz;   // nz need not be a power of two
        const int x = (int)(i & (a.nx - 1)), y = (int)((i >> a.lx) & (a.ny - 1)), z = plane - vol * a.nz;
        const float4 c = ld4(a.chibar + i), m = a.mask ? ld4(a.mask + i) : one;
        const float cn = x + 4 < a.nx ? a.chibar[i + 4] : c.w;                         // Neumann: last x difference is 0
        const float4 gx = make_float4(c.y - c.x, c.z - c.y, c.w - c.z, cn - c.w);
        const float4 gy = y + 1 < a.ny ? sub4(ld4(a.chibar + i + sy), c) : zero;
        const float4 gz = z + 1 < a.nz ? sub4(ld4(a.chibar + i + sz), c) : zero;
        float4 qx = ld4(a.qx + i), qy = ld4(a.qy + i), qz = ld4(a.qz + i);
        const float alpha = a.alpha * a.cscale[vol];
        auto one_voxel = [&](float &px, float &py, float &pz, float mm, float dx, float dy, float dz) {
            const float tx = px + a.sigma * mm * dx, ty = py + a.sigma * mm * dy, tz = pz + a.sigma * mm * dz;
            const float nrm = sqrtf(tx * tx + ty * ty + tz * tz);
            const float s = nrm > alpha ? alpha / nrm : 1.f;
            px = tx * s; py = ty * s; pz = tz * s;
        };
        one_voxel(qx.x, qy.x, qz.x, m.x, gx.x, gy.x, gz.x);
        one_voxel(qx.y, qy.y, qz.y, m.y, gx.y, gy.y, gz.y);
        one_voxel(qx.z, qy.z, qz.z, m.z, gx.z, gy.z, gz.z);
        one_voxel(qx.w, qy.w, qz.w, m.w, gx.w, gy.w, gz.w);
        st4(a.qx + i, qx); st4(a.qy + i, qy); st4(a.qz + i, qz);
        if (a.weight) {   // literal path: p <- (p + sigma W (K chi_bar - phi))/(1 + sigma)  (PAPER.md:49 line 1; R3); a.kp holds K chi_bar
            const float cs = a.cscale[vol];
            const float4 w = ld4(a.weight + i), u = ld4(a.kp + i), f = ld4(a.field + i);
            float4 pp = ld4(a.p + i);
            pp.x = (pp.x + a.sigma * w.x * (u.x - cs * f.x)) * a.inv1ps;
            pp.y = (pp.y + a.sigma * w.y * (u.y - cs * f.y)) * a.inv1ps;
            pp.z = (pp.z + a.sigma * w.z * (u.z - cs * f.z)) * a.inv1ps;
            pp.w = (pp.w + a.sigma * w.w * (u.w - cs * f.w)) * a.inv1ps;
            st4(a.p + i, pp);
            st4(a.wp + i, make_float4(w.x * pp.x, w.y * pp.y, w.z * pp.z, w.w * pp.w));
        }
    }
}

// chi+ = chi - tau (K p + G^T (M q)) ; chi_bar = chi+ + theta (chi+ - chi)   (PAPER.md:49 lines 3, 4)
// G^T v at a voxel = v_x(x-1) [x >= 1] - v_x(x) [x <= nx-2] + the same along y and z, v = M q.
// Four voxels along x starting at voxel i = (.., z, y, x); k = K p there.  Stores chi+ and chi_bar, returns chi_bar.
__device__ __forceinline__ float4 chi_quad(const VoxArgs &a, long long i, int x, int y, int z, float4 k) {
    const long long sy = a.nx, sz = (long long)a.nx << a.ly;
    const float4 one = make_float4(1.f, 1.f, 1.f, 1.f);
    auto mul4 = [](float4 u, float4 w) { return make_float4(u.x * w.x, u.y * w.y, u.z * w.z, u.w * w.w); };
    const float4 m = a.mask ? ld4(a.mask + i) : one;
    float4 vx = mul4(m, ld4(a.qx + i));
    const float4 vy = mul4(m, ld4(a.qy + i)), vz = mul4(m, ld4(a.qz + i));
    const float vxl = x >= 1 ? (a.mask ? a.mask[i - 1] : 1.f) * a.qx[i - 1] : 0.f;
    if (x + 4 == a.nx) vx.w = 0.f;                                                 // no difference leaves the last column
    float4 div = make_float4(vxl - vx.x, vx.x - vx.y, vx.y - vx.z, vx.z - vx.w);
    if (y >= 1) { const float4 t = mul4(a.mask ? ld4(a.mask + i - sy) : one, ld4(a.qy + i - sy)); div.x += t.x; div.y += t.y; div.z += t.z; div.w += t.w; }
    if (y + 1 < a.ny) { div.x -= vy.x; div.y -= vy.y; div.z -= vy.z; div.w -= vy.w; }
    if (z >= 1) { const float4 t = mul4(a.mask ? ld4(a.mask + i - sz) : one, ld4(a.qz + i - sz)); div.x += t.x; div.y += t.y; div.z += t.z; div.w += t.w; }
    if (z + 1 < a.nz) { div.x -= vz.x; div.y -= vz.y; div.z -= vz.z; div.w -= vz.w; }
    const float4 c = ld4(a.chi + i);
    const float4 n = make_float4(c.x - a.tau * (k.x + div.x), c.y - a.tau * (k.y + div.y), c.z - a.tau * (k.z + div.z), c.w - a.tau * (k.w + div.w));
    const float4 bar = make_float4(n.x + a.theta * (n.x - c.x), n.y + a.theta * (n.y - c.y), n.z + a.theta * (n.z - c.z), n.w + a.theta * (n.w - c.w));
    st4(a.chi + i, n);
    st4(a.chibar + i, bar);
    return bar;
}

__global__ void __launch_bounds__(kThreads) chi_update3_kernel(const VoxArgs a) {
    const long long nquad = a.nvox >> 2;
    for (long long i4 = (long long)blockIdx.x * kThreads + threadIdx.x; i4 < nquad; i4 += (long long)gridDim.x * kThreads) {
        const long long i = i4 << 2;
        const int plane = (int)(i >> (a.lx + a.ly)), vol = a.lz >= 0 ? plane >> a.lz : plane / a.nz;   // nz need not be a power of two
        const int x = (int)(i & (a.nx - 1)), y = (int)((i >> a.lx) & (a.ny - 1)), z = plane - vol * a.nz;
        chi_quad(a, i, x, y, z, ld4(a.kp + i));
    }
}

// W = identity, nx in {64, 128, 256}: the x lines back, the chi-update and the x lines of the NEXT iteration in one
// kernel -- K p never goes to memory and chi_bar is not read back (12 of 118 bytes per voxel and iteration).  The 16 lines
// of the tile come out of the inverse transform in the thread map of fft_regs.cuh; they are laid into shared memory as
// (K p_a, K p_b) rows, the chi-update runs over the rows with coalesced float4 accesses (both volumes of the pair) and
// leaves (chi_bar_a, chi_bar_b) in their place, from where the forward transform picks its points up again.
template <int N>
__global__ void __launch_bounds__(kTL * pdk::FftCfg<N>::T, 1024 / (kTL * pdk::FftCfg<N>::T)) fused_x_kernel(const FftArgs a, const VoxArgs va, const int do_fwd) {
    using Cfg = pdk::FftCfg<N>;
    constexpr int E = Cfg::E, T = Cfg::T, LD = T + 1, NT = kTL * T, REG = E * LD + 1;
    static_assert(kTL * REG >= kTL * N, "the exchange buffer doubles as the tile of rows");
    __shared__ float2 tws[E * T];
    __shared__ float2 ex[kTL * REG];
    pdk::TwiddlesSmem<N>::fill(tws, a.tw, threadIdx.x, NT);
    const int l = threadIdx.x / T, j = threadIdx.x % T;
    pdk::TwiddlesSmem<N> tw;
    tw.w = tws + j;
    float2 *sm = ex + l * REG;
    const long long L0 = (long long)blockIdx.x * kTL;
    const bool live = L0 + l < a.nlines;
    float2 *const zl = a.z + (L0 + l) * N;
    float2 v[E];
#pragma unroll
    for (int m = 0; m < E; ++m) v[m] = live ? zl[j + T * m] : make_float2(0.f, 0.f);
    __syncthreads();   // twiddle table filled
#pragma unroll
    for (int m = 0; m < E; ++m) v[m] = make_float2(v[m].y, v[m].x);   // inverse = forward of the swapped halves
    pdk::fft_line<N, LD>(v, sm, j, tw, pdk::WarpSync());
    __syncthreads();   // every line is through its exchange: the buffer becomes the tile of rows
#pragma unroll
    for (int m = 0; m < E; ++m) ex[l * N + j + T * m] = make_float2(v[m].y * a.out_scale, v[m].x * a.out_scale);
    __syncthreads();
    for (int idx = threadIdx.x; idx < kTL * (N / 4); idx += NT) {
        const int row = idx / (N / 4), x = (idx % (N / 4)) * 4;
        const long long L = L0 + row;
        if (L >= a.nlines) continue;
        const long long pv = L / a.lines_per_vol;
        const int r = (int)(L - pv * a.lines_per_vol), y = r & (va.ny - 1), z = r >> va.ly;
        float2 *t = ex + row * N + x;
        const long long i = (2 * pv) * a.V + (long long)r * N + x;
        const float4 ba = chi_quad(va, i, x, y, z, make_float4(t[0].x, t[1].x, t[2].x, t[3].x));
        float4 bb = make_float4(0.f, 0.f, 0.f, 0.f);
        if (2 * pv + 1 < a.nvol) bb = chi_quad(va, i + a.V, x, y, z, make_float4(t[0].y, t[1].y, t[2].y, t[3].y));
        t[0] = make_float2(ba.x, bb.x); t[1] = make_float2(ba.y, bb.y); t[2] = make_float2(ba.z, bb.z); t[3] = make_float2(ba.w, bb.w);
    }
    if (!do_fwd) return;
    __syncthreads();
#pragma unroll
    for (int m = 0; m < E; ++m) v[m] = ex[l * N + j + T * m];
    __syncthreads();   // the rows have been read: the buffer is the exchange region again
    pdk::fft_line<N, LD>(v, sm, j, tw, pdk::WarpSync());
    if (!live) return;
#pragma unroll
    for (int m = 0; m < E; ++m) zl[j + T * m] = v[m];
}

// Per-volume normalisation (the 2-D path's pair_scale): the iteration is exactly invariant under
// (phi, alpha) -> (c phi, c alpha) with chi -> c chi, and a power of two is exact in floating point, so every volume is
// iterated at c_v = 2^-floor(log2 rms(phi_v)) and the two volumes of a pair meet at the same magnitude.  Two kernels,
// fixed summation order: bitwise repeatable.
constexpr int kScaleParts = 64;
__global__ void __launch_bounds__(kThreads) vol_sumsq_kernel(const float *__restrict__ field, long long V, float *__restrict__ part) {
    const long long chunk = V / kScaleParts, b0 = (long long)blockIdx.y * V + (long long)blockIdx.x * chunk;
    float s = 0.f;
    if ((chunk & 3) == 0) {
        for (long long i = threadIdx.x * 4LL; i < chunk; i += kThreads * 4LL) {
            const float4 f = ld4(field + b0 + i);
            s += f.x * f.x + f.y * f.y + f.z * f.z + f.w * f.w;
        }
    } else {   // an odd number of planes: chunks of 2 nz (nx ny / 128) floats are not 16-byte aligned
        for (long long i = threadIdx.x; i < chunk; i += kThreads) { const float f = field[b0 + i]; s += f * f; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    __shared__ float ws[kThreads / 32];
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        float t = 0.f;
        for (int w = 0; w < kThreads / 32; ++w) t += ws[w];
        part[blockIdx.y * kScaleParts + blockIdx.x] = t;
    }
}
__global__ void vol_scale_kernel(const float *__restrict__ part, long long V, int nvol, float *__restrict__ cscale) {
    const int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= nvol) return;
    float t = 0.f;
    for (int k = 0; k < kScaleParts; ++k) t += part[v * kScaleParts + k];
    const float rms = sqrtf(t / (float)V);
    const float c = (rms > 0.f && rms < 3.0e38f) ? scalbnf(1.0f, -ilogbf(rms)) : 1.0f;
    cscale[v] = c;
    cscale[nvol + v] = t > 0.f ? 1.0f / c : 0.f;   // factor of the final store; a zero field returns chi = 0 exactly (R13b),
                                                   // whatever rounding noise its pair partner left in its lane
}
// chi <- chi / c_v at the end (exact)
__global__ void __launch_bounds__(kThreads) vol_unscale_kernel(float *__restrict__ chi, long long nvox, int lxy, int nz, const float *__restrict__ rscale) {
    for (long long i4 = (long long)blockIdx.x * kThreads + threadIdx.x; i4 < (nvox >> 2); i4 += (long long)gridDim.x * kThreads) {
        const long long i = i4 << 2;
        const float r = rscale[(int)(i >> lxy) / nz];
        float4 c = ld4(chi + i);
        c.x *= r; c.y *= r; c.z *= r; c.w *= r;
        st4(chi + i, c);
    }
}

bool pow2_in(int n, int lo, int hi) { return n >= lo && n <= hi && (n & (n - 1)) == 0; }

template <int N, bool STRIDED>
void launch_reg(dim3 grid, const FftArgs &a, int mode, cudaStream_t st) {
    constexpr int NT = kTL * pdk::FftCfg<N>::T;
    if constexpr (STRIDED) {
        if (mode == kModeDual) fft_lines_reg_kernel<N, STRIDED, kModeDual><<<grid, NT, 0, st>>>(a);
        else if (mode == kModeMulD) fft_lines_reg_kernel<N, STRIDED, kModeMulD><<<grid, NT, 0, st>>>(a);
        else if (mode == kModeStoreSpectrum) fft_lines_reg_kernel<N, STRIDED, kModeStoreSpectrum><<<grid, NT, 0, st>>>(a);
        else fft_lines_reg_kernel<N, STRIDED, kModePlain><<<grid, NT, 0, st>>>(a);
    } else {
        if (mode == kModeInReal) fft_lines_reg_kernel<N, STRIDED, kModeInReal><<<grid, NT, 0, st>>>(a);
        else if (mode == kModeInRealScaled) fft_lines_reg_kernel<N, STRIDED, kModeInRealScaled><<<grid, NT, 0, st>>>(a);
        else if (mode == kModeOutReal) fft_lines_reg_kernel<N, STRIDED, kModeOutReal><<<grid, NT, 0, st>>>(a);
        else fft_lines_reg_kernel<N, STRIDED, kModePlain><<<grid, NT, 0, st>>>(a);
    }
}

template <bool STRIDED>
void launch_fft(int n, dim3 grid, const FftArgs &a, int mode, cudaStream_t st) {
    switch (n) {
        case 8: fft_lines_kernel<8, STRIDED><<<grid, kThreads, 0, st>>>(a, mode); break;
        case 16: fft_lines_kernel<16, STRIDED><<<grid, kThreads, 0, st>>>(a, mode); break;
        case 32: fft_lines_kernel<32, STRIDED><<<grid, kThreads, 0, st>>>(a, mode); break;
        case 64: launch_reg<64, STRIDED>(grid, a, mode, st); break;
        case 128: launch_reg<128, STRIDED>(grid, a, mode, st); break;
        default: launch_reg<256, STRIDED>(grid, a, mode, st); break;
    }
}

}  // namespace

struct pd_plan3d_s {
    int nx, ny, nz, nvol, b0_axis, num_sms;
    float lambda, sigma, tau, theta;
    float *D, *chibar, *kp, *q;     // q: three volumes
    float *cscale, *spart;          // [nvol] normalisation, [nvol][kScaleParts] partial sums
    const float *weight;            // caller-owned W or NULL (identity)
    float *pimg;                    // literal path: p and W p, two volumes (allocated by pd_set_weight3d)
    float2 *tw[3], *z, *phihat, *phat;
    int last_launches;
};

extern "C" {

int pd_destroy3d(pd_plan3d_t p) {
    if (!p) return PD_EINVAL;
    void *ptrs[] = {p->D, p->chibar, p->kp, p->q, p->tw[0], p->tw[1], p->tw[2], p->z, p->phihat, p->phat, p->cscale, p->spart, p->pimg};
    for (void *q : ptrs)
        if (q) cudaFree(q);
    delete p;
    return PD_OK;
}

int pd_plan3d(pd_plan3d_t *out, int nx, int ny, int nz, int nvol, int B0_axis, float lambda, float sigma, float tau, float theta) {
    if (!out) return PD_EINVAL;
    *out = nullptr;
    if (nvol < 1 || B0_axis < 0 || B0_axis > 2) return PD_EINVAL;
    if (!pow2_in(nx, 16, 256) || !pow2_in(ny, 8, 256) || !(pow2_in(nz, 8, 256) || (nz >= 2 && nz <= kDenseMax))) return PD_ESIZE;
    if ((long long)((nvol + 1) / 2) * nz > 65535) return PD_ESIZE;   // the y passes put (pair, z) on gridDim.y
    if (!(lambda >= 0.f) || !(theta >= 0.f && theta <= 1.f) || std::isnan(sigma) || std::isnan(tau)) return PD_EINVAL;
    const double bound = 4.0 / 9.0 + 12.0;   // ||K||^2 <= 4/9, ||G||^2 <= 12 in three dimensions (tau = sigma = 1/L)
    if (!(sigma > 0.f) || !(tau > 0.f)) sigma = tau = (float)(1.0 / std::sqrt(bound));
    else if ((double)sigma * (double)tau * bound >= 1.0) return PD_ESTEP;
    pd_plan3d_s *p = new (std::nothrow) pd_plan3d_s;
    if (!p) return PD_ENOMEM;
    std::memset(p, 0, sizeof(*p));
    p->nx = nx; p->ny = ny; p->nz = nz; p->nvol = nvol; p->b0_axis = B0_axis;
    p->lambda = lambda; p->sigma = sigma; p->tau = tau; p->theta = theta;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&p->num_sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) { delete p; return pd_cuda_fail_((int)e, "cudaGetDevice"); }
    const size_t V = (size_t)nx * ny * nz, T = V * (size_t)nvol;
    const int dims[3] = {nx, ny, nz};
    auto alloc = [&](void **ptr, size_t bytes) {
        if (e != cudaSuccess) return;
        e = cudaMalloc(ptr, bytes);
    };
    alloc((void **)&p->D, V * sizeof(float));
    alloc((void **)&p->chibar, T * sizeof(float));
    alloc((void **)&p->kp, T * sizeof(float));
    alloc((void **)&p->q, 3 * T * sizeof(float));
    alloc((void **)&p->cscale, 2 * (size_t)nvol * sizeof(float));   // c_v, then the factors of the final store
    alloc((void **)&p->spart, (size_t)nvol * kScaleParts * sizeof(float));
    const size_t TP = V * (size_t)((nvol + 1) / 2);   // complex volumes: two real volumes ride one complex transform
    alloc((void **)&p->z, TP * sizeof(float2));
    alloc((void **)&p->phihat, TP * sizeof(float2));
    alloc((void **)&p->phat, TP * sizeof(float2));
    for (int k = 0; k < 3; ++k) alloc((void **)&p->tw[k], (size_t)dims[k] * sizeof(float2));
    if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); pd_destroy3d(p); return PD_ENOMEM; }
    if (e != cudaSuccess) { pd_destroy3d(p); return pd_cuda_fail_((int)e, "cudaMalloc"); }
    {   // tables in double on the host (R17): D3 = 1/3 - k_b^2/|k|^2, D3(0) = 0, k = (fi/nx, fj/ny, fk/nz) signed (R23)
        std::vector<float> D(V);
        for (int kz = 0; kz < nz; ++kz) {
            const double fz = (double)(kz < (nz + 1) / 2 ? kz : kz - nz) / nz;
            for (int ky = 0; ky < ny; ++ky) {
                const double fy = (double)(ky < (ny + 1) / 2 ? ky : ky - ny) / ny;
                for (int kx = 0; kx < nx; ++kx) {
                    const double fx = (double)(kx < (nx + 1) / 2 ? kx : kx - nx) / nx;
                    const double k2 = fx * fx + fy * fy + fz * fz, kb = B0_axis == 0 ? fx : B0_axis == 1 ? fy : fz;
                    D[((size_t)kz * ny + ky) * nx + kx] = (float)(k2 == 0.0 ? 0.0 : 1.0 / 3.0 - kb * kb / k2);
                }
            }
        }
        e = cudaMemcpy(p->D, D.data(), V * sizeof(float), cudaMemcpyHostToDevice);
        const double pi = 3.14159265358979323846264338327950288;
        for (int k = 0; k < 3 && e == cudaSuccess; ++k) {
            std::vector<float2> tw(dims[k]);
            for (int j = 0; j < dims[k]; ++j) {
                const double ang = -2.0 * pi * (double)j / (double)dims[k];
                tw[j] = make_float2((float)std::cos(ang), (float)std::sin(ang));
            }
            e = cudaMemcpy(p->tw[k], tw.data(), tw.size() * sizeof(float2), cudaMemcpyHostToDevice);
        }
        if (e == cudaSuccess) e = cudaStreamSynchronize(nullptr);
        if (e != cudaSuccess) { pd_destroy3d(p); return pd_cuda_fail_((int)e, "3-D plan table upload"); }
    }
    *out = p;
    return PD_OK;
}

int pd_solve3d(pd_plan3d_t p, const float *field, const float *mask, float *chi_out, int max_iters, void *cuda_stream) {
    if (!p || !field || !chi_out || max_iters < 0) return PD_EINVAL;
    if (((unsigned long long)field | (unsigned long long)mask | (unsigned long long)chi_out) & 15ull) return PD_EINVAL;   // float4 accesses
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int nx = p->nx, ny = p->ny, nz = p->nz, nvol = p->nvol;
    const long long V = (long long)nx * ny * nz, T = V * nvol;
    const int npairs = (nvol + 1) / 2;
    cudaError_t e = cudaMemsetAsync(p->phat, 0, V * npairs * sizeof(float2), st);
    if (e == cudaSuccess) e = cudaMemsetAsync(p->q, 0, 3 * T * sizeof(float), st);
    if (e == cudaSuccess) e = cudaMemsetAsync(p->chibar, 0, T * sizeof(float), st);
    if (e == cudaSuccess) e = cudaMemsetAsync(chi_out, 0, T * sizeof(float), st);
    if (e != cudaSuccess) return pd_cuda_fail_((int)e, "cudaMemsetAsync (3-D state)");

    FftArgs f;
    std::memset(&f, 0, sizeof(f));
    f.z = p->z; f.phihat = p->phihat; f.phat = p->phat; f.D = p->D;
    f.sigma = p->sigma; f.inv1ps = 1.0f / (1.0f + p->sigma); f.out_scale = (float)(1.0 / (double)V);
    f.V = V; f.lines_per_vol = nz * ny; f.nvol = nvol;
    const long long xlines = (long long)npairs * nz * ny;
    const dim3 gx((unsigned)((xlines + kTL - 1) / kTL)), gy((unsigned)(nx / kTL), (unsigned)(npairs * nz)),
        gz((unsigned)((long long)nx * ny / kTL), (unsigned)npairs);
    int launches = 0;
    auto pass_x = [&](const float *in_real, float *out_real, bool inverse) {
        FftArgs a = f;
        a.tw = p->tw[0]; a.nlines = xlines; a.inverse = inverse ? 1 : 0; a.in_real = in_real; a.out_real = out_real;
        launch_fft<false>(nx, gx, a, in_real ? (a.cscale ? kModeInRealScaled : kModeInReal) : out_real ? kModeOutReal : kModePlain, st);
        ++launches;
    };
    auto pass_y = [&](bool inverse) {
        FftArgs a = f;
        a.tw = p->tw[1]; a.S = nx; a.inverse = inverse ? 1 : 0;
        launch_fft<true>(ny, gy, a, kModePlain, st);
        ++launches;
    };
    auto pass_z = [&](int mode) {
        FftArgs a = f;
        a.tw = p->tw[2]; a.S = (long long)nx * ny; a.inverse = 0;
        if (pow2_in(nz, 8, 256)) launch_fft<true>(nz, gz, a, mode, st);
        else dft_lines_dense_kernel<<<gz, kThreads, 0, st>>>(a, mode, nz);   // any other slice count up to 64
        ++launches;
    };
    // per-volume normalisation, then phi^ = F (c phi), once (everything else starts at zero)
    vol_sumsq_kernel<<<dim3(kScaleParts, (unsigned)nvol), kThreads, 0, st>>>(field, V, p->spart);
    vol_scale_kernel<<<(nvol + 63) / 64, 64, 0, st>>>(p->spart, V, nvol, p->cscale);
    launches += 2;
    f.cscale = p->cscale;
    pass_x(field, nullptr, false);
    f.cscale = nullptr;
    pass_y(false);
    pass_z(kModeStoreSpectrum);

    VoxArgs v;
    std::memset(&v, 0, sizeof(v));
    v.nx = nx; v.ny = ny; v.nz = nz; v.nvox = T; v.mask = mask;
    for (v.lx = 0; (1 << v.lx) < nx; ++v.lx) {}
    for (v.ly = 0; (1 << v.ly) < ny; ++v.ly) {}
    for (v.lv = 0; (1LL << v.lv) < V; ++v.lv) {}
    v.lz = -1;
    for (int b = 0; b < 9; ++b) if ((1 << b) == nz) v.lz = b;
    v.cscale = p->cscale;
    v.chi = chi_out; v.chibar = p->chibar; v.qx = p->q; v.qy = p->q + T; v.qz = p->q + 2 * T; v.kp = p->kp;
    v.sigma = p->sigma; v.tau = p->tau; v.theta = p->theta; v.alpha = p->lambda;
    const long long need = (T / 4 + kThreads - 1) / kThreads, cap = (long long)p->num_sms * 8;
    const int vgrid = (int)(need < cap ? need : cap);
    const bool literal = p->weight != nullptr;   // W set: p stays in the image domain and K is applied twice (PAPER.md:49 literally)
    if (literal) {
        v.weight = p->weight; v.field = field; v.p = p->pimg; v.wp = p->pimg + T; v.inv1ps = 1.0f / (1.0f + p->sigma);
        e = cudaMemsetAsync(p->pimg, 0, T * sizeof(float), st);
        if (e != cudaSuccess) return pd_cuda_fail_((int)e, "cudaMemsetAsync (3-D dual)");
    }
    const bool fused = !literal && nx >= 64;      // the chi-update rides the x passes (fused_x_kernel)
    for (int n = 0; n < max_iters; ++n) {
        if (fused) {   // the q-update needs chi_bar_n, which the fused kernel at the end of the iteration overwrites
            q_update3_kernel<<<vgrid, kThreads, 0, st>>>(v);
            ++launches;
        }
        if (!fused || n == 0) pass_x(p->chibar, nullptr, false);     // F chi_bar
        pass_y(false);
        if (!literal) {
            pass_z(kModeDual);                 // p-update in the Fourier domain, spectrum of K p, z lines back
        } else {
            pass_z(kModeMulD);                 // K chi_bar ...
            pass_y(true);
            pass_x(nullptr, p->kp, true);
            q_update3_kernel<<<vgrid, kThreads, 0, st>>>(v);   // ... q-update and p-update, W p ...
            ++launches;
            pass_x(v.wp, nullptr, false);      // ... and K (W p)
            pass_y(false);
            pass_z(kModeMulD);
        }
        pass_y(true);
        if (fused) {   // x lines back + chi-update + x lines of the next iteration
            FftArgs a = f;
            a.tw = p->tw[0]; a.nlines = xlines;
            const int fwd = n + 1 < max_iters ? 1 : 0;
            if (nx == 64) fused_x_kernel<64><<<gx, kTL * pdk::FftCfg<64>::T, 0, st>>>(a, v, fwd);
            else if (nx == 128) fused_x_kernel<128><<<gx, kTL * pdk::FftCfg<128>::T, 0, st>>>(a, v, fwd);
            else fused_x_kernel<256><<<gx, kTL * pdk::FftCfg<256>::T, 0, st>>>(a, v, fwd);
            ++launches;
            continue;
        }
        pass_x(nullptr, p->kp, true);          // K p
        if (!literal) {
            q_update3_kernel<<<vgrid, kThreads, 0, st>>>(v);
            ++launches;
        }
        chi_update3_kernel<<<vgrid, kThreads, 0, st>>>(v);
        ++launches;
    }
    if (max_iters > 0) {
        vol_unscale_kernel<<<vgrid, kThreads, 0, st>>>(chi_out, T, v.lx + v.ly, nz, p->cscale + nvol);
        ++launches;
    }
    p->last_launches = launches;
    e = cudaGetLastError();
    return e == cudaSuccess ? PD_OK : pd_cuda_fail_((int)e, "pd_solve3d launch");
}

int pd_set_weight3d(pd_plan3d_t p, const float *W) {
    if (!p || ((unsigned long long)W & 15ull)) return PD_EINVAL;
    if (W && !p->pimg) {   // workspace of the literal path: p and W p
        const size_t T = (size_t)p->nx * p->ny * p->nz * (size_t)p->nvol;
        const cudaError_t e = cudaMalloc((void **)&p->pimg, 2 * T * sizeof(float));
        if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); p->pimg = nullptr; return PD_ENOMEM; }
        if (e != cudaSuccess) return pd_cuda_fail_((int)e, "cudaMalloc");
    }
    p->weight = W;
    return PD_OK;
}

int pd_last_launch_count3d(pd_plan3d_t p) { return p ? p->last_launches : PD_EINVAL; }

}  // extern "C"
