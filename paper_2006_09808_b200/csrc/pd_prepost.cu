// pd_prepost.cu -- the steps either side of the iteration: pd_preprocess (flow step (1),
// field map, weighting matrix W and Mask from the two echo-shifted complex volumes; R20, R21)
// and pd_combine_coils (one susceptibility map per slice from the per-coil maps; R22).  Elementwise,
// HBM-bound: 16-byte accesses, four pixels per thread and trip, grid-stride over a grid of a few CTAs per SM.
// Where floating point decides an integer (the mask, the stack maximum behind the scale of W) the arithmetic is a fixed
// sequence of correctly rounded fp32 operations (__fmul_rn / __fadd_rn / __fsqrt_rn / __fdiv_rn: no contraction into
// FMAs), so that the decision is reproducible bit for bit by anybody who follows the same sequence.
#include "../../include/pd.h"

#include <cuda_runtime.h>

int pd_cuda_fail_(int cuda_error, const char *where);   // pd_api.cu: records the text behind PD_ECUDA

namespace {

constexpr int kThreads = 256;
constexpr int kCtasPerSm = 8;

// m = (|s0|^2 |s1|^2)^(1/4) = sqrt(|s0| |s1|), every step rounded to nearest (R21)
__device__ __forceinline__ float magnitude_rn(float r0, float i0, float r1, float i1) {
    const float a0 = __fadd_rn(__fmul_rn(r0, r0), __fmul_rn(i0, i0));
    const float a1 = __fadd_rn(__fmul_rn(r1, r1), __fmul_rn(i1, i1));
    return __fsqrt_rn(__fsqrt_rn(__fmul_rn(a0, a1)));
}

__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// pass 1 (automatic scale only): max of m over the whole stack.  m >= 0, so the unsigned order of the bit patterns is
// the order of the values and an integer atomicMax is exact and order-independent.
__global__ void __launch_bounds__(kThreads) pre_max_kernel(const float4 *__restrict__ s0, const float4 *__restrict__ s1,
                                                            long long npix, float *__restrict__ wmax) {
    const long long nvec = npix / 2;   // float4 = two complex pixels
    float mx = 0.f;
    for (long long i = (long long)blockIdx.x * kThreads + threadIdx.x; i < nvec; i += (long long)gridDim.x * kThreads) {
        const float4 a = __ldg(s0 + i), b = __ldg(s1 + i);
        mx = fmaxf(mx, fmaxf(magnitude_rn(a.x, a.y, b.x, b.y), magnitude_rn(a.z, a.w, b.z, b.w)));
    }
    if ((npix & 1) && blockIdx.x == 0 && threadIdx.x == 0) {   // odd pixel count: the last pixel
        const float2 a = reinterpret_cast<const float2 *>(s0)[npix - 1], b = reinterpret_cast<const float2 *>(s1)[npix - 1];
        mx = fmaxf(mx, magnitude_rn(a.x, a.y, b.x, b.y));
    }
    mx = warp_max(mx);
    __shared__ float part[kThreads / 32];
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = mx;
    __syncthreads();
    if (threadIdx.x < 32) {
        mx = warp_max(threadIdx.x < kThreads / 32 ? part[threadIdx.x] : 0.f);
        if (threadIdx.x == 0) atomicMax(reinterpret_cast<unsigned *>(wmax), __float_as_uint(mx));
    }
}

struct PreOut { float f, w, m; };

__device__ __forceinline__ PreOut pre_pixel(float r0, float i0, float r1, float i1, float fscale, float winv, float thr) {
    // s1 * conj(s0); its argument is the phase the echo shift added (R20); a zero product has no phase: field 0
    const float re = fmaf(r1, r0, i1 * i0), im = fmaf(i1, r0, -(r1 * i0));
    PreOut o;
    o.f = (re == 0.f && im == 0.f) ? 0.f : atan2f(im, re) * fscale;
    o.w = __fmul_rn(magnitude_rn(r0, i0, r1, i1), winv);
    o.m = o.w > thr ? 1.f : 0.f;
    return o;
}

// pass 2: four pixels per thread and trip (two float4 of each echo in, one float4 of each output out)
__global__ void __launch_bounds__(kThreads) pre_kernel(const float4 *__restrict__ s0, const float4 *__restrict__ s1, long long npix,
                                                        float fscale, float wscale, float thr, const float *__restrict__ wmax,
                                                        float *__restrict__ field, float *__restrict__ weight, float *__restrict__ mask) {
    float winv = wscale;
    if (!(wscale > 0.f)) {
        const float mx = *wmax;
        winv = mx > 0.f ? __fdiv_rn(1.0f, mx) : 0.f;
    }
    const long long nquad = npix / 4;
    for (long long i = (long long)blockIdx.x * kThreads + threadIdx.x; i < nquad; i += (long long)gridDim.x * kThreads) {
        const float4 a0 = __ldg(s0 + 2 * i), a1 = __ldg(s0 + 2 * i + 1), b0 = __ldg(s1 + 2 * i), b1 = __ldg(s1 + 2 * i + 1);
        const PreOut p0 = pre_pixel(a0.x, a0.y, b0.x, b0.y, fscale, winv, thr), p1 = pre_pixel(a0.z, a0.w, b0.z, b0.w, fscale, winv, thr);
        const PreOut p2 = pre_pixel(a1.x, a1.y, b1.x, b1.y, fscale, winv, thr), p3 = pre_pixel(a1.z, a1.w, b1.z, b1.w, fscale, winv, thr);
        if (field) reinterpret_cast<float4 *>(field)[i] = make_float4(p0.f, p1.f, p2.f, p3.f);
        if (weight) reinterpret_cast<float4 *>(weight)[i] = make_float4(p0.w, p1.w, p2.w, p3.w);
        if (mask) reinterpret_cast<float4 *>(mask)[i] = make_float4(p0.m, p1.m, p2.m, p3.m);
    }
    if (blockIdx.x == 0 && threadIdx.x < (int)(npix & 3)) {   // ragged tail: up to three pixels
        const long long k = 4 * nquad + threadIdx.x;
        const float2 a = reinterpret_cast<const float2 *>(s0)[k], b = reinterpret_cast<const float2 *>(s1)[k];
        const PreOut p = pre_pixel(a.x, a.y, b.x, b.y, fscale, winv, thr);
        if (field) field[k] = p.f;
        if (weight) weight[k] = p.w;
        if (mask) mask[k] = p.m;
    }
}

// chi(x) = sum_c W_c^2 chi_c / sum_c W_c^2, coils in the order c = 0 .. ncoils-1, 0 where no coil sees the pixel (R22).
// VEC = 4: pixels per thread (P a multiple of 4); VEC = 1: any P.
template <int VEC>
__global__ void __launch_bounds__(kThreads) combine_kernel(const float *__restrict__ chi, const float *__restrict__ wgt, int nslices,
                                                            int ncoils, long long P, float *__restrict__ out) {
    const long long per = P / VEC, total = (long long)nslices * per;
    for (long long i = (long long)blockIdx.x * kThreads + threadIdx.x; i < total; i += (long long)gridDim.x * kThreads) {
        const long long s = i / per, q = (i - s * per) * VEC;
        const float *c0 = chi + (s * ncoils) * P + q, *w0 = wgt + (s * ncoils) * P + q;
        float num[VEC], den[VEC];
#pragma unroll
        for (int v = 0; v < VEC; ++v) num[v] = den[v] = 0.f;
        for (int c = 0; c < ncoils; ++c) {
            float x[VEC], w[VEC];
            if (VEC == 4) {
                const float4 xv = __ldg(reinterpret_cast<const float4 *>(c0 + (long long)c * P));
                const float4 wv = __ldg(reinterpret_cast<const float4 *>(w0 + (long long)c * P));
                x[0] = xv.x; x[VEC > 1 ? 1 : 0] = xv.y; x[VEC > 2 ? 2 : 0] = xv.z; x[VEC > 3 ? 3 : 0] = xv.w;
                w[0] = wv.x; w[VEC > 1 ? 1 : 0] = wv.y; w[VEC > 2 ? 2 : 0] = wv.z; w[VEC > 3 ? 3 : 0] = wv.w;
            } else {
                x[0] = __ldg(c0 + (long long)c * P);
                w[0] = __ldg(w0 + (long long)c * P);
            }
#pragma unroll
            for (int v = 0; v < VEC; ++v) {
                const float w2 = w[v] * w[v];
                num[v] = fmaf(w2, x[v], num[v]);
                den[v] += w2;
            }
        }
        float r[VEC];
#pragma unroll
        for (int v = 0; v < VEC; ++v) r[v] = den[v] > 0.f ? __fdiv_rn(num[v], den[v]) : 0.f;
        if (VEC == 4) reinterpret_cast<float4 *>(out + s * P + q)[0] = make_float4(r[0], r[VEC > 1 ? 1 : 0], r[VEC > 2 ? 2 : 0], r[VEC > 3 ? 3 : 0]);
        else out[s * P + q] = r[0];
    }
}

int grid_for(long long items, int *grid) {
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return pd_cuda_fail_((int)e, "cudaGetDevice");
    const long long need = (items + kThreads - 1) / kThreads, cap = (long long)sms * kCtasPerSm;   // whole waves of the SMs
    *grid = (int)(need < 1 ? 1 : need < cap ? need : cap);
    return PD_OK;
}

bool aligned16(const void *p) { return (reinterpret_cast<unsigned long long>(p) & 15ull) == 0; }

}  // namespace

extern "C" {

int pd_preprocess(const float *s0, const float *s1, long long npixels, float fscale, float wscale, float threshold,
                  float *field, float *weight, float *mask, float *wmax, void *cuda_stream) {
    if (!s0 || !s1 || npixels < 0 || !(fscale == fscale) || !(threshold == threshold)) return PD_EINVAL;
    if (!(wscale > 0.f) && !wmax) return PD_EINVAL;   // the automatic scale needs its one float of device memory
    if (!aligned16(s0) || !aligned16(s1) || !aligned16(field) || !aligned16(weight) || !aligned16(mask)) return PD_EINVAL;
    if (npixels == 0) return PD_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int grid = 1, rc;
    if (!(wscale > 0.f)) {
        cudaError_t e = cudaMemsetAsync(wmax, 0, sizeof(float), st);
        if (e != cudaSuccess) return pd_cuda_fail_((int)e, "cudaMemsetAsync(wmax)");
        if ((rc = grid_for(npixels / 2, &grid)) != PD_OK) return rc;
        pre_max_kernel<<<grid, kThreads, 0, st>>>(reinterpret_cast<const float4 *>(s0), reinterpret_cast<const float4 *>(s1), npixels, wmax);
    }
    if (field || weight || mask) {
        if ((rc = grid_for(npixels / 4, &grid)) != PD_OK) return rc;
        pre_kernel<<<grid, kThreads, 0, st>>>(reinterpret_cast<const float4 *>(s0), reinterpret_cast<const float4 *>(s1), npixels, fscale,
                                              wscale, threshold, wmax, field, weight, mask);
    }
    const cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? PD_OK : pd_cuda_fail_((int)e, "pd_preprocess launch");
}

int pd_combine_coils(const float *chi, const float *weight, int nslices, int ncoils, int ny, int nx, float *chi_out,
                     void *cuda_stream) {
    if (!chi || !weight || !chi_out || nslices < 0 || ncoils < 1 || ny < 1 || nx < 1) return PD_EINVAL;
    if (nslices == 0) return PD_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const long long P = (long long)ny * nx;
    const bool vec = (P % 4 == 0) && aligned16(chi) && aligned16(weight) && aligned16(chi_out);
    int grid = 1, rc;
    if ((rc = grid_for((long long)nslices * (vec ? P / 4 : P), &grid)) != PD_OK) return rc;
    if (vec) combine_kernel<4><<<grid, kThreads, 0, st>>>(chi, weight, nslices, ncoils, P, chi_out);
    else combine_kernel<1><<<grid, kThreads, 0, st>>>(chi, weight, nslices, ncoils, P, chi_out);
    const cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? PD_OK : pd_cuda_fail_((int)e, "pd_combine_coils launch");
}

}  // extern "C"
