// pd_api.cu -- host side of the C ABI declared in include/pd.h: plan construction (dipole table, twiddle
// tables, workspace), launch sequencing of the PD iteration on a caller-provided stream.
// No CPU fallback exists: every arithmetic step of the path runs in the kernels of pd_resident*.cuh / pd_streaming_fd.cuh.
#include "../../include/pd.h"
#include "pd_resident.cuh"
#include "pd_resident_tm.cuh"
#include "pd_streaming_fd.cuh"
#include "pd_streaming_gen.cuh"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

using pdk::ResidentArgs;
using pdk::ResidentTmArgs;
using pdk::StreamFdArgs;

namespace {

thread_local char g_cuda_err[256] = "no CUDA error recorded";

int cuda_fail(cudaError_t e, const char *where) {
    snprintf(g_cuda_err, sizeof(g_cuda_err), "CUDA error at %s: %s", where, cudaGetErrorString(e));
    return PD_ECUDA;
}
#define PD_CUDA(call)                                          \
    do {                                                       \
        cudaError_t e_ = (call);                               \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call);    \
    } while (0)

bool size_ok(int n) { return n == 64 || n == 128 || n == 256 || n == 512; }
// sizes of the general-length streaming kernels (pd_streaming_gen.cuh): any even length; the paper's are 258 and 132
bool gen_size_ok(int n) { return n >= 4 && n <= 1024 && (n % 2) == 0; }
// most balanced factorisation n = n1 * n2, n1 <= n2 (n1 = 1 for a prime: one dense stage)
void balanced_factors(int n, int *n1, int *n2) {
    int best = 1;
    for (int f = 1; f * f <= n; ++f)
        if (n % f == 0) best = f;
    *n1 = best;
    *n2 = n / best;
}

// ||K_full||^2 <= max|W|^2 max|D|^2 + max|M|^2 ||G||^2 = 4/9 w^2 + 8 m^2 (R14); w = m = 1 unless pd_set_norm_bounds says otherwise
double norm_bound(double w, double m) { return 4.0 / 9.0 * w * w + 8.0 * m * m; }

}  // namespace

// for the other translation units of the library (pd_prepost.cu): record the text behind PD_ECUDA
int pd_cuda_fail_(int cuda_error, const char *where) { return cuda_fail((cudaError_t)cuda_error, where); }

constexpr int kGraphSlots = 8, kMaxChunks = 6;

struct pd_plan_s {
    int nx, ny, batch, npairs, b0_dir;
    // user-facing parameters (as given) and the effective ones of the rescaled problem (R2)
    float lambda_user, sigma_user, tau_user, theta;
    int tv_mode, lambda_conv, variant, check_every, mask_shared, unsafe_steps, no_fd;
    int generic;           // a size that is not a power of two: general-length kernels (pd_streaming_gen.cuh), literal iteration
    pdk::GenDims gdims;
    int host_chunking;     // PD_OPT_HOST_CHUNKING: 0 automatic, 1 always, 2 never
    int reg_l1;            // PD_OPT_REGULARISER = PD_REG_L1
    double max_w, max_m;   // bounds on |W| and |M| behind the automatic steps and the PD_ESTEP check (pd_set_norm_bounds; 1, 1)
    int use_angle;         // oblique in-plane B0 (pd_set_b0_angle)
    double b0_angle;
    const float *weight;
    // device tables and workspace
    float *Dtab;
    float2 *tw_row, *tw_col;
    int *stop_iter, *iters_done;
    float *P0, *relgap, *relres;
    float *cscale;         // [batch] power-of-two normalisation of every slice (streaming variant; pair_scale)
    int nparts;
    // resident variant (pd_resident.cuh): per-cluster scratch, kResidentScratchArrays arrays of nx*ny float2 per cluster
    int res_ok;            // this size has a resident kernel
    int res_clusters;      // clusters launched (= scratch slots)
    int res_max_clusters;  // what the occupancy query allows
    int num_sms;
    int res_csize;         // CTAs per cluster
    float2 *res_scratch;   // [kResidentScratchArrays][res_clusters][nx*ny]
    float *rk_part;        // [res_clusters][res_csize][8]
    float *Dpriv;          // D/(nx*ny) in the thread-private order of the Fourier-domain-dual kernel (pd_resident_tm.cuh)
    // streaming variant with the Fourier-domain dual (pd_streaming_fd.cuh): allocated on first use
    float2 *sfd_planes;    // 11 arrays of [npairs][ny][nx] float2
    float *sfd_parts;      // per-CTA partial sums
    int sfd_ncolparts, sfd_nrowparts;
    size_t sfd_pairs_alloc; // slice pairs the Fourier-domain streaming workspace holds
    // hybrid schedule (256x256, W = I, PD_VARIANT_AUTO): the resident clusters cover 120 of the 148 SMs; the last
    // `tail` slice pairs run through the streaming kernels on a second stream, on the SMs the clusters leave free
    int hybrid_tail;       // -1: automatic ; >= 0: slice pairs given to the streaming kernels
    double hybrid_rho;     // streaming pairs per resident pair and cluster, measured at plan time (calibrate_hybrid)
    cudaStream_t aux;
    // graphed streaming loop (PD_OPT_GRAPH_LOOP, default on): init -> WHILE { iteration kernels, loop control } -> finish,
    // one cached executable graph per use (slot 0: whole-batch streaming solve; slot 1: tail of the hybrid schedule)
    int graph_loop;
    cudaStream_t cap_stream;
    struct GraphSlot {
        cudaGraphExec_t exec;
        cudaGraph_t graph;
        StreamFdArgs key;     // the arguments the graph was built for
        int key_valid;
        int literal;          // built for the literal (four-kernel) iteration
        int *iter;            // device iteration counter
    } gslot[kGraphSlots];      // executable graphs cached by their arguments (whole batch, hybrid tail, chunks of pd_solve_host)
    int gslot_next;            // round-robin replacement
    unsigned graph_used;       // bit k: slot k was launched by the last pd_solve / pd_solve_host
    // pd_solve_host pipeline: copies on their own streams, one event pair per chunk
    cudaStream_t h2d_stream, d2h_stream;
    cudaEvent_t ev_chunk[2 * kMaxChunks + 2];
    cudaEvent_t ev_fork, ev_join;
    // host-buffer entry point staging
    float *h_field, *h_mask, *h_chi;
    int last_launches;
    int device;
    // optional per-kernel-class device timing (PD_OPT_KERNEL_TIMING): events around every launch of the last solve
    int timing;
    std::vector<cudaEvent_t> *ev;      // pool, two per launch
    std::vector<int> *ev_class;        // kernel class of launch i
};

namespace {

template <typename T>
int dev_alloc(T **ptr, size_t count) {
    cudaError_t e = cudaMalloc((void **)ptr, count * sizeof(T));
    if (e == cudaErrorMemoryAllocation) {
        cudaGetLastError();
        *ptr = nullptr;
        return PD_ENOMEM;
    }
    if (e != cudaSuccess) return cuda_fail(e, "cudaMalloc");
    return PD_OK;
}

int check_params(float lambda, float sigma, float tau, float theta, bool unsafe, double bound) {
    if (!(lambda >= 0.f) || !(theta >= 0.f && theta <= 1.f) || std::isnan(sigma) || std::isnan(tau)) return PD_EINVAL;
    if (sigma > 0.f && tau > 0.f && !unsafe && (double)sigma * (double)tau * bound >= 1.0) return PD_ESTEP;
    return PD_OK;
}

// Effective (alpha, sigma, tau) of the problem the kernels iterate (convention B); convention A is the exact
// rescaling A(lambda, sigma, tau) == B(1/lambda, sigma/lambda, tau*lambda) (R2, oracle pin P9).
void effective_params(const pd_plan_s *p, float *alpha, float *sigma, float *tau) {
    float s = p->sigma_user, t = p->tau_user;
    if (!(s > 0.f) || !(t > 0.f)) s = t = (float)(1.0 / std::sqrt(norm_bound(p->max_w, p->max_m)));
    if (p->lambda_conv == PD_LAMBDA_DATA) {
        *alpha = 1.0f / p->lambda_user;
        *sigma = s / p->lambda_user;
        *tau = t * p->lambda_user;
    } else {
        *alpha = p->lambda_user;
        *sigma = s;
        *tau = t;
    }
}

void build_dipole(std::vector<float> &D, int nx, int ny, int b0_dir, bool use_angle = false, double angle = 0.0) {
    // D(kx,ky) = 1/3 - k_b^2/(kx^2+ky^2), D(0,0)=0, kx = fi/nx, ky = fj/ny (BASELINE.json north_star; R6);
    // the 1/(nx*ny) of the inverse transform is folded in.  k_b = ky (PD_B0_Y), kx (PD_B0_X), or k . (cos a, sin a) for an
    // oblique in-plane B0 (pd_set_b0_angle).  K is defined as the REAL part of F^-1 D F (R12), i.e. only the even part of D
    // acts on a real image; for an oblique B0 the table is not even on the Nyquist lines (index n/2 stands for -n/2), so
    // the even part (D(k) + D(-k))/2 is what is stored -- which is also what lets two real slices ride one complex
    // transform.
    const double scale = 1.0 / ((double)nx * (double)ny);
    const double bx = std::cos(angle), by = std::sin(angle);
    std::vector<double> d2((size_t)nx * ny);
    for (int jy = 0; jy < ny; ++jy) {
        const double ky = (double)(jy < (ny + 1) / 2 ? jy : jy - ny) / (double)ny;
        for (int ix = 0; ix < nx; ++ix) {
            const double kx = (double)(ix < (nx + 1) / 2 ? ix : ix - nx) / (double)nx;
            const double k2 = kx * kx + ky * ky;
            const double kb = use_angle ? kx * bx + ky * by : (b0_dir == PD_B0_Y) ? ky : kx;
            d2[(size_t)jy * nx + ix] = (ix == 0 && jy == 0) ? 0.0 : 1.0 / 3.0 - kb * kb / k2;
        }
    }
    for (int jy = 0; jy < ny; ++jy)
        for (int ix = 0; ix < nx; ++ix) {
            const size_t i = (size_t)jy * nx + ix, im = (size_t)((ny - jy) % ny) * nx + (size_t)((nx - ix) % nx);
            D[i] = (float)(0.5 * (d2[i] + d2[im]) * scale);
        }
}

void build_twiddles(std::vector<float2> &tw, int n) {
    const double pi = 3.14159265358979323846264338327950288;
    for (int k = 0; k < n; ++k) {
        const double ang = -2.0 * pi * (double)k / (double)n;
        tw[k] = make_float2((float)std::cos(ang), (float)std::sin(ang));
    }
}

#define PD_DISPATCH(n, F, ...)                    \
    switch (n) {                                  \
        case 64: F<64>(__VA_ARGS__); break;       \
        case 128: F<128>(__VA_ARGS__); break;     \
        case 256: F<256>(__VA_ARGS__); break;     \
        default: F<512>(__VA_ARGS__); break;      \
    }

// ---- resident variant: configuration per size, occupancy query, launch
template <int N> struct ResChoice;
#ifndef PD_RES256_C
#define PD_RES256_C 8
#define PD_RES256_NT 512
#define PD_RES256_MINB 1
#endif
template <> struct ResChoice<64>  { static constexpr int C = 2, NT = 256, MINB = 1; };
template <> struct ResChoice<128> { static constexpr int C = 4, NT = 256, MINB = 1; };
template <> struct ResChoice<256> { static constexpr int C = PD_RES256_C, NT = PD_RES256_NT, MINB = PD_RES256_MINB; };

template <int N, bool HAS_W, bool ANISO>
cudaError_t resident_launch_config(cudaLaunchConfig_t *cfg, cudaLaunchAttribute *attr, int nclusters, cudaStream_t st) {
    using Ch = ResChoice<N>;
    using Cfg = pdk::ResCfg<N, Ch::C, Ch::NT>;
    cudaError_t e = cudaFuncSetAttribute(pdk::resident_kernel<N, Ch::C, Ch::NT, Ch::MINB, HAS_W, ANISO>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    if (Ch::C > 8) {
        e = cudaFuncSetAttribute(pdk::resident_kernel<N, Ch::C, Ch::NT, Ch::MINB, HAS_W, ANISO>,
                                 cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (e != cudaSuccess) return e;
    }
    std::memset(cfg, 0, sizeof(*cfg));
    cfg->gridDim = dim3((unsigned)(nclusters * Ch::C), 1, 1);
    cfg->blockDim = dim3(Ch::NT, 1, 1);
    cfg->dynamicSmemBytes = Cfg::SMEM_BYTES;
    cfg->stream = st;
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = Ch::C;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg->attrs = attr;
    cfg->numAttrs = 1;
    return cudaSuccess;
}

template <int N>
int resident_max_clusters(int *out) {
    using Ch = ResChoice<N>;
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute attr[1];
    cudaError_t e = resident_launch_config<N, false, false>(&cfg, attr, 1, nullptr);
    if (e != cudaSuccess) return cuda_fail(e, "resident kernel attributes");
    int n = 0;
    e = cudaOccupancyMaxActiveClusters(&n, pdk::resident_kernel<N, Ch::C, Ch::NT, Ch::MINB, false, false>, &cfg);
    if (e != cudaSuccess) return cuda_fail(e, "cudaOccupancyMaxActiveClusters");
    *out = n;
    return PD_OK;
}

template <int N, bool HAS_W, bool ANISO>
cudaError_t resident_launch2(const ResidentArgs &a, int nclusters, cudaStream_t st) {
    using Ch = ResChoice<N>;
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute attr[1];
    cudaError_t e = resident_launch_config<N, HAS_W, ANISO>(&cfg, attr, nclusters, st);
    if (e != cudaSuccess) return e;
    return cudaLaunchKernelEx(&cfg, pdk::resident_kernel<N, Ch::C, Ch::NT, Ch::MINB, HAS_W, ANISO>, a);
}
template <int N>
cudaError_t resident_launch(const ResidentArgs &a, bool w, bool aniso, int nclusters, cudaStream_t st) {
    if (w) return aniso ? resident_launch2<N, true, true>(a, nclusters, st) : resident_launch2<N, true, false>(a, nclusters, st);
    return aniso ? resident_launch2<N, false, true>(a, nclusters, st) : resident_launch2<N, false, false>(a, nclusters, st);
}

// ---- resident kernel with the state on chip (W = identity; pd_resident_tm.cuh): same cluster shape
template <int N, int MODE>
cudaError_t resident_tm_launch2(const ResidentTmArgs &a, int nclusters, cudaStream_t st) {
    using Ch = ResChoice<N>;
    using TCfg = pdk::ResTmCfg<N, Ch::C, Ch::NT>;
    auto kern = pdk::resident_tm_kernel<N, Ch::C, Ch::NT, MODE>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, TCfg::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    if (Ch::C > 8) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (e != cudaSuccess) return e;
    }
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute attr[1];
    std::memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3((unsigned)(nclusters * Ch::C), 1, 1);
    cfg.blockDim = dim3(Ch::NT, 1, 1);
    cfg.dynamicSmemBytes = TCfg::SMEM_BYTES;
    cfg.stream = st;
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = Ch::C;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, a);
}
template <int N>
cudaError_t resident_tm_launch(const ResidentTmArgs &a, int mode, int nclusters, cudaStream_t st) {
    return mode == pdk::kModeL1 ? resident_tm_launch2<N, pdk::kModeL1>(a, nclusters, st)
         : mode == pdk::kModeAniso ? resident_tm_launch2<N, pdk::kModeAniso>(a, nclusters, st)
                                   : resident_tm_launch2<N, pdk::kModeIso>(a, nclusters, st);
}

// D/(N*N) in the order the column phase of resident_tm_kernel reads it: [rank][m][tid] (pd_resident_tm.cuh)
template <int N>
void build_dipole_private(std::vector<float> &out, const std::vector<float> &D) {
    using Ch = ResChoice<N>;
    constexpr int T = pdk::FftCfg<N>::T, E = pdk::FftCfg<N>::E, NT = Ch::NT, C = Ch::C;
    out.assign((size_t)N * N, 0.f);
    for (int rank = 0; rank < C; ++rank)
        for (int m = 0; m < E; ++m)
            for (int tid = 0; tid < NT; ++tid) {
                const int cgi = tid / (16 * T), cc = tid % 16, cj = (tid / 16) % T;
                const int kx = pdk::fd_column_of(N, rank, cgi, cc), ky = cj + T * m;
                out[(size_t)rank * (N / C) * N + (size_t)m * NT + tid] = D[(size_t)ky * N + kx];
            }
}


// ---- streaming workspace: allocated when a streaming solve is first possible (plan time for sizes without a
// resident kernel or with a hybrid tail, pd_set_option(PD_OPT_VARIANT, PD_VARIANT_STREAMING) otherwise) so that
// resident plans stay small
constexpr int kSfdPlanes = 13;   // Z, phi^ (or phi), M, W; p^ (or p), qx, qy twice each; chi three times

// columns one CTA of the column kernels owns (SfdColCfg<ny>::COLS)
int sfd_cols_per_cta(int ny) {
    return ny == 64 ? pdk::SfdColCfg<64>::COLS : ny == 128 ? pdk::SfdColCfg<128>::COLS : ny == 256 ? pdk::SfdColCfg<256>::COLS : pdk::SfdColCfg<512>::COLS;
}

int ensure_sfd_workspace(pd_plan_s *p, size_t npairs) {
    if (p->sfd_planes && p->sfd_pairs_alloc >= npairs) return PD_OK;
    if (p->sfd_planes) { cudaFree(p->sfd_planes); p->sfd_planes = nullptr; }
    if (p->sfd_parts) { cudaFree(p->sfd_parts); p->sfd_parts = nullptr; }
    const size_t PP = (size_t)p->nx * p->ny * npairs;
    p->sfd_ncolparts = p->generic ? p->nparts : p->nx / sfd_cols_per_cta(p->ny);
    p->sfd_nrowparts = p->nparts;
    int rc;
    if ((rc = dev_alloc(&p->sfd_planes, PP * kSfdPlanes)) != PD_OK) return rc;
    // p0_part [2], gap_row [2], res_part [4] per (pair, row part); gap_col x2 [2] per (pair, column part) -- sized for
    // the literal path too, whose data-term partials come from the dual row kernel (row parts)
    const int ncp = p->sfd_ncolparts > p->sfd_nrowparts ? p->sfd_ncolparts : p->sfd_nrowparts;
    const size_t nparts = npairs * (size_t)(8 * p->sfd_nrowparts + 4 * ncp);
    if ((rc = dev_alloc(&p->sfd_parts, nparts)) != PD_OK) return rc;
    // cudaMemset runs on the NULL stream and may return early; the solve may be on a non-blocking stream (the hybrid
    // schedule's second stream always is), so the zeroing must have finished before anything is enqueued
    cudaError_t e = cudaMemset(p->sfd_parts, 0, nparts * sizeof(float));
    if (e == cudaSuccess) e = cudaStreamSynchronize(nullptr);
    if (e != cudaSuccess) return cuda_fail(e, "streaming partial sums init");
    p->sfd_pairs_alloc = npairs;
    return PD_OK;
}

template <int NX> void sfd_launch_init_rows(const StreamFdArgs &a, cudaStream_t st) {
    dim3 grid(a.ny / pdk::SfdRowCfg<NX>::G, a.npairs);
    pdk::sfd_init_rows_kernel<NX><<<grid, pdk::SfdRowCfg<NX>::THREADS, 0, st>>>(a);
}
template <int NX> void sfd_launch_rows(const StreamFdArgs &a, int n, cudaStream_t st) {
    dim3 grid(a.ny / pdk::SfdRowCfg<NX>::G, a.npairs);
    if (a.reg_l1) {
        if (a.mask) pdk::sfd_rows_l1_kernel<NX, true><<<grid, pdk::SfdRowCfg<NX>::THREADS, 0, st>>>(a, n);
        else pdk::sfd_rows_l1_kernel<NX, false><<<grid, pdk::SfdRowCfg<NX>::THREADS, 0, st>>>(a, n);
        return;
    }
    if (a.aniso) {
        if (a.mask) pdk::sfd_rows_kernel<NX, true, true><<<grid, pdk::SfdRowCfg<NX>::THREADS, 0, st>>>(a, n);
        else pdk::sfd_rows_kernel<NX, false, true><<<grid, pdk::SfdRowCfg<NX>::THREADS, 0, st>>>(a, n);
        return;
    }
    if (a.mask) pdk::sfd_rows_kernel<NX, true, false><<<grid, pdk::SfdRowCfg<NX>::THREADS, 0, st>>>(a, n);
    else pdk::sfd_rows_kernel<NX, false, false><<<grid, pdk::SfdRowCfg<NX>::THREADS, 0, st>>>(a, n);
}
template <int NY> void sfd_launch_init_cols(const StreamFdArgs &a, cudaStream_t st) {
    dim3 grid(a.nx / pdk::SfdColCfg<NY>::COLS, a.npairs);
    pdk::sfd_init_cols_kernel<NY><<<grid, pdk::SfdColCfg<NY>::THREADS, pdk::SfdColCfg<NY>::SMEM_BYTES, st>>>(a);
}
template <int NY> void sfd_launch_cols(const StreamFdArgs &a, int n, cudaStream_t st) {
    dim3 grid(a.nx / pdk::SfdColCfg<NY>::COLS, a.npairs);
    if (a.nx == NY) pdk::sfd_cols_kernel<NY, false, NY><<<grid, pdk::SfdColCfg<NY>::THREADS, pdk::SfdColCfg<NY>::SMEM_BYTES, st>>>(a, n, 1);
    else pdk::sfd_cols_kernel<NY, false, 0><<<grid, pdk::SfdColCfg<NY>::THREADS, pdk::SfdColCfg<NY>::SMEM_BYTES, st>>>(a, n, 1);
}
template <int NY> void sfd_launch_cols_plain(const StreamFdArgs &a, int n, int decide, cudaStream_t st) {
    using PC = pdk::SfdColCfg<NY, true>;
    dim3 grid((a.nx + PC::COLS - 1) / PC::COLS, a.npairs);
    if (a.nx == NY) pdk::sfd_cols_kernel<NY, true, NY><<<grid, PC::THREADS, PC::SMEM_BYTES, st>>>(a, n, decide);
    else pdk::sfd_cols_kernel<NY, true, 0><<<grid, PC::THREADS, PC::SMEM_BYTES, st>>>(a, n, decide);
}
template <int NX> void sfd_launch_dual_rows(const StreamFdArgs &a, int n, cudaStream_t st) {
    dim3 grid(a.ny / pdk::SfdRowCfg<NX>::G, a.npairs);
    pdk::sfd_dual_rows_kernel<NX><<<grid, pdk::SfdRowCfg<NX>::THREADS, 0, st>>>(a, n);
}
template <int NY>
cudaError_t sfd_set_col_smem() {
    cudaError_t e = cudaSuccess;
    auto set = [&](auto kern, int bytes) { if (e == cudaSuccess) e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes); };
    set(pdk::sfd_cols_kernel<NY, false, NY>, pdk::SfdColCfg<NY>::SMEM_BYTES); set(pdk::sfd_cols_kernel<NY, false, 0>, pdk::SfdColCfg<NY>::SMEM_BYTES);
    set(pdk::sfd_cols_kernel<NY, true, NY>, pdk::SfdColCfg<NY, true>::SMEM_BYTES); set(pdk::sfd_cols_kernel<NY, true, 0>, pdk::SfdColCfg<NY, true>::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(pdk::sfd_init_cols_kernel<NY>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                pdk::SfdColCfg<NY>::SMEM_BYTES);
}

// (Re)build the dipole tables of the plan -- D/(nx ny) in [ny][nx] order and, for the resident kernel with the state on
// chip, in its thread-private order -- and upload them.  Synchronous (plan time, pd_set_b0_angle).
int upload_dipole(pd_plan_s *p) {
    const size_t P = (size_t)p->nx * p->ny;
    std::vector<float> D(P), Dp;
    build_dipole(D, p->nx, p->ny, p->b0_dir, p->use_angle != 0, p->b0_angle);
    PD_CUDA(cudaMemcpy(p->Dtab, D.data(), P * sizeof(float), cudaMemcpyHostToDevice));
    if (p->Dpriv) {
        if (p->nx == 64) build_dipole_private<64>(Dp, D);
        else if (p->nx == 128) build_dipole_private<128>(Dp, D);
        else build_dipole_private<256>(Dp, D);
        PD_CUDA(cudaMemcpy(p->Dpriv, Dp.data(), P * sizeof(float), cudaMemcpyHostToDevice));
    }
    return PD_OK;
}

// The resident variant runs this plan's next solve: the size has a resident kernel, streaming is not forced, and the
// combination l1 regulariser + (W set or PD_OPT_FOURIER_DUAL = 0) -- which only the streaming kernels implement -- is not asked for
bool use_resident(const pd_plan_s *p) {
    return p->res_ok && p->variant != PD_VARIANT_STREAMING && !(p->reg_l1 && (p->weight || p->no_fd));
}

int resident_csize(int n) { return n == 64 ? ResChoice<64>::C : n == 128 ? ResChoice<128>::C : ResChoice<256>::C; }

int solve_streaming_fd(pd_plan_s *p, const float *field, const float *mask, float *chi_out, int max_iters, float tol,
                       cudaStream_t st, int first = 0, int *launches_out = nullptr, int count = 0);

// Hybrid schedule: slice pairs handed to the streaming kernels.  The resident clusters finish
// `ncl` pairs per wave; the streaming kernels on the SMs they leave free finish about rho * ncl in the same time.
// rho is MEASURED on the plan's device when the plan is made (calibrate_hybrid below); kHybridRhoDefault is only the
// value of a plan whose batch is too small to calibrate.  Choose the number of resident waves w that minimises
// max(w, tail / (rho ncl)).
constexpr double kHybridRhoDefault = 0.15;
int hybrid_tail_rule(int npairs, int ncl, double rho) {
    if (npairs < 1 || ncl < 1 || !(rho > 0.0)) return 0;
    int best_tail = 0;
    double best_t = 1e30;
    for (int w = (npairs + ncl - 1) / ncl; w >= 1; --w) {
        const int tail = npairs > w * ncl ? npairs - w * ncl : 0;
        const double ts = (double)tail / (rho * ncl), t = ts > w ? ts : (double)w;
        if (t < best_t - 1e-9) { best_t = t; best_tail = tail; }
    }
    return best_tail;
}
bool hybrid_possible(const pd_plan_s *p) {
    return p->nx == 256 && p->aux && p->res_max_clusters * 8 + 16 <= p->num_sms;   // SMs left over beside the clusters
}
// tail of a solve over `npairs` slice pairs (the whole batch, or one chunk of pd_solve_host: `whole` false)
int hybrid_tail_pairs(const pd_plan_s *p, int npairs, bool whole) {
    if (p->nx != 256 || p->weight || p->no_fd || p->variant != PD_VARIANT_AUTO || !p->aux) return 0;
    if (p->hybrid_tail >= 0 && whole) return p->hybrid_tail < npairs ? p->hybrid_tail : npairs - 1;
    if (p->hybrid_tail == 0 || !hybrid_possible(p)) return 0;
    return hybrid_tail_rule(npairs, p->res_max_clusters, p->hybrid_rho);
}
int hybrid_tail_pairs(const pd_plan_s *p) { return hybrid_tail_pairs(p, p->npairs, true); }

// The resident kernel over res_pairs slice pairs (res_batch slices) starting at slice `first` of the caller's arrays
cudaError_t launch_resident(pd_plan_s *p, const float *field, const float *mask, float *chi_out, int max_iters, float tol,
                            cudaStream_t st, int res_pairs, int res_batch, int first = 0) {
    const size_t P = (size_t)p->nx * p->ny, off = (size_t)first * P;
    ResidentArgs a;
    std::memset(&a, 0, sizeof(a));
    a.batch = res_batch; a.npairs = res_pairs; a.max_iters = max_iters; a.check_every = p->check_every;
    effective_params(p, &a.alpha, &a.sigma, &a.tau);
    a.theta = p->theta;
    a.inv_one_plus_sigma = 1.0f / (1.0f + a.sigma);
    a.tol = tol;
    a.mask_bstride = p->mask_shared ? 0 : (long long)P;
    a.field = field + off; a.mask = mask ? mask + (size_t)first * (size_t)a.mask_bstride : nullptr;
    a.weight = p->weight ? p->weight + off : nullptr;
    a.chi_out = chi_out + off;
    const size_t stride = (size_t)p->res_clusters * P;
    float2 *base = p->res_scratch;
    a.Z = base; a.qy = base + stride; a.chi = base + 2 * stride; a.chibar = base + 3 * stride;
    a.phi2 = base + 4 * stride; a.M2 = base + 5 * stride; a.W2 = base + 6 * stride;
    a.Dtab = p->Dtab; a.tw_tab = p->tw_row;
    a.part = p->rk_part;
    a.iters_done = p->iters_done + first; a.relgap = p->relgap + first; a.relres = p->relres + first;
    const bool w = p->weight != nullptr, aniso = p->tv_mode == PD_TV_ANISO;
    const int nclusters = res_pairs < p->res_clusters ? res_pairs : p->res_clusters;
    if (!w && !p->no_fd) {
        // W = identity: Fourier-domain dual, state in tensor memory and shared memory (pd_resident_tm.cuh)
        ResidentTmArgs f;
        std::memset(&f, 0, sizeof(f));
        f.batch = a.batch; f.npairs = a.npairs; f.max_iters = a.max_iters; f.check_every = a.check_every;
        f.alpha = a.alpha; f.sigma = a.sigma; f.tau = a.tau; f.theta = a.theta;
        f.inv_one_plus_sigma = a.inv_one_plus_sigma; f.tol = a.tol;
        f.field = a.field; f.mask = a.mask; f.mask_bstride = a.mask_bstride; f.chi_out = a.chi_out;
        f.Z = a.Z; f.M2 = a.M2;
        f.Dpriv = p->Dpriv; f.tw_tab = p->tw_row; f.part = p->rk_part;
        f.iters_done = a.iters_done; f.relgap = a.relgap; f.relres = a.relres;
        const int mode = p->reg_l1 ? pdk::kModeL1 : aniso ? pdk::kModeAniso : pdk::kModeIso;
        switch (p->nx) {
            case 64: return resident_tm_launch<64>(f, mode, nclusters, st);
            case 128: return resident_tm_launch<128>(f, mode, nclusters, st);
            default: return resident_tm_launch<256>(f, mode, nclusters, st);
        }
    }
    switch (p->nx) {
        case 64: return resident_launch<64>(a, w, aniso, nclusters, st);
        case 128: return resident_launch<128>(a, w, aniso, nclusters, st);
        default: return resident_launch<256>(a, w, aniso, nclusters, st);
    }
}

// rho of the hybrid schedule, measured at plan time on this device: one wave of resident clusters and a few slice pairs
// through the streaming kernels run CONCURRENTLY (as in a hybrid solve: the streaming CTAs land on the SMs the clusters
// leave free) on a constant synthetic field, iteration counts chosen so that both sides take about the same time; rho =
// (streaming pair-iterations per ms) / (resident pair-iterations per ms per cluster) / clusters.  Costs a few ms.
int calibrate_hybrid(pd_plan_s *p) {
    const int ncl = p->res_max_clusters;
    const int ps = p->npairs - ncl < 6 ? p->npairs - ncl : 6;   // streaming pairs of the calibration
    p->hybrid_rho = kHybridRhoDefault;
    if (!hybrid_possible(p) || ps < 1) return PD_OK;
    const size_t P = (size_t)p->nx * p->ny, nsl = 2 * (size_t)(ncl + ps);
    float *buf = nullptr;
    int rc = dev_alloc(&buf, 2 * nsl * P);
    if (rc != PD_OK) return rc;
    rc = ensure_sfd_workspace(p, (size_t)ps);
    cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};
    cudaStream_t st = nullptr;
    cudaError_t e = cudaSuccess;
    if (rc == PD_OK) {
        e = cudaMemset(buf, 0x3c, nsl * P * sizeof(float));   // field = 0.0115 everywhere; the work does not depend on the data
        if (e == cudaSuccess) e = cudaStreamSynchronize(nullptr);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking);
        for (int k = 0; k < 3 && e == cudaSuccess; ++k) e = cudaEventCreate(&ev[k]);
    }
    if (rc == PD_OK && e == cudaSuccess) {
        const int graph_loop = p->graph_loop;
        p->graph_loop = 0;
        const int it_res = 48, it_str = (int)(it_res * kHybridRhoDefault * ncl / ps + 0.5);
        float *field = buf, *chi = buf + nsl * P;
        for (int rep = 0; rep < 2 && rc == PD_OK && e == cudaSuccess; ++rep) {   // first repetition warms up
            e = cudaEventRecord(ev[0], st);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(p->aux, ev[0], 0);
            if (e == cudaSuccess) e = launch_resident(p, field, nullptr, chi, it_res, 0.f, st, ncl, 2 * ncl);
            if (e == cudaSuccess) e = cudaEventRecord(ev[1], st);
            int launches = 0;
            if (e == cudaSuccess) rc = solve_streaming_fd(p, field, nullptr, chi, it_str < 1 ? 1 : it_str, 0.f, p->aux, 2 * ncl, &launches, 2 * ps);
            if (rc == PD_OK && e == cudaSuccess) e = cudaEventRecord(ev[2], p->aux);
            if (e == cudaSuccess) e = cudaStreamSynchronize(st);
            if (e == cudaSuccess) e = cudaStreamSynchronize(p->aux);
        }
        p->graph_loop = graph_loop;
        float t_res = 0.f, t_str = 0.f;
        if (rc == PD_OK && e == cudaSuccess) e = cudaEventElapsedTime(&t_res, ev[0], ev[1]);
        if (rc == PD_OK && e == cudaSuccess) e = cudaEventElapsedTime(&t_str, ev[0], ev[2]);
        if (rc == PD_OK && e == cudaSuccess && t_res > 0.f && t_str > 0.f) {
            const double rho = ((double)ps * (it_str < 1 ? 1 : it_str) / t_str) / ((double)ncl * it_res / t_res);
            if (rho > 0.01 && rho < 1.0) p->hybrid_rho = rho;
        }
    }
    for (int k = 0; k < 3; ++k) if (ev[k]) cudaEventDestroy(ev[k]);
    if (st) cudaStreamDestroy(st);
    cudaFree(buf);
    if (rc != PD_OK) return rc;
    if (e != cudaSuccess) return cuda_fail(e, "hybrid calibration");
    return PD_OK;
}

// Slices [first, first + count) of the plan through the resident kernel (count = 0: to the end of the batch), with the
// hybrid schedule's streaming tail where it applies.  field, mask and chi_out are the caller's whole-batch pointers.
int solve_resident(pd_plan_s *p, const float *field, const float *mask, float *chi_out, int max_iters, float tol,
                   cudaStream_t st, int first = 0, int count = 0) {
    const bool whole = (first == 0 && count == 0);
    const int nb = count > 0 ? count : p->batch - first, np = (nb + 1) / 2;
    const int tail = hybrid_tail_pairs(p, np, whole);
    const int res_pairs = np - tail, res_batch = tail ? 2 * res_pairs : nb;
    if (whole) p->ev_class->clear();
    if (p->timing && whole) {
        while (p->ev->size() < 2) {
            cudaEvent_t evn_;
            PD_CUDA(cudaEventCreate(&evn_));
            p->ev->push_back(evn_);
        }
        PD_CUDA(cudaEventRecord((*p->ev)[0], st));
    }
    if (tail) {   // fork: the streaming kernels of the tail run on the plan's second stream
        PD_CUDA(cudaEventRecord(p->ev_fork, st));
        PD_CUDA(cudaStreamWaitEvent(p->aux, p->ev_fork, 0));
    }
    const cudaError_t e = launch_resident(p, field, mask, chi_out, max_iters, tol, st, res_pairs, res_batch, first);
    if (e != cudaSuccess) return cuda_fail(e, "resident kernel launch");
    int tail_launches = 0;
    if (tail) {   // the tail, then join
        const int timing = p->timing;
        p->timing = 0;   // the class-5 bracket below covers the whole hybrid step
        const int rc = solve_streaming_fd(p, field, mask, chi_out, max_iters, tol, p->aux, first + 2 * res_pairs, &tail_launches,
                                          nb - 2 * res_pairs);
        p->timing = timing;
        if (rc != PD_OK) return rc;
        PD_CUDA(cudaEventRecord(p->ev_join, p->aux));
        PD_CUDA(cudaStreamWaitEvent(st, p->ev_join, 0));
    }
    if (p->timing && whole) {
        PD_CUDA(cudaEventRecord((*p->ev)[1], st));
        p->ev_class->push_back(PD_KERNEL_RESIDENT);
    }
    p->last_launches += 1 + tail_launches;
    return PD_OK;
}

int solve_range(pd_plan_s *p, const float *field, const float *mask, float *chi_out, int max_iters, float tol,
                cudaStream_t st, int first, int count) {
    if (use_resident(p)) return solve_resident(p, field, mask, chi_out, max_iters, tol, st, first, count);
    int launches = 0;
    const int rc = solve_streaming_fd(p, field, mask, chi_out, max_iters, tol, st, first, &launches, count);
    p->last_launches += launches;
    return rc;
}


// One launch bracket for PD_OPT_KERNEL_TIMING (shared by the streaming paths)
#define PD_LAUNCH(cls, stmt)                                                                       \
    do {                                                                                           \
        if (p->timing) {                                                                           \
            while (p->ev->size() < 2 * (size_t)(launches + 1)) {                                   \
                cudaEvent_t evn_;                                                                  \
                PD_CUDA(cudaEventCreate(&evn_));                                                   \
                p->ev->push_back(evn_);                                                            \
            }                                                                                      \
            PD_CUDA(cudaEventRecord((*p->ev)[2 * launches], st));                                  \
        }                                                                                          \
        stmt;                                                                                      \
        if (p->timing) {                                                                           \
            PD_CUDA(cudaEventRecord((*p->ev)[2 * launches + 1], st));                              \
            p->ev_class->push_back(cls);                                                           \
        }                                                                                          \
        ++launches;                                                                                \
    } while (0)

// The iteration kernels of one PD iteration (n < 0: inside the graphed loop, the kernels read the device counter)
size_t gen_rows_smem(const pd_plan_s *p) { return (size_t)(pdk::gen_wsize(p->nx) + 2 * pdk::kGenRows * p->nx) * sizeof(float2); }
size_t gen_cols_smem(const pd_plan_s *p) { return (size_t)(pdk::gen_wsize(p->ny) + 2 * pdk::kGenColsB * p->ny) * sizeof(float2); }
void gen_launch_cols(const pd_plan_s *p, const StreamFdArgs &a, int n, int decide, cudaStream_t st) {
    dim3 grid((a.nx + pdk::kGenColsB - 1) / pdk::kGenColsB, a.npairs);
    pdk::gen_cols_kernel<<<grid, 32 * pdk::kGenColsB, gen_cols_smem(p), st>>>(a, p->gdims, n, decide);
}
void gen_launch_dual_rows(const pd_plan_s *p, const StreamFdArgs &a, int n, cudaStream_t st) {
    dim3 grid((a.ny + pdk::kGenRows - 1) / pdk::kGenRows, a.npairs);
    pdk::gen_dual_rows_kernel<<<grid, pdk::kGenLT * pdk::kGenRows, gen_rows_smem(p), st>>>(a, p->gdims, n);
}
void gen_launch_rows(const pd_plan_s *p, const StreamFdArgs &a, int n, cudaStream_t st) {
    dim3 grid((a.ny + pdk::kGenRows - 1) / pdk::kGenRows, a.npairs);
    pdk::gen_rows_kernel<<<grid, pdk::kGenLT * pdk::kGenRows, gen_rows_smem(p), st>>>(a, p->gdims, n);
}
void gen_launch_init(const pd_plan_s *p, const StreamFdArgs &a, int which, cudaStream_t st) {
    if (which == 0) {
        dim3 grid((a.ny + pdk::kGenRows - 1) / pdk::kGenRows, a.npairs);
        pdk::gen_init_kernel<<<grid, 32 * pdk::kGenRows, 0, st>>>(a);
    } else {
        pdk::gen_init_finish_kernel<<<(a.batch + 127) / 128, 128, 0, st>>>(a);
    }
}

// column pass of the general-length path: ny a power of two -> the tuned PLAIN column kernel over contiguous column
// blocks (run-time row pitch); else the dense general-length kernel
void gen_cols_any(const pd_plan_s *p, const StreamFdArgs &a, int n, int decide, cudaStream_t st) {
    if (a.cols_contig) { PD_DISPATCH(p->ny, sfd_launch_cols_plain, a, n, decide, st); }
    else gen_launch_cols(p, a, n, decide, st);
}

void sfd_enqueue_iteration(const pd_plan_s *p, const StreamFdArgs &a, bool literal, int n, cudaStream_t st) {
    if (p->generic) {   // general-length kernels, literal iteration; a power-of-two ny keeps the tuned column transform
        if (n != 0) gen_cols_any(p, a, n, 1, st);
        gen_launch_dual_rows(p, a, n, st);
        gen_cols_any(p, a, n, 0, st);
        gen_launch_rows(p, a, n, st);
        return;
    }
    if (literal) {
        if (n != 0) { PD_DISPATCH(p->ny, sfd_launch_cols_plain, a, n, 1, st); }   // K1 (chibar_0 = 0; in the loop the kernel skips n = 0 itself)
        PD_DISPATCH(p->nx, sfd_launch_dual_rows, a, n, st);
        PD_DISPATCH(p->ny, sfd_launch_cols_plain, a, n, 0, st);                    // K2
    } else {
        PD_DISPATCH(p->ny, sfd_launch_cols, a, n, st);
    }
    PD_DISPATCH(p->nx, sfd_launch_rows, a, n, st);
}

void graph_slot_release(pd_plan_s::GraphSlot &g) {
    if (g.exec) cudaGraphExecDestroy(g.exec);
    if (g.graph) cudaGraphDestroy(g.graph);
    g.exec = nullptr; g.graph = nullptr; g.key_valid = 0;
}

// Build (or reuse) the executable graph of one streaming solve with arguments `a`:
//   memset(iter) -> scale -> init_rows -> init_cols -> WHILE (handle) { iteration kernels ; sfd_loop_ctl } -> finish
// The WHILE node's handle is set on the device by sfd_loop_ctl: when every slice has stopped (or n = max_iters) the
// body is not launched again -- no no-op launches, no host round trip.
int sfd_graph_prepare(pd_plan_s *p, StreamFdArgs &a, bool literal, int *slot_out) {
    // the iteration counter belongs to the slot: look the arguments up with each slot's own counter in place
    for (int k = 0; k < kGraphSlots; ++k) {
        pd_plan_s::GraphSlot &c = p->gslot[k];
        a.iter = c.iter;
        if (c.key_valid && c.literal == (literal ? 1 : 0) && std::memcmp(&c.key, &a, sizeof(a)) == 0) { *slot_out = k; return PD_OK; }
    }
    const int slot = p->gslot_next;
    p->gslot_next = (p->gslot_next + 1) % kGraphSlots;
    *slot_out = slot;
    pd_plan_s::GraphSlot &g = p->gslot[slot];
    if (g.exec) PD_CUDA(cudaDeviceSynchronize());   // a graph being replaced may still be running (chunks of an earlier call)
    graph_slot_release(g);
    if (!g.iter) {
        const int rc_ = dev_alloc(&g.iter, 1);
        if (rc_ != PD_OK) return rc_;
    }
    a.iter = g.iter;
    if (!p->cap_stream) PD_CUDA(cudaStreamCreateWithFlags(&p->cap_stream, cudaStreamNonBlocking));
    cudaStream_t cs = p->cap_stream;
    const size_t P = (size_t)p->nx * p->ny;
    PD_CUDA(cudaGraphCreate(&g.graph, 0));
    // prologue
    PD_CUDA(cudaStreamBeginCaptureToGraph(cs, g.graph, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed));
    cudaError_t e = cudaMemsetAsync(a.iter, 0, sizeof(int), cs);
    pdk::sfd_scale_kernel<<<a.batch, 256, 0, cs>>>(a);
    if (p->generic) {
        gen_launch_init(p, a, 0, cs);
        gen_launch_init(p, a, 1, cs);
    } else {
        PD_DISPATCH(p->nx, sfd_launch_init_rows, a, cs);
        PD_DISPATCH(p->ny, sfd_launch_init_cols, a, cs);
    }
    cudaStreamCaptureStatus status;
    const cudaGraphNode_t *deps = nullptr;
    size_t ndeps = 0;
    if (e == cudaSuccess) e = cudaStreamGetCaptureInfo_v2(cs, &status, nullptr, nullptr, &deps, &ndeps);
    std::vector<cudaGraphNode_t> pro(deps, deps + (e == cudaSuccess ? ndeps : 0));
    cudaGraph_t dummy = nullptr;
    cudaError_t e2 = cudaStreamEndCapture(cs, &dummy);
    if (e == cudaSuccess) e = e2;
    if (e != cudaSuccess) { graph_slot_release(g); return cuda_fail(e, "graph capture (prologue)"); }
    // WHILE node
    cudaGraphConditionalHandle handle;
    PD_CUDA(cudaGraphConditionalHandleCreate(&handle, g.graph, a.max_iters > 0 ? 1u : 0u, cudaGraphCondAssignDefault));
    cudaGraphNodeParams cp = {};
    cp.type = cudaGraphNodeTypeConditional;
    cp.conditional.handle = handle;
    cp.conditional.type = cudaGraphCondTypeWhile;
    cp.conditional.size = 1;
    cudaGraphNode_t wnode;
    PD_CUDA(cudaGraphAddNode(&wnode, g.graph, pro.data(), pro.size(), &cp));
    cudaGraph_t body = cp.conditional.phGraph_out[0];
    PD_CUDA(cudaStreamBeginCaptureToGraph(cs, body, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed));
    sfd_enqueue_iteration(p, a, literal, -1, cs);
    pdk::sfd_loop_ctl_kernel<<<1, 256, 0, cs>>>(a, handle);
    e = cudaStreamEndCapture(cs, &dummy);
    if (e != cudaSuccess) { graph_slot_release(g); return cuda_fail(e, "graph capture (loop body)"); }
    // epilogue
    PD_CUDA(cudaStreamBeginCaptureToGraph(cs, g.graph, &wnode, nullptr, 1, cudaStreamCaptureModeRelaxed));
    {
        const int gx = (int)((P + 256 * 8 - 1) / (256 * 8));
        pdk::sfd_finish_kernel<<<dim3(gx, a.npairs), 256, 0, cs>>>(a);
    }
    e = cudaStreamEndCapture(cs, &dummy);
    if (e != cudaSuccess) { graph_slot_release(g); return cuda_fail(e, "graph capture (epilogue)"); }
    e = cudaGraphInstantiate(&g.exec, g.graph, 0);
    if (e != cudaSuccess) { graph_slot_release(g); return cuda_fail(e, "cudaGraphInstantiate"); }
    g.key = a;
    g.key_valid = 1;
    g.literal = literal ? 1 : 0;
    return PD_OK;
}

// Streaming variant, W = identity: two launches per iteration (pd_streaming_fd.cuh)
// Slices [first, batch) of the plan (first even); field, mask and chi_out are the caller's whole-batch pointers.
int solve_streaming_fd(pd_plan_s *p, const float *field, const float *mask, float *chi_out, int max_iters, float tol,
                       cudaStream_t st, int first, int *launches_out, int count) {
    const int nb = count > 0 ? count : p->batch - first, np = (nb + 1) / 2;
    int rc = ensure_sfd_workspace(p, (size_t)np);
    if (rc != PD_OK) return rc;
    const size_t P = (size_t)p->nx * p->ny, PP = P * (size_t)np;
    StreamFdArgs a;
    std::memset(&a, 0, sizeof(a));
    a.nx = p->nx; a.ny = p->ny; a.batch = nb; a.npairs = np;
    a.max_iters = max_iters; a.check_every = p->check_every; a.aniso = p->tv_mode == PD_TV_ANISO;
    effective_params(p, &a.alpha, &a.sigma, &a.tau);
    a.theta = p->theta;
    a.inv_one_plus_sigma = 1.0f / (1.0f + a.sigma);
    a.tol = tol;
    a.mask_bstride = p->mask_shared ? 0 : (long long)P;
    const bool literal = p->weight != nullptr || p->no_fd || p->generic;   // p in the image domain, K applied twice (PAPER.md:49 literally)
    a.literal = literal ? 1 : 0;
    a.reg_l1 = p->reg_l1;
    a.cols_contig = (p->generic && size_ok(p->ny)) ? 1 : 0;
    a.weight = p->weight ? p->weight + (size_t)first * P : nullptr;
    a.field = field + (size_t)first * P;
    a.mask = mask ? mask + (size_t)first * (size_t)a.mask_bstride : nullptr;
    a.chi_out = chi_out + (size_t)first * P;
    float2 *b = p->sfd_planes;
    a.Z = b; a.phihat = b + PP; a.M2 = b + 2 * PP;
    for (int k = 0; k < 2; ++k) { a.phat[k] = b + (3 + k) * PP; a.qx2[k] = b + (5 + k) * PP; a.qy2[k] = b + (7 + k) * PP; }
    for (int k = 0; k < 3; ++k) a.chi3[k] = b + (9 + k) * PP;
    a.W2 = b + 12 * PP;
    a.Dtab = p->Dtab; a.tw_row = p->tw_row; a.tw_col = p->tw_col;
    a.stop_iter = p->stop_iter + first; a.P0 = p->P0 + first; a.relgap = p->relgap + first;
    a.relres = p->relres + first; a.iters_done = p->iters_done + first;
    a.cscale = p->cscale + first;
    a.nrowparts = p->sfd_nrowparts;
    a.ncolparts = literal ? p->sfd_nrowparts : p->sfd_ncolparts;   // who writes the data term of the gap
    const size_t nr = (size_t)np * a.nrowparts, nc = (size_t)np * (size_t)(p->sfd_ncolparts > p->sfd_nrowparts ? p->sfd_ncolparts : p->sfd_nrowparts);
    float *q = p->sfd_parts;
    a.p0_part = q; q += 2 * nr;
    a.gap_row = q; q += 2 * nr;
    a.res_part = q; q += 4 * nr;
    a.gap_col[0] = q; q += 2 * nc;
    a.gap_col[1] = q;

    int launches = 0;
    if (!launches_out) p->ev_class->clear();
    if (p->graph_loop && !p->timing) {
        // one graph launch: the loop over iterations and its termination live on the device
        int slot = 0;
        if ((rc = sfd_graph_prepare(p, a, literal, &slot)) != PD_OK) return rc;
        PD_CUDA(cudaGraphLaunch(p->gslot[slot].exec, st));
        p->graph_used |= 1u << slot;   // its kernels are counted on demand (pd_last_launch_count)
        if (launches_out) *launches_out = 0; else p->last_launches = 0;
        return PD_OK;
    }
    PD_LAUNCH(PD_KERNEL_INIT, (pdk::sfd_scale_kernel<<<a.batch, 256, 0, st>>>(a)));
    if (p->generic) {
        PD_LAUNCH(PD_KERNEL_INIT, gen_launch_init(p, a, 0, st));
        PD_LAUNCH(PD_KERNEL_INIT, gen_launch_init(p, a, 1, st));
    } else {
        PD_LAUNCH(PD_KERNEL_INIT, PD_DISPATCH(p->nx, sfd_launch_init_rows, a, st));
        PD_LAUNCH(PD_KERNEL_INIT, PD_DISPATCH(p->ny, sfd_launch_init_cols, a, st));
    }
    for (int n = 0; n < max_iters; ++n) {
        if (p->generic) {
            if (n > 0) PD_LAUNCH(PD_KERNEL_COLS, gen_cols_any(p, a, n, 1, st));
            PD_LAUNCH(PD_KERNEL_DUAL, gen_launch_dual_rows(p, a, n, st));
            PD_LAUNCH(PD_KERNEL_COLS, gen_cols_any(p, a, n, 0, st));
            PD_LAUNCH(PD_KERNEL_FD_ROWS, gen_launch_rows(p, a, n, st));
            continue;
        }
        if (literal) {
            if (n > 0) PD_LAUNCH(PD_KERNEL_COLS, PD_DISPATCH(p->ny, sfd_launch_cols_plain, a, n, 1, st));   // K1 (chibar_0 = 0)
            PD_LAUNCH(PD_KERNEL_DUAL, PD_DISPATCH(p->nx, sfd_launch_dual_rows, a, n, st));
            PD_LAUNCH(PD_KERNEL_COLS, PD_DISPATCH(p->ny, sfd_launch_cols_plain, a, n, 0, st));              // K2
        } else {
            PD_LAUNCH(PD_KERNEL_FD_COLS, PD_DISPATCH(p->ny, sfd_launch_cols, a, n, st));
        }
        PD_LAUNCH(PD_KERNEL_FD_ROWS, PD_DISPATCH(p->nx, sfd_launch_rows, a, n, st));
    }
    {
        const int gx = (int)((P + 256 * 8 - 1) / (256 * 8));
        PD_LAUNCH(PD_KERNEL_FINISH, (pdk::sfd_finish_kernel<<<dim3(gx, np), 256, 0, st>>>(a)));
    }
    PD_CUDA(cudaGetLastError());
    if (launches_out) *launches_out = launches; else p->last_launches = launches;
    return PD_OK;
}

}  // namespace

// ---- pd_solve_static: the streaming solve (Fourier-domain dual, pd_streaming_fd.cuh) with its WHOLE workspace -- the 13
// state planes, the per-CTA partial sums, the dipole and twiddle tables, the per-slice state variables -- in one
// file-scope device array instead of cudaMalloc'ed memory, for callers that may not allocate (CUDA-graph capture, tight
// serving loops).  Every GPU that loads the library holds the array until the process exits.  In host code the NAME of
// the array is only a host-side stand-in: its device address comes from cudaGetSymbolAddress, once per device.
constexpr size_t kStaticCells = PD_STATIC_MAX_CELLS;                 // nx * ny * ceil(batch / 2) of one call, at most
constexpr size_t kStaticAlign = 256;
constexpr size_t static_round(size_t bytes) { return (bytes + kStaticAlign - 1) / kStaticAlign * kStaticAlign; }
constexpr size_t kStaticPartsFloats = 16384;                         // per-CTA partial sums (checked per call)
constexpr size_t kStaticOffPlanes = 0;
constexpr size_t kStaticOffD = kStaticOffPlanes + static_round(kSfdPlanes * kStaticCells * sizeof(float2));
constexpr size_t kStaticOffTwRow = kStaticOffD + static_round(kStaticCells * sizeof(float));
constexpr size_t kStaticOffTwCol = kStaticOffTwRow + static_round(PD_STATIC_MAX_N * sizeof(float2));
// from here on: cleared by every call (what a fresh plan's cudaMemset clears)
constexpr size_t kStaticOffZero = kStaticOffTwCol + static_round(PD_STATIC_MAX_N * sizeof(float2));
constexpr size_t kStaticSlot = static_round((PD_STATIC_MAX_BATCH + 1) * sizeof(float));
constexpr size_t kStaticOffStop = kStaticOffZero;                    // stop_iter [batch + 1]
constexpr size_t kStaticOffIters = kStaticOffStop + kStaticSlot;     // iters_done [batch]
constexpr size_t kStaticOffP0 = kStaticOffIters + kStaticSlot;
constexpr size_t kStaticOffGap = kStaticOffP0 + kStaticSlot;
constexpr size_t kStaticOffRes = kStaticOffGap + kStaticSlot;
constexpr size_t kStaticOffScale = kStaticOffRes + kStaticSlot;      // cscale [batch + 1]
constexpr size_t kStaticOffParts = kStaticOffScale + kStaticSlot;
constexpr size_t kStaticBytes = kStaticOffParts + static_round(kStaticPartsFloats * sizeof(float));
static_assert(kStaticBytes == PD_STATIC_SCRATCH_BYTES, "include/pd.h states the size of the static workspace");

static __device__ __align__(256) unsigned char pd_static_scratch[kStaticBytes];

namespace {

constexpr int kStaticMaxDevices = 64;
struct StaticDev {
    int ready;              // cudaGetSymbolAddress done on this device
    unsigned char *base;    // DEVICE address of pd_static_scratch on this device
    int nx, ny, b0;         // what the tables in the array were built for (nx = 0: nothing yet)
};
StaticDev g_static_dev[kStaticMaxDevices];

bool static_size_ok(int n) { return n == 64 || n == 128 || n == 256; }

// Set-up, once per device (address of the array, shared-memory attributes of the column kernels) and once per
// (nx, ny, B0_dir) change on it (tables: built on the host in double like pd_plan's, uploaded synchronously).
int static_setup(int nx, int ny, int b0_dir, StaticDev **out) {
    int dev = -1;
    PD_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) return PD_EINVAL;
    StaticDev &sd = g_static_dev[dev];
    if (!sd.ready) {
        void *ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&ptr, pd_static_scratch);   // the current device's copy of the array
        if (e != cudaSuccess || !ptr) return cuda_fail(e, "cudaGetSymbolAddress(pd_static_scratch)");
        if (e == cudaSuccess) e = sfd_set_col_smem<64>();
        if (e == cudaSuccess) e = sfd_set_col_smem<128>();
        if (e == cudaSuccess) e = sfd_set_col_smem<256>();
        if (e != cudaSuccess) return cuda_fail(e, "static workspace set-up");
        sd.base = (unsigned char *)ptr;
        sd.nx = sd.ny = 0;
        sd.ready = 1;
    }
    if (sd.nx != nx || sd.ny != ny || sd.b0 != b0_dir) {
        static float hD[kStaticCells];
        static float2 htw[2][PD_STATIC_MAX_N];
        PD_CUDA(cudaDeviceSynchronize());   // an earlier call may still be reading the tables
        sd.nx = 0;
        const double pi = 3.14159265358979323846264338327950288, scale = 1.0 / ((double)nx * (double)ny);
        // D/(nx ny), the same arithmetic as build_dipole (axis-aligned B0: the table is even, no symmetrisation needed)
        for (int jy = 0; jy < ny; ++jy) {
            const double ky = (double)(jy < (ny + 1) / 2 ? jy : jy - ny) / (double)ny;
            for (int ix = 0; ix < nx; ++ix) {
                const double kx = (double)(ix < (nx + 1) / 2 ? ix : ix - nx) / (double)nx;
                const double k2 = kx * kx + ky * ky, kb = (b0_dir == PD_B0_Y) ? ky : kx;
                hD[(size_t)jy * nx + ix] = (float)(((ix == 0 && jy == 0) ? 0.0 : 1.0 / 3.0 - kb * kb / k2) * scale);
            }
        }
        for (int w = 0; w < 2; ++w) {
            const int n = w ? ny : nx;
            for (int k = 0; k < n; ++k) {
                const double ang = -2.0 * pi * (double)k / (double)n;
                htw[w][k] = make_float2((float)std::cos(ang), (float)std::sin(ang));
            }
        }
        PD_CUDA(cudaMemcpy(sd.base + kStaticOffD, hD, (size_t)nx * ny * sizeof(float), cudaMemcpyHostToDevice));
        PD_CUDA(cudaMemcpy(sd.base + kStaticOffTwRow, htw[0], (size_t)nx * sizeof(float2), cudaMemcpyHostToDevice));
        PD_CUDA(cudaMemcpy(sd.base + kStaticOffTwCol, htw[1], (size_t)ny * sizeof(float2), cudaMemcpyHostToDevice));
        PD_CUDA(cudaDeviceSynchronize());
        sd.nx = nx; sd.ny = ny; sd.b0 = b0_dir;
    }
    *out = &sd;
    return PD_OK;
}

}  // namespace

extern "C" {

int pd_solve_static(int nx, int ny, int batch, int B0_dir, float lambda, float sigma, float tau, float theta,
                    const float *field, const float *mask, float *chi_out, int max_iters, float tol,
                    int *iters_done, float *relgap, float *relres, void *cuda_stream) {
    if (!field || !chi_out || max_iters < 0 || batch < 1 || (B0_dir != PD_B0_X && B0_dir != PD_B0_Y)) return PD_EINVAL;
    if (nx < 1 || ny < 1) return PD_EINVAL;
    const int np = (batch + 1) / 2;
    if (!static_size_ok(nx) || !static_size_ok(ny) || batch > PD_STATIC_MAX_BATCH ||
        (size_t)nx * (size_t)ny * (size_t)np > kStaticCells)
        return PD_ESTATIC;
    int rc = check_params(lambda, sigma, tau, theta, false, norm_bound(1.0, 1.0));
    if (rc != PD_OK) return rc;
    const int nrowparts = ny / (nx == 64 ? pdk::SfdRowCfg<64>::G : nx == 128 ? pdk::SfdRowCfg<128>::G : pdk::SfdRowCfg<256>::G);
    const int ncolparts = nx / sfd_cols_per_cta(ny);
    const size_t nr = (size_t)np * nrowparts, nc = (size_t)np * (size_t)(ncolparts > nrowparts ? ncolparts : nrowparts);
    if (8 * nr + 4 * nc > kStaticPartsFloats) return PD_ESTATIC;
    StaticDev *sd = nullptr;
    if ((rc = static_setup(nx, ny, B0_dir, &sd)) != PD_OK) return rc;

    cudaStream_t st = (cudaStream_t)cuda_stream;
    unsigned char *base = sd->base;
    const size_t P = (size_t)nx * ny, PP = P * (size_t)np;
    pd_plan_s q;   // only the fields effective_params reads: the same steps as a fresh plan with default options
    std::memset(&q, 0, sizeof(q));
    q.lambda_user = lambda; q.sigma_user = sigma; q.tau_user = tau; q.theta = theta; q.max_w = q.max_m = 1.0;
    StreamFdArgs a;
    std::memset(&a, 0, sizeof(a));
    a.nx = nx; a.ny = ny; a.batch = batch; a.npairs = np;
    a.max_iters = max_iters; a.check_every = 1;
    effective_params(&q, &a.alpha, &a.sigma, &a.tau);
    a.theta = theta;
    a.inv_one_plus_sigma = 1.0f / (1.0f + a.sigma);
    a.tol = tol;
    a.mask_bstride = (long long)P;
    a.field = field; a.mask = mask; a.chi_out = chi_out;
    float2 *b = (float2 *)(base + kStaticOffPlanes);
    a.Z = b; a.phihat = b + PP; a.M2 = b + 2 * PP;
    for (int k = 0; k < 2; ++k) { a.phat[k] = b + (3 + k) * PP; a.qx2[k] = b + (5 + k) * PP; a.qy2[k] = b + (7 + k) * PP; }
    for (int k = 0; k < 3; ++k) a.chi3[k] = b + (9 + k) * PP;
    a.W2 = b + 12 * PP;
    a.Dtab = (const float *)(base + kStaticOffD);
    a.tw_row = (const float2 *)(base + kStaticOffTwRow);
    a.tw_col = (const float2 *)(base + kStaticOffTwCol);
    a.stop_iter = (int *)(base + kStaticOffStop);
    a.P0 = (float *)(base + kStaticOffP0);
    a.cscale = (float *)(base + kStaticOffScale);
    a.iters_done = iters_done ? iters_done : (int *)(base + kStaticOffIters);
    a.relgap = relgap ? relgap : (float *)(base + kStaticOffGap);
    a.relres = relres ? relres : (float *)(base + kStaticOffRes);
    a.nrowparts = nrowparts;
    a.ncolparts = ncolparts;
    float *parts = (float *)(base + kStaticOffParts);
    a.p0_part = parts; parts += 2 * nr;
    a.gap_row = parts; parts += 2 * nr;
    a.res_part = parts; parts += 4 * nr;
    a.gap_col[0] = parts; parts += 2 * nc;
    a.gap_col[1] = parts;

    // the array keeps the last call's contents: clear what a fresh plan starts at zero (state variables, partial sums)
    PD_CUDA(cudaMemsetAsync(base + kStaticOffZero, 0, kStaticBytes - kStaticOffZero, st));
    if (iters_done) PD_CUDA(cudaMemsetAsync(iters_done, 0, (size_t)batch * sizeof(int), st));
    if (relgap) PD_CUDA(cudaMemsetAsync(relgap, 0, (size_t)batch * sizeof(float), st));
    if (relres) PD_CUDA(cudaMemsetAsync(relres, 0, (size_t)batch * sizeof(float), st));
    pdk::sfd_scale_kernel<<<a.batch, 256, 0, st>>>(a);
    PD_DISPATCH(nx, sfd_launch_init_rows, a, st);
    PD_DISPATCH(ny, sfd_launch_init_cols, a, st);
    for (int n = 0; n < max_iters; ++n) {
        PD_DISPATCH(ny, sfd_launch_cols, a, n, st);
        PD_DISPATCH(nx, sfd_launch_rows, a, n, st);
    }
    pdk::sfd_finish_kernel<<<dim3((unsigned)((P + 256 * 8 - 1) / (256 * 8)), np), 256, 0, st>>>(a);
    PD_CUDA(cudaGetLastError());
    return PD_OK;
}

int pd_plan(pd_plan_t *out, int nx, int ny, int batch, int B0_dir, float lambda, float sigma, float tau, float theta) {
    if (!out) return PD_EINVAL;
    *out = nullptr;
    if (batch < 1 || (B0_dir != PD_B0_X && B0_dir != PD_B0_Y)) return PD_EINVAL;
    const bool generic = !(size_ok(nx) && size_ok(ny));
    if (generic && !(gen_size_ok(nx) && gen_size_ok(ny))) return PD_ESIZE;
    int rc = check_params(lambda, sigma, tau, theta, false, norm_bound(1.0, 1.0));
    if (rc != PD_OK) return rc;

    pd_plan_s *p = new (std::nothrow) pd_plan_s;
    if (!p) return PD_ENOMEM;
    std::memset(p, 0, sizeof(*p));
    p->ev = new (std::nothrow) std::vector<cudaEvent_t>();
    p->ev_class = new (std::nothrow) std::vector<int>();
    if (!p->ev || !p->ev_class) { delete p->ev; delete p->ev_class; delete p; return PD_ENOMEM; }
    p->nx = nx; p->ny = ny; p->batch = batch; p->npairs = (batch + 1) / 2; p->b0_dir = B0_dir;
    p->lambda_user = lambda; p->sigma_user = sigma; p->tau_user = tau; p->theta = theta;
    p->check_every = 1;
    p->max_w = p->max_m = 1.0;
    p->hybrid_tail = -1;
    p->graph_loop = 1;
    {
        cudaError_t e = cudaGetDevice(&p->device);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&p->num_sms, cudaDevAttrMultiProcessorCount, p->device);
        if (e != cudaSuccess) { pd_destroy(p); return cuda_fail(e, "cudaGetDevice"); }
    }
    p->generic = generic ? 1 : 0;
    balanced_factors(nx, &p->gdims.n1x, &p->gdims.n2x);
    balanced_factors(ny, &p->gdims.n1y, &p->gdims.n2y);
    const int rows_per_cta = generic ? pdk::kGenRows : nx == 64 ? pdk::SfdRowCfg<64>::G : nx == 128 ? pdk::SfdRowCfg<128>::G
                           : nx == 256 ? pdk::SfdRowCfg<256>::G : pdk::SfdRowCfg<512>::G;
    p->nparts = (ny + rows_per_cta - 1) / rows_per_cta;

    const size_t P = (size_t)nx * ny;
#define PD_TRY(expr) do { rc = (expr); if (rc != PD_OK) { pd_destroy(p); return rc; } } while (0)
    PD_TRY(dev_alloc(&p->Dtab, P));
    PD_TRY(dev_alloc(&p->tw_row, (size_t)nx));
    PD_TRY(dev_alloc(&p->tw_col, (size_t)ny));
    PD_TRY(dev_alloc(&p->stop_iter, (size_t)batch + 1));
    PD_TRY(dev_alloc(&p->iters_done, (size_t)batch));
    PD_TRY(dev_alloc(&p->P0, (size_t)batch));
    PD_TRY(dev_alloc(&p->relgap, (size_t)batch));
    PD_TRY(dev_alloc(&p->relres, (size_t)batch));
    PD_TRY(dev_alloc(&p->cscale, (size_t)batch + 1));
#undef PD_TRY
    {
        std::vector<float2> twr(nx), twc(ny);
        build_twiddles(twr, nx);
        build_twiddles(twc, ny);
        if ((rc = upload_dipole(p)) != PD_OK) { pd_destroy(p); return rc; }
        cudaError_t e = cudaMemcpy(p->tw_row, twr.data(), nx * sizeof(float2), cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMemcpy(p->tw_col, twc.data(), ny * sizeof(float2), cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMemset(p->iters_done, 0, batch * sizeof(int));
        if (e == cudaSuccess) e = cudaMemset(p->relgap, 0, batch * sizeof(float));
        if (e == cudaSuccess) e = cudaMemset(p->relres, 0, batch * sizeof(float));
        if (e == cudaSuccess) e = sfd_set_col_smem<64>();
        if (e == cudaSuccess) e = sfd_set_col_smem<128>();
        if (e == cudaSuccess) e = sfd_set_col_smem<256>();
        if (e == cudaSuccess) e = sfd_set_col_smem<512>();
        if (e == cudaSuccess && generic) {
            // the attribute belongs to the function, not to the plan: always the largest supported length (1024)
            const int cmax = (pdk::gen_wsize(1024) + 2 * pdk::kGenColsB * 1024) * (int)sizeof(float2), rmax = (pdk::gen_wsize(1024) + 2 * pdk::kGenRows * 1024) * (int)sizeof(float2);
            e = cudaFuncSetAttribute(pdk::gen_cols_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, cmax);
            if (e == cudaSuccess) e = cudaFuncSetAttribute(pdk::gen_dual_rows_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, rmax);
            if (e == cudaSuccess) e = cudaFuncSetAttribute(pdk::gen_rows_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, rmax);
        }
        if (e != cudaSuccess) { pd_destroy(p); return cuda_fail(e, "plan table upload"); }
    }
    // resident variant: square slices up to 256x256
    if (!generic && nx == ny && nx <= 256) {
        int maxc = 0;
        rc = (nx == 64) ? resident_max_clusters<64>(&maxc) : (nx == 128) ? resident_max_clusters<128>(&maxc)
                                                                          : resident_max_clusters<256>(&maxc);
        if (rc == PD_OK && maxc >= 1) {
            p->res_csize = resident_csize(nx);
            p->res_clusters = maxc < p->npairs ? maxc : p->npairs;
            p->res_max_clusters = maxc;
            rc = dev_alloc(&p->res_scratch, (size_t)pdk::kResidentScratchArrays * p->res_clusters * P);
            if (rc == PD_OK) rc = dev_alloc(&p->rk_part, (size_t)p->res_clusters * p->res_csize * 8);
            if (rc != PD_OK) { pd_destroy(p); return rc; }
            if (rc == PD_OK) rc = dev_alloc(&p->Dpriv, P);
            if (rc != PD_OK) { pd_destroy(p); return rc; }
            if ((rc = upload_dipole(p)) != PD_OK) { pd_destroy(p); return rc; }
            cudaError_t e = cudaMemset(p->rk_part, 0, (size_t)p->res_clusters * p->res_csize * 8 * sizeof(float));
            if (e != cudaSuccess) { pd_destroy(p); return cuda_fail(e, "resident scratch init"); }
            p->res_ok = 1;
            if (nx == 256) {   // second stream of the hybrid schedule, and the workspace of its automatic tail
                cudaError_t e3 = cudaStreamCreateWithFlags(&p->aux, cudaStreamNonBlocking);
                if (e3 == cudaSuccess) e3 = cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming);
                if (e3 == cudaSuccess) e3 = cudaEventCreateWithFlags(&p->ev_join, cudaEventDisableTiming);
                if (e3 != cudaSuccess) { pd_destroy(p); return cuda_fail(e3, "hybrid stream"); }
                if ((rc = calibrate_hybrid(p)) != PD_OK) { pd_destroy(p); return rc; }
                const int tail = hybrid_tail_pairs(p);
                if (tail > 0 && (rc = ensure_sfd_workspace(p, (size_t)tail)) != PD_OK) { pd_destroy(p); return rc; }
            }
        } else {
            cudaGetLastError();  // no cluster launch possible on this device: the streaming variant remains
        }
    }
    {   // table uploads and memsets above ran on the NULL stream: finish them before a solve on any other stream
        cudaError_t e = cudaStreamSynchronize(nullptr);
        if (e != cudaSuccess) { pd_destroy(p); return cuda_fail(e, "plan synchronize"); }
    }
    if (!p->res_ok) {   // streaming is the only path of this plan: take its workspace now
        rc = ensure_sfd_workspace(p, (size_t)p->npairs);
        if (rc != PD_OK) { pd_destroy(p); return rc; }
    }
    *out = p;
    return PD_OK;
}

int pd_set_weight(pd_plan_t p, const float *W) {
    if (!p) return PD_EINVAL;
    p->weight = W;
    return PD_OK;
}

int pd_set_b0_angle(pd_plan_t p, float angle_rad) {
    if (!p || !std::isfinite(angle_rad)) return PD_EINVAL;
    PD_CUDA(cudaDeviceSynchronize());   // no solve of this plan may still be reading the tables
    p->use_angle = 1;
    p->b0_angle = (double)angle_rad;
    return upload_dipole(p);
}

int pd_set_steps(pd_plan_t p, float lambda, float sigma, float tau, float theta) {
    if (!p) return PD_EINVAL;
    int rc = check_params(lambda, sigma, tau, theta, p->unsafe_steps != 0, norm_bound(p->max_w, p->max_m));
    if (rc != PD_OK) return rc;
    p->lambda_user = lambda; p->sigma_user = sigma; p->tau_user = tau; p->theta = theta;
    return PD_OK;
}

int pd_set_norm_bounds(pd_plan_t p, float max_abs_w, float max_abs_m) {
    if (!p || !(max_abs_w > 0.f) || !(max_abs_m > 0.f) || !std::isfinite(max_abs_w) || !std::isfinite(max_abs_m)) return PD_EINVAL;
    // explicit steps already in the plan must satisfy the new bound too
    const int rc = check_params(p->lambda_user, p->sigma_user, p->tau_user, p->theta, p->unsafe_steps != 0,
                                norm_bound((double)max_abs_w, (double)max_abs_m));
    if (rc != PD_OK) return rc;
    p->max_w = (double)max_abs_w;
    p->max_m = (double)max_abs_m;
    return PD_OK;
}

int pd_set_option(pd_plan_t p, int key, int value) {
    if (!p) return PD_EINVAL;
    switch (key) {
        case PD_OPT_TV_MODE:
            if (value != PD_TV_ISO && value != PD_TV_ANISO) return PD_EINVAL;
            p->tv_mode = value; return PD_OK;
        case PD_OPT_LAMBDA_CONV:
            if (value != PD_LAMBDA_REG && value != PD_LAMBDA_DATA) return PD_EINVAL;
            p->lambda_conv = value; return PD_OK;
        case PD_OPT_VARIANT:
            if (value != PD_VARIANT_AUTO && value != PD_VARIANT_STREAMING && value != PD_VARIANT_RESIDENT) return PD_EINVAL;
            if (value == PD_VARIANT_RESIDENT && !p->res_ok) return PD_EVARIANT;
            p->variant = value;
            return value == PD_VARIANT_STREAMING ? ensure_sfd_workspace(p, (size_t)p->npairs) : PD_OK;
        case PD_OPT_CHECK_EVERY:
            if (value < 1) return PD_EINVAL;
            p->check_every = value; return PD_OK;
        case PD_OPT_MASK_SHARED:
            if (value != 0 && value != 1) return PD_EINVAL;
            p->mask_shared = value; return PD_OK;
        case PD_OPT_UNSAFE_STEPS:
            if (value != 0 && value != 1) return PD_EINVAL;
            p->unsafe_steps = value; return PD_OK;
        case PD_OPT_FOURIER_DUAL:
            if (value != 0 && value != 1) return PD_EINVAL;
            p->no_fd = !value; return PD_OK;
        case PD_OPT_KERNEL_TIMING:
            if (value != 0 && value != 1) return PD_EINVAL;
            p->timing = value; return PD_OK;
        case PD_OPT_HYBRID_TAIL:
            if (value < -1) return PD_EINVAL;
            p->hybrid_tail = value; return PD_OK;
        case PD_OPT_REGULARISER:
            if (value != PD_REG_TV && value != PD_REG_L1) return PD_EINVAL;
            p->reg_l1 = (value == PD_REG_L1); return PD_OK;
        case PD_OPT_HOST_CHUNKING:
            if (value < 0 || value > 2) return PD_EINVAL;
            p->host_chunking = value; return PD_OK;
        case PD_OPT_GRAPH_LOOP:
            if (value != 0 && value != 1) return PD_EINVAL;
            p->graph_loop = value; return PD_OK;
        default: return PD_EINVAL;
    }
}

int pd_solve(pd_plan_t p, const float *field, const float *mask, float *chi_out, int max_iters, float tol,
             void *cuda_stream) {
    if (!p || !field || !chi_out || max_iters < 0) return PD_EINVAL;
    if (p->lambda_conv == PD_LAMBDA_DATA && !(p->lambda_user > 0.f)) return PD_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    p->last_launches = 0;
    p->graph_used = 0u;
    if (use_resident(p)) return solve_resident(p, field, mask, chi_out, max_iters, tol, st);
    return solve_streaming_fd(p, field, mask, chi_out, max_iters, tol, st);
}

// Chunks of pd_solve_host, in slices (even counts, the last takes the rest).  Slices are independent, so
// the batch is cut into a short first chunk (its upload is the only one nobody hides), a long middle and short last
// chunks (the download of the very last one is the only one nobody hides): H2D(k+1) || solve(k) || D2H(k-1).
// Resident variant: the unit is one wave of clusters (no chunk leaves clusters idle) and a solve costs about ten times
// its upload, so the chunks grow 1, 4, rest and shrink 4, 2.  Streaming variant: a small chunk cannot fill the GPU with
// its launches, so three chunks of 1/8, 6/8, 1/8 of the batch (measured on C4: five chunks lose more than they hide).
int host_chunks(const pd_plan_s *p, int *count /*[kMaxChunks]*/) {
    const bool res = use_resident(p);
    int unit = res ? p->res_max_clusters : (p->npairs + 7) / 8;   // pairs
    if (unit < 1) unit = 1;
    const int np = p->npairs;
    int n = 0, left = np;
    // A streaming chunk must still fill the GPU with every launch (its time per iteration is bounded below by launch
    // latency, not by work): automatic chunking only when the smallest chunk has at least two row CTAs per SM.  E1
    // (13 pairs of 256x258) in three chunks took 126 ms end to end against 75 ms on device buffers.
    bool chunk = p->host_chunking != 2;
    if (chunk && p->host_chunking == 0 && !res) chunk = (long long)unit * p->nparts >= 2LL * p->num_sms;
    if (!chunk) {
    } else if (res && np >= 24 * unit) {     // 1, 4, middle, 4, 2 units
        const int head[2] = {unit, 4 * unit}, tail[2] = {4 * unit, 2 * unit};
        count[n++] = 2 * head[0]; count[n++] = 2 * head[1];
        count[n++] = 2 * (np - head[0] - head[1] - tail[0] - tail[1]);
        count[n++] = 2 * tail[0]; count[n++] = 2 * tail[1];
        left = 0;
    } else if (np >= 6 * unit) {      // 1, middle, 1 units
        count[n++] = 2 * unit; count[n++] = 2 * (np - 2 * unit); count[n++] = 2 * unit;
        left = 0;
    }
    if (left) count[n++] = 2 * left;
    int used = 0;
    for (int k = 0; k < n; ++k) used += count[k];
    count[n - 1] -= used - p->batch;   // an odd batch: the last pair is half empty
    return n;
}

int pd_solve_host(pd_plan_t p, const float *field_host, const float *mask_host, float *chi_out_host, int max_iters,
                  float tol, void *cuda_stream) {
    if (!p || !field_host || !chi_out_host || max_iters < 0) return PD_EINVAL;
    if (p->lambda_conv == PD_LAMBDA_DATA && !(p->lambda_user > 0.f)) return PD_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t P = (size_t)p->nx * p->ny, BP = P * (size_t)p->batch;
    int rc;
    if (!p->h_field && (rc = dev_alloc(&p->h_field, BP)) != PD_OK) return rc;
    if (!p->h_chi && (rc = dev_alloc(&p->h_chi, BP)) != PD_OK) return rc;
    if (mask_host && !p->h_mask && (rc = dev_alloc(&p->h_mask, p->mask_shared ? P : BP)) != PD_OK) return rc;
    if (!p->h2d_stream) {
        PD_CUDA(cudaStreamCreateWithFlags(&p->h2d_stream, cudaStreamNonBlocking));
        PD_CUDA(cudaStreamCreateWithFlags(&p->d2h_stream, cudaStreamNonBlocking));
        for (cudaEvent_t &ev : p->ev_chunk) PD_CUDA(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
    }
    int count[kMaxChunks];
    const int nchunks = (p->timing || p->weight) ? 1 : host_chunks(p, count);
    if (nchunks == 1) count[0] = p->batch;
    {   // workspaces the chunks need must exist before anything is in flight (an allocation synchronises and may free)
        size_t need = 0;
        for (int k = 0; k < nchunks; ++k) {
            const int np = (count[k] + 1) / 2;
            const bool res = use_resident(p);
            const size_t t = res ? (size_t)hybrid_tail_pairs(p, np, nchunks == 1) : (size_t)np;
            need = t > need ? t : need;
        }
        if (need && (rc = ensure_sfd_workspace(p, need)) != PD_OK) return rc;
    }
    p->last_launches = 0;
    p->graph_used = 0u;
    cudaEvent_t *ev_up = p->ev_chunk, *ev_done = p->ev_chunk + kMaxChunks, ev_start = p->ev_chunk[2 * kMaxChunks],
                ev_end = p->ev_chunk[2 * kMaxChunks + 1];
    // the copies start when the caller's stream reaches this call
    PD_CUDA(cudaEventRecord(ev_start, st));
    PD_CUDA(cudaStreamWaitEvent(p->h2d_stream, ev_start, 0));
    PD_CUDA(cudaStreamWaitEvent(p->d2h_stream, ev_start, 0));
    if (mask_host && p->mask_shared)
        PD_CUDA(cudaMemcpyAsync(p->h_mask, mask_host, P * sizeof(float), cudaMemcpyHostToDevice, p->h2d_stream));
    int first = 0;
    for (int k = 0; k < nchunks; ++k) {          // flow step (2) of the paper, chunk by chunk
        const size_t off = (size_t)first * P, nby = (size_t)count[k] * P * sizeof(float);
        PD_CUDA(cudaMemcpyAsync(p->h_field + off, field_host + off, nby, cudaMemcpyHostToDevice, p->h2d_stream));
        if (mask_host && !p->mask_shared)
            PD_CUDA(cudaMemcpyAsync(p->h_mask + off, mask_host + off, nby, cudaMemcpyHostToDevice, p->h2d_stream));
        PD_CUDA(cudaEventRecord(ev_up[k], p->h2d_stream));
        first += count[k];
    }
    first = 0;
    for (int k = 0; k < nchunks; ++k) {
        const size_t off = (size_t)first * P, nby = (size_t)count[k] * P * sizeof(float);
        PD_CUDA(cudaStreamWaitEvent(st, ev_up[k], 0));
        if (nchunks == 1) {
            rc = (use_resident(p))
                     ? solve_resident(p, p->h_field, mask_host ? p->h_mask : nullptr, p->h_chi, max_iters, tol, st)
                     : solve_streaming_fd(p, p->h_field, mask_host ? p->h_mask : nullptr, p->h_chi, max_iters, tol, st);
        } else {
            rc = solve_range(p, p->h_field, mask_host ? p->h_mask : nullptr, p->h_chi, max_iters, tol, st, first, count[k]);
        }
        if (rc != PD_OK) return rc;
        PD_CUDA(cudaEventRecord(ev_done[k], st));
        PD_CUDA(cudaStreamWaitEvent(p->d2h_stream, ev_done[k], 0));   // flow step (6), chunk by chunk
        PD_CUDA(cudaMemcpyAsync(chi_out_host + off, p->h_chi + off, nby, cudaMemcpyDeviceToHost, p->d2h_stream));
        first += count[k];
    }
    PD_CUDA(cudaEventRecord(ev_end, p->d2h_stream));
    PD_CUDA(cudaStreamWaitEvent(st, ev_end, 0));
    PD_CUDA(cudaStreamSynchronize(st));
    return PD_OK;
}

int pd_get_stats(pd_plan_t p, const int **iters_done, const float **relgap, const float **relres) {
    if (!p) return PD_EINVAL;
    if (iters_done) *iters_done = p->iters_done;
    if (relgap) *relgap = p->relgap;
    if (relres) *relres = p->relres;
    return PD_OK;
}

int pd_get_stats_host(pd_plan_t p, int *iters_done_host, float *relgap_host, float *relres_host, void *cuda_stream) {
    if (!p) return PD_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t n = (size_t)p->batch;
    if (iters_done_host) PD_CUDA(cudaMemcpyAsync(iters_done_host, p->iters_done, n * sizeof(int), cudaMemcpyDeviceToHost, st));
    if (relgap_host) PD_CUDA(cudaMemcpyAsync(relgap_host, p->relgap, n * sizeof(float), cudaMemcpyDeviceToHost, st));
    if (relres_host) PD_CUDA(cudaMemcpyAsync(relres_host, p->relres, n * sizeof(float), cudaMemcpyDeviceToHost, st));
    PD_CUDA(cudaStreamSynchronize(st));
    return PD_OK;
}

int pd_get_kernel_times(pd_plan_t p, float *ms_host, int *launches_host) {
    if (!p) return PD_EINVAL;
    for (int c = 0; c < PD_NUM_KERNEL_CLASSES; ++c) {
        if (ms_host) ms_host[c] = 0.f;
        if (launches_host) launches_host[c] = 0;
    }
    if (!p->timing) return PD_EINVAL;
    const size_t n = p->ev_class->size();
    if (n == 0) return PD_OK;
    PD_CUDA(cudaEventSynchronize((*p->ev)[2 * n - 1]));
    for (size_t i = 0; i < n; ++i) {
        float ms = 0.f;
        PD_CUDA(cudaEventElapsedTime(&ms, (*p->ev)[2 * i], (*p->ev)[2 * i + 1]));
        const int c = (*p->ev_class)[i];
        if (ms_host) ms_host[c] += ms;
        if (launches_host) launches_host[c] += 1;
    }
    return PD_OK;
}

int pd_last_launch_count(pd_plan_t p) {
    if (!p) return PD_EINVAL;
    int n = p->last_launches;
    if (p->graph_used) {   // kernels the graphed loops executed: decided on the device, so ask the device
        if (cudaDeviceSynchronize() != cudaSuccess) return PD_ECUDA;
        for (int k = 0; k < kGraphSlots; ++k) {
            if (!(p->graph_used & (1u << k))) continue;
            int iters = 0;
            if (cudaMemcpy(&iters, p->gslot[k].iter, sizeof(int), cudaMemcpyDeviceToHost) != cudaSuccess) return PD_ECUDA;
            n += 4 + iters * (p->gslot[k].literal ? 5 : 3);   // scale, init rows + cols, finish ; per iteration its kernels + loop control
        }
    }
    return n;
}

int pd_get_info(pd_plan_t p, int *variant, int *clusters, int *cluster_size) {
    if (!p) return PD_EINVAL;
    const bool res = use_resident(p);
    if (variant) *variant = res ? PD_VARIANT_RESIDENT : PD_VARIANT_STREAMING;
    if (clusters) *clusters = res ? p->res_clusters : 0;
    if (cluster_size) *cluster_size = res ? p->res_csize : 0;
    return PD_OK;
}

int pd_line_factors(int n, int *n1, int *n2) {
    if (!n1 || !n2) return PD_EINVAL;
    switch (n) {   // the tuned kernels: threads per line x points per thread of the row configuration (fft_regs.cuh)
        case 64: *n1 = pdk::FftCfg<64>::T; *n2 = pdk::FftCfg<64>::E; return 1;
        case 128: *n1 = pdk::FftCfg<128>::T; *n2 = pdk::FftCfg<128>::E; return 1;
        case 256: *n1 = pdk::FftCfg<256>::T; *n2 = pdk::FftCfg<256>::E; return 1;
        case 512: *n1 = pdk::FftCfg<512>::T; *n2 = pdk::FftCfg<512>::E; return 1;
        default: break;
    }
    if (!gen_size_ok(n)) return PD_ESIZE;
    balanced_factors(n, n1, n2);
    return 0;
}

int pd_hybrid_tail_rule(int npairs, int clusters, float rho) { return hybrid_tail_rule(npairs, clusters, (double)rho); }

int pd_get_hybrid_rho(pd_plan_t p, float *rho) {
    if (!p || !rho) return PD_EINVAL;
    *rho = (float)p->hybrid_rho;
    return PD_OK;
}

int pd_get_hybrid_tail(pd_plan_t p, int *tail_pairs) {
    if (!p || !tail_pairs) return PD_EINVAL;
    *tail_pairs = (use_resident(p)) ? hybrid_tail_pairs(p) : 0;
    return PD_OK;
}

int pd_destroy(pd_plan_t p) {
    if (!p) return PD_EINVAL;
    void *ptrs[] = {p->Dtab, p->tw_row, p->tw_col, p->stop_iter, p->iters_done,
                    p->P0, p->relgap, p->relres, p->cscale, p->h_field, p->h_mask, p->h_chi, p->res_scratch, p->rk_part, p->Dpriv,
                    p->sfd_planes, p->sfd_parts};
    for (void *q : ptrs)
        if (q) cudaFree(q);
    for (int k = 0; k < kGraphSlots; ++k) {
        if (p->gslot[k].exec) cudaGraphExecDestroy(p->gslot[k].exec);
        if (p->gslot[k].graph) cudaGraphDestroy(p->gslot[k].graph);
        if (p->gslot[k].iter) cudaFree(p->gslot[k].iter);
    }
    if (p->cap_stream) cudaStreamDestroy(p->cap_stream);
    if (p->h2d_stream) cudaStreamDestroy(p->h2d_stream);
    if (p->d2h_stream) cudaStreamDestroy(p->d2h_stream);
    for (cudaEvent_t ev : p->ev_chunk) if (ev) cudaEventDestroy(ev);
    if (p->aux) cudaStreamDestroy(p->aux);
    if (p->ev_fork) cudaEventDestroy(p->ev_fork);
    if (p->ev_join) cudaEventDestroy(p->ev_join);
    if (p->ev) for (cudaEvent_t e : *p->ev) cudaEventDestroy(e);
    delete p->ev;
    delete p->ev_class;
    delete p;
    return PD_OK;
}

const char *pd_strerror(int code) {
    switch (code) {
        case PD_OK: return "success";
        case PD_EINVAL: return "invalid argument";
        case PD_ESIZE: return "nx and ny must each be one of 64, 128, 256, 512 (tuned kernels) or both even and in [4, 1024] (general-length kernels)";
        case PD_ESTEP: return "sigma*tau*(4/9+8) >= 1: step sizes violate the convergence bound";
        case PD_ENOMEM: return "out of device memory";
        case PD_ECUDA: return g_cuda_err;
        case PD_EVARIANT: return "requested variant is not available for this size";
        case PD_ESTATIC: return "pd_solve_static: nx and ny must each be 64, 128 or 256, batch <= 32 and nx*ny*ceil(batch/2) <= 65536 "
                                "(the static workspace of PD_STATIC_SCRATCH_BYTES bytes holds no more); use pd_plan / pd_solve";
        default: return "unknown error code";
    }
}

}  // extern "C"
