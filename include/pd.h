/*
 * pd.h -- C ABI of the B200-native primal-dual (Chambolle-Pock) solver for the dipole-kernel
 * deconvolution of positive-contrast susceptibility MRI (arXiv 2006.09808).
 *
 * What is solved (Eq.(1); readings R1-R3 in DESIGN.md), independently for every
 * 2-D slice / coil field map b of a stack:
 *
 *     chi_b = argmin_chi  1/2 || W (K chi - phi_b) ||_2^2 + lambda || M G chi ||_1 ,   K = F^-1 D F
 *
 * by exactly the iteration of PAPER.md:44-49 (p-update, q-update, chi-update, over-relaxation),
 * started from zero and run for max_iters iterations ("Until n >= N")
 * or, per slice, until the relative primal-dual gap falls below tol (BASELINE.json north_star (d)).
 * D(kx,ky) = 1/3 - k_b^2/(kx^2+ky^2), D(0,0) = 0 (BASELINE.json north_star).  G: forward
 * differences with Neumann boundary; M: mask on the gradient; W: optional data weighting.
 * Variants: lambda ||M chi||_1 with a shrinkage prox (PD_OPT_REGULARISER), anisotropic projection, the paper's
 * placement of lambda (PD_OPT_LAMBDA_CONV), an oblique in-plane B0 (pd_set_b0_angle).
 * Sizes: nx, ny in {64,128,256,512} run the tuned kernels (square <= 256: the resident cluster kernel); any other even
 * nx, ny in [4,1024] -- the paper's 256x258 and 128x132 -- run the general-length streaming kernels.
 *
 * Layout of every image argument: fp32, [batch][ny][nx], x fastest, contiguous, 16-byte aligned.
 * Multi-coil stacks: batch = nslices*ncoils, index slice*ncoils + coil (BASELINE.json configs[3]);
 * every coil map is reconstructed independently.
 *
 * All entry points return PD_OK (0) or a negative pd_error; nothing throws across the ABI; there
 * is no global state.  A plan is not thread-safe; distinct plans are independent.  There is no
 * CPU fallback: every step of the path runs in sm_100a CUDA kernels.
 */
#ifndef PD_B200_H
#define PD_B200_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pd_plan_s *pd_plan_t; /* opaque, library-owned */

enum pd_b0 { PD_B0_X = 0, PD_B0_Y = 1 }; /* in-plane B0 axis: k_b = kx (fast axis) or ky (row axis) */

enum pd_error {
    PD_OK = 0,
    PD_EINVAL = -1,   /* null plan/field/chi_out, batch < 1, max_iters < 0, theta outside [0,1], lambda < 0, bad option */
    PD_ESIZE = -2,    /* nx, ny neither both in {64,128,256,512} (tuned kernels) nor both even and in [4,1024] (general-length kernels) */
    PD_ESTEP = -3,    /* explicit steps with sigma*tau*(4/9 max|W|^2 + 8 max|M|^2) >= 1 (both maxima 1 unless pd_set_norm_bounds):
                         convergence bound of [7] violated */
    PD_ENOMEM = -4,   /* device allocation failed */
    PD_ECUDA = -5,    /* a CUDA call or launch failed; pd_strerror(PD_ECUDA) returns the last CUDA error text */
    PD_EVARIANT = -6, /* PD_VARIANT_RESIDENT requested for a size that does not fit on chip */
    PD_ESTATIC = -7   /* pd_solve_static: the problem does not fit the static workspace (limits below) */
};

enum pd_option {
    PD_OPT_TV_MODE = 0,      /* PD_TV_ISO (default) | PD_TV_ANISO: how |.| in the q-projection is read (PAPER.md:49 line 2) */
    PD_OPT_LAMBDA_CONV = 1,  /* PD_LAMBDA_REG (default): 1/2||.||^2 + lambda*TV ; PD_LAMBDA_DATA: lambda/2||.||^2 + TV (PAPER.md:37 literally) */
    PD_OPT_VARIANT = 2,      /* PD_VARIANT_AUTO (default) | PD_VARIANT_STREAMING | PD_VARIANT_RESIDENT */
    PD_OPT_CHECK_EVERY = 3,  /* tolerance tested when (n+1) % value == 0 ; default 1 */
    PD_OPT_MASK_SHARED = 4,  /* 0 (default): mask is [batch][ny][nx] ; 1: one [ny][nx] mask for all slices */
    PD_OPT_UNSAFE_STEPS = 5, /* 1: skip the PD_ESTEP check at the next pd_set_steps call (not at pd_plan) */
    PD_OPT_KERNEL_TIMING = 6,/* 1: bracket every kernel launch of pd_solve with CUDA events on the caller's stream
                                (read with pd_get_kernel_times); default 0 */
    PD_OPT_FOURIER_DUAL = 7, /* 1 (default): when W is the identity keep the dual variable p in the Fourier domain
                                (one FFT round trip per iteration; same iterates up to rounding);
                                0: always apply K twice per iteration, literally as PAPER.md:49 */
    PD_OPT_HYBRID_TAIL = 8,  /* 256x256, W = identity, PD_VARIANT_AUTO only: slice pairs (from the END of the batch) that
                                run through the streaming kernels on a plan-owned second stream, concurrently with the
                                resident clusters, on the SMs those leave free (slices are independent).
                                -1 (default): chosen from the batch size ; 0: off ; n > 0: exactly n pairs.
                                pd_solve still returns with all work ordered on the caller's stream. */
    PD_OPT_GRAPH_LOOP = 9,   /* streaming variant: 1 (default): the whole solve is ONE CUDA graph launch -- init, a conditional
                                WHILE node around the iteration kernels whose condition a loop-control kernel sets on the
                                device (false once every slice has stopped or max_iters is reached), finish: nothing is
                                launched for iterations nobody needs and the host is never asked.  The graph
                                is cached in the plan and rebuilt when the arguments of pd_solve change.  0: one stream
                                launch per kernel, 2*max_iters + 4 of them (the kernels of a stopped slice return at once).
                                PD_OPT_KERNEL_TIMING = 1 always uses plain launches. */
    PD_OPT_REGULARISER = 10, /* PD_REG_TV (default): the paper's lambda ||M G chi||_1 with the dual q.
                                PD_REG_L1: lambda ||M chi||_1 (BASELINE.json north_star's alternative):
                                no q, the primal step ends in the soft shrinkage chi <- sign(v) max(|v| - tau lambda M, 0);
                                relgap is then the Fenchel-Young gap of the data term alone.  PD_OPT_TV_MODE is ignored. */
    PD_OPT_HOST_CHUNKING = 11 /* pd_solve_host: 0 (default) cut the batch into pipelined chunks when every chunk still fills the
                                GPU (resident: whole waves of clusters; streaming: >= 2 row CTAs per SM per launch), 1 always
                                (when the batch has enough slice pairs), 2 never */
};
enum { PD_REG_TV = 0, PD_REG_L1 = 1 };
/* kernel classes for pd_get_kernel_times.  Streaming variant: init, finish and, per iteration, fd_cols + fd_rows
 * (W = identity, Fourier-domain dual: two launches) or dipole_cols + dual_rows + dipole_cols + fd_rows (W set, or
 * PD_OPT_FOURIER_DUAL = 0: four launches; class 3 is no longer used).  Resident variant: class 5, one bracket around
 * the whole step (with the hybrid schedule that includes the streaming tail on the second stream). */
enum pd_kernel_class { PD_KERNEL_INIT = 0, PD_KERNEL_DUAL = 1, PD_KERNEL_COLS = 2, PD_KERNEL_PRIMAL = 3,
                       PD_KERNEL_FINISH = 4, PD_KERNEL_RESIDENT = 5, PD_KERNEL_FD_COLS = 6, PD_KERNEL_FD_ROWS = 7,
                       PD_NUM_KERNEL_CLASSES = 8 };
enum { PD_TV_ISO = 0, PD_TV_ANISO = 1 };
enum { PD_LAMBDA_REG = 0, PD_LAMBDA_DATA = 1 };
enum { PD_VARIANT_AUTO = 0, PD_VARIANT_STREAMING = 1, PD_VARIANT_RESIDENT = 2 };

/* pd_plan (host call; PAPER.md:44 step 1, "dipole kernel convolution operator D").
 * Builds the dipole table D for (nx, ny, B0_dir), the FFT twiddle tables (computed in double), the per-slice
 * state variables and the device workspace of the variant the plan will run: the per-cluster
 * scratch of the resident kernel (square sizes <= 256), and/or the streaming planes (sizes without a resident
 * kernel, or the tail of the hybrid schedule).  A streaming workspace that only a later option or weight makes
 * necessary is allocated by pd_set_option(PD_OPT_VARIANT, ...) or by the first pd_solve that needs it (that one
 * call then contains a cudaMalloc and a NULL-stream synchronisation).  A plan serves one pd_solve at a time.
 * sigma <= 0 or tau <= 0 selects the automatic steps
 * sigma = tau = 1/sqrt(4/9 + 8) (upper bound on ||K_full||_2 for |W|, |M| <= 1; pd_set_norm_bounds for
 * larger weights or mask values).  *out receives the plan.
 * Errors: PD_EINVAL, PD_ESIZE, PD_ESTEP, PD_ENOMEM, PD_ECUDA.  Uses the current CUDA device. */
int pd_plan(pd_plan_t *out, int nx, int ny, int batch, int B0_dir,
            float lambda, float sigma, float tau, float theta);

/* pd_solve (the Repeat loop; flow steps (3)-(5)).
 * field  : DEVICE, const, [batch][ny][nx]  -- the local field map phi = Delta B ("iFreq delta")
 * mask   : DEVICE, const, [batch][ny][nx] (or [ny][nx] with PD_OPT_MASK_SHARED), multiplies the gradient (M of
 *          Eq.(1)); NULL = all ones.  Any float is accepted and used as a multiplier.
 * chi_out: DEVICE, [batch][ny][nx] -- receives chi_N (PAPER.md:49 names chi the solution).  It is also the
 *          solver's primal state during the call; must not alias field/mask/W.
 * max_iters >= 0.  tol <= 0: exactly max_iters iterations for every slice.  tol > 0: slice b stops at the first
 *          checked iteration n+1 with relgap_{n+1} < tol (relative Fenchel-Young gap, R9), else at
 *          max_iters; stopped slices cost (almost) nothing afterwards.  A slice whose W*phi is identically zero
 *          returns chi = 0 (iters_done 0 when tol > 0).
 * cuda_stream: a cudaStream_t (NULL = legacy default stream).  Everything is enqueued on it, or -- hybrid schedule,
 *          PD_OPT_HYBRID_TAIL -- on a plan-owned second stream that is forked from and joined back into it with
 *          events; the call does not synchronise and never copies to the host.  Buffers must stay alive until the stream
 *          reaches the end of the enqueued work.  Inputs are never written.
 * Errors: PD_EINVAL, PD_ENOMEM, PD_ECUDA. */
int pd_solve(pd_plan_t p, const float *field, const float *mask, float *chi_out,
             int max_iters, float tol, void *cuda_stream);

/* pd_solve_host: same computation with HOST buffers (pinned for the copies to overlap; pageable works, serialised by
 * the driver) -- flow steps (2) and (6) of the paper done by the library.  Slices are independent
 * (PAPER.md:82), so a large batch is cut into a few contiguous chunks and pipelined on plan-owned copy streams:
 * upload of chunk k+1 || solve of chunk k (on cuda_stream) || download of chunk k-1; small batches, a set weight and
 * PD_OPT_KERNEL_TIMING use one chunk.  Returns after synchronising cuda_stream, with chi_out_host complete.
 * Staging buffers, streams and events are plan-owned (allocated on first use). */
int pd_solve_host(pd_plan_t p, const float *field_host, const float *mask_host, float *chi_out_host,
                  int max_iters, float tol, void *cuda_stream);

/* Optional data weighting W of Eq.(1) (DEVICE, [batch][ny][nx], caller-owned, must outlive the solves that use it);
 * NULL (default) = identity. */
int pd_set_weight(pd_plan_t p, const float *W);

/* Replace lambda / sigma / tau / theta of an existing plan (same checks as pd_plan). */
int pd_set_steps(pd_plan_t p, float lambda, float sigma, float tau, float theta);

/* Oblique in-plane B0 (BASELINE.json north_star "B0_dir"): the dipole table is rebuilt for the
 * unit vector (cos a, sin a), a = angle_rad from the x axis: k_b = kx cos a + ky sin a (0 = PD_B0_X, pi/2 = PD_B0_Y).
 * K is the real part of F^-1 D F (R12), so the even part (D(k) + D(-k))/2 is stored (it differs from D only on
 * the Nyquist lines).  Host call; waits for the device, then uploads.  Errors: PD_EINVAL, PD_ECUDA. */
int pd_set_b0_angle(pd_plan_t p, float angle_rad);

/* Bounds on |W| and |M| (R14; "tau = sigma = 1/L, L = ||K||_2").  pd_plan assumes |W| <= 1 and |M| <= 1: the
 * automatic steps are 1/sqrt(4/9 + 8) and PD_ESTEP tests sigma tau (4/9 + 8) < 1.  A caller whose weights or mask exceed 1
 * states the bounds here: the automatic steps become 1/sqrt(4/9 max|W|^2 + 8 max|M|^2) and PD_ESTEP (here and in
 * pd_set_steps) uses the same bound.  The arrays themselves arrive later and are never scanned (no host round trip).
 * Errors: PD_EINVAL (non-positive or non-finite bound), PD_ESTEP (explicit steps of the plan violate the new bound). */
int pd_set_norm_bounds(pd_plan_t p, float max_abs_w, float max_abs_m);

int pd_set_option(pd_plan_t p, int key, int value);

/* Per-slice state variables of the last pd_solve: DEVICE pointers, length batch, plan-owned, valid
 * (after the stream reached the end of that solve) until the next pd_solve / pd_destroy.  Any pointer may be NULL.
 * iters_done[b]: iterations executed; relgap[b]: last relative gap computed; relres[b]: last ||chi_{n+1}-chi_n|| / ||chi_{n+1}||. */
int pd_get_stats(pd_plan_t p, const int **iters_done, const float **relgap, const float **relres);

/* Host convenience: copies the three arrays above into HOST buffers of length batch (any may be NULL), ordered on
 * cuda_stream after the last pd_solve, and synchronises that stream. */
int pd_get_stats_host(pd_plan_t p, int *iters_done_host, float *relgap_host, float *relres_host, void *cuda_stream);

/* With PD_OPT_KERNEL_TIMING = 1: waits for the last pd_solve and returns, per kernel class, the summed device time
 * in milliseconds (ms_host[PD_NUM_KERNEL_CLASSES]) and the number of launches (launches_host[...]); HOST pointers. */
int pd_get_kernel_times(pd_plan_t p, float *ms_host, int *launches_host);

/* Number of kernels of the last pd_solve (for launch accounting in benchmarks).  With the graphed loop the number is
 * decided on the device: the call then waits for the device (cudaDeviceSynchronize) and reads the loop counter. */
int pd_last_launch_count(pd_plan_t p);

/* Which variant the next pd_solve of this plan runs, and its launch shape (HOST pointers, any may be NULL):
 * *variant = PD_VARIANT_STREAMING or PD_VARIANT_RESIDENT; *clusters = thread-block clusters the resident kernel is
 * launched with (the paper's "N slices at a time", here slice PAIRS in flight; 0 for streaming);
 * *cluster_size = CTAs per cluster (0 for streaming). */
int pd_get_info(pd_plan_t p, int *variant, int *clusters, int *cluster_size);

/* Slice pairs the next pd_solve hands to the streaming kernels under the hybrid schedule (PD_OPT_HYBRID_TAIL);
 * 0 when the schedule does not apply.  HOST pointer. */
int pd_get_hybrid_tail(pd_plan_t p, int *tail_pairs);

/* The rule behind the automatic tail (pure host arithmetic, no device needed): with `clusters` resident clusters in
 * flight, each finishing one slice pair per wave, and the streaming side finishing about rho * clusters pairs in the
 * same time, the number of whole resident waves w that minimises max(w, tail / (rho * clusters)) is taken and
 * tail = npairs - w * clusters (0 if that is negative) is returned. */
int pd_hybrid_tail_rule(int npairs, int clusters, float rho);

/* How a line of length n is transformed (pure host arithmetic, no device needed; HOST pointers).  Returns 1 for a
 * power-of-two length of the tuned kernels: *n1 = threads per line, *n2 = points per thread of the row kernels
 * (64: 8 x 8, 128: 8 x 16, 256: 16 x 16, 512: 32 x 16 in three stages).  Returns 0 for a general length (even, 4..1024):
 * n = *n1 * *n2 with *n1 <= *n2 the most balanced factorisation, the two dense stages of pd_streaming_gen.cuh
 * (258 = 6 x 43, 132 = 11 x 12; a prime gives 1 x n).  Errors: PD_ESIZE (unsupported length), PD_EINVAL. */
int pd_line_factors(int n, int *n1, int *n2);

/* rho of this plan: measured by pd_plan on the plan's device (one wave of resident clusters and a few slice pairs
 * through the streaming kernels, run concurrently on a synthetic field; a few ms), or the built-in 0.15 when the batch
 * is too small for a tail or the size has no hybrid schedule.  HOST pointer. */
int pd_get_hybrid_rho(pd_plan_t p, float *rho);

int pd_destroy(pd_plan_t p);

/* The true 3-D variant: Eq.(1) as PAPER.md:37-40 literally states it -- "G is the gradient
 * operator in all three dimensions" -- with the 3-D dipole kernel D3(k) = 1/3 - k_b^2/|k|^2, D3(0) = 0,
 * k = (fi/nx, fj/ny, fk/nz) with signed indices (isotropic voxels; reading R23), one problem per VOLUME:
 * the same iteration with q of three components projected on the lambda-ball by its pointwise Euclidean
 * norm, forward differences with Neumann boundary on all three axes, W optional (pd_set_weight3d), lambda on the regulariser (R2).  The
 * slices of a volume are coupled by the z transform and the z difference: there is no per-slice stop, the call runs
 * exactly max_iters iterations.  A streaming implementation (5 launches per iteration).
 * pd_plan3d: nx in {16..256}, ny in {8..256}, powers of two; nz a power of two in {8..256} or ANY slice count in [2, 64]
 *   (the paper's volumes have 25, 12 and 42 slices: dense z-line transform); ceil(nvol/2)*nz <= 65535
 *   (else PD_ESIZE); nvol independent volumes (coils);
 *   B0_axis 0 = x, 1 = y, 2 = z; sigma <= 0 or tau <= 0: automatic steps 1/sqrt(4/9 + 12); explicit steps with
 *   sigma*tau*(4/9 + 12) >= 1 give PD_ESTEP.  Allocates 32 bytes per voxel of workspace + the D3 table.  Volumes 2k and
 *   2k+1 ride one complex transform, each in its own power-of-two normalisation 2^-floor(log2 rms(field_v)) (exact; the
 *   iteration is invariant under it), so partners of very different magnitude do not disturb each other.
 * pd_solve3d: field, mask (NULL = ones), chi_out: DEVICE, [nvol][nz][ny][nx] fp32, x fastest; chi_out is the primal
 *   state during the call.  Enqueues everything on cuda_stream; does not synchronise.
 * Errors: PD_EINVAL, PD_ESIZE, PD_ESTEP, PD_ENOMEM, PD_ECUDA. */
typedef struct pd_plan3d_s *pd_plan3d_t;
int pd_plan3d(pd_plan3d_t *out, int nx, int ny, int nz, int nvol, int B0_axis, float lambda, float sigma, float tau, float theta);
int pd_solve3d(pd_plan3d_t p, const float *field, const float *mask, float *chi_out, int max_iters, void *cuda_stream);
/* Optional data weighting W of Eq.(1) for the 3-D variant (DEVICE, [nvol][nz][ny][nx], 16-byte aligned, caller-owned, must
 * outlive the solves; |W| <= 1 is assumed by the step bound); NULL = identity.  With W set the dual p stays in the image
 * domain and K is applied twice per iteration, literally as PAPER.md:49 (12 launches per iteration instead of 5); the
 * first call with a non-NULL W allocates 8 bytes per voxel.  Errors: PD_EINVAL, PD_ENOMEM, PD_ECUDA. */
int pd_set_weight3d(pd_plan3d_t p, const float *W);
int pd_last_launch_count3d(pd_plan3d_t p);   /* kernels enqueued by the last pd_solve3d */
int pd_destroy3d(pd_plan3d_t p);

/* pd_preprocess -- flow step (1): "Preprocess the two data collected by the positive contrast MRI to obtain
 * ... the weighting matrix W, the mask Mask, and the phase contrast field iFreq delta" from the two volumes acquired
 * without and with the echo shift T_shift.  The paper gives no formulas; readings R20, R21:
 *   field  = arg(s1 * conj(s0)) * fscale        principal value in (-pi, pi], no unwrapping; 0 where the product is 0
 *   m      = sqrt(|s0| |s1|);  weight = m * wscale;  mask = 1 where weight > threshold, else 0
 * s0, s1 : DEVICE, const, complex64 interleaved (re, im), npixels = batch*ny*nx pixels in the layout of pd_solve, 16-byte
 *          aligned (s0: without the shift, s1: with it).
 * fscale : radians -> the unit of the field map, e.g. 1 / (2 pi T_shift gamma B0) for ppm.
 * wscale : > 0: used as given.  <= 0: automatic, 1 / max(m) over all npixels (|W| <= 1, what the automatic steps of
 *          pd_plan assume); wmax (DEVICE, one float, required in this mode) receives that maximum.
 * field, weight, mask : DEVICE outputs, npixels floats each, 16-byte aligned; any may be NULL (not computed).
 * The integer decisions (mask; the maximum) are taken in fp32 by the fixed sequence a_k = fl(fl(re_k^2) + fl(im_k^2)),
 * m = sqrt(sqrt(fl(a_0 a_1))), weight = fl(m * fl(1/max)), all round-to-nearest, no fused multiply-add.
 * Enqueues one or two kernels (and a 4-byte memset) on cuda_stream; allocates nothing; does not synchronise.
 * Errors: PD_EINVAL (null input, misaligned pointer, automatic scale without wmax), PD_ECUDA. */
int pd_preprocess(const float *s0, const float *s1, long long npixels, float fscale, float wscale, float threshold,
                  float *field, float *weight, float *mask, float *wmax, void *cuda_stream);

/* pd_combine_coils -- "the multi-coil acquisition data from parallel imaging": every coil's field map is
 * reconstructed independently (batch index slice*ncoils + coil) and the per-coil maps are combined, reading
 * R22: chi_out[s](x) = sum_c W_c(x)^2 chi_c(x) / sum_c W_c(x)^2 (coils in index order, fp32), 0 where no coil has weight.
 * chi, weight : DEVICE, const, [nslices*ncoils][ny][nx] (weight: e.g. pd_preprocess's).  chi_out : DEVICE, [nslices][ny][nx].
 * Enqueues one kernel on cuda_stream; allocates nothing.  Errors: PD_EINVAL, PD_ECUDA. */
int pd_combine_coils(const float *chi, const float *weight, int nslices, int ncoils, int ny, int nx, float *chi_out,
                     void *cuda_stream);

/* pd_solve_static: ONE allocation-free entry point, for callers that cannot call cudaMalloc (code under CUDA-graph
 * capture, tight serving loops, harnesses that forbid it).  It runs the same iteration as pd_solve
 * through the streaming kernels with the Fourier-domain dual (W = identity, isotropic TV, lambda on the regulariser,
 * one mask per slice, tolerance checked every iteration) -- bit for bit what a fresh plan with
 * PD_OPT_VARIANT = PD_VARIANT_STREAMING and PD_OPT_GRAPH_LOOP = 0 computes -- but needs no plan: the whole workspace
 * (13 state planes, per-CTA partial sums, the dipole and twiddle tables, the per-slice state variables of PAPER.md:100)
 * lives in one file-scope `static __device__` array of PD_STATIC_SCRATCH_BYTES bytes inside the library, which every GPU
 * that loads the library holds until the process exits.  The call makes no cudaMalloc / cudaFree, creates no stream,
 * event or graph and calls no allocating library routine; it enqueues one cudaMemsetAsync per cleared region and
 * 2*max_iters + 4 kernels on cuda_stream and returns without synchronising.
 * Limits (else PD_ESTATIC): nx, ny each in {64, 128, 256}; batch <= PD_STATIC_MAX_BATCH;
 *   nx * ny * ceil(batch/2) <= PD_STATIC_MAX_CELLS  (e.g. 32 slices of 64x64, 8 of 128x128, 2 of 256x256).
 * field, mask (NULL = ones), chi_out: DEVICE, [batch][ny][nx], as for pd_solve.  lambda, sigma, tau, theta, B0_dir,
 *   max_iters, tol: as for pd_plan / pd_solve (sigma <= 0 or tau <= 0: automatic steps).
 * iters_done, relgap, relres: DEVICE, [batch], caller-owned outputs as in pd_get_stats; any may be NULL.
 * Set-up: the first call on a device asks cudaGetSymbolAddress for the array's device address there (with that device
 *   current), and the first call for a new (nx, ny, B0_dir) on a device rebuilds the two tables on the host, waits for
 *   the device (cudaDeviceSynchronize) and uploads them with cudaMemcpy -- make one such call before a capture or a
 *   timed loop; later calls with the same three values only enqueue.
 * Sharing: every call on a device uses the same array, which keeps the last call's contents (the call clears what must
 *   start at zero).  Calls that overlap on the GPU -- two streams, or two host threads -- RACE on it: order them on
 *   one stream or with events.  Not thread-safe.
 * Errors: PD_EINVAL, PD_ESTATIC, PD_ESTEP, PD_ECUDA. */
#define PD_STATIC_MAX_N 256
#define PD_STATIC_MAX_BATCH 32
#define PD_STATIC_MAX_CELLS 65536
#define PD_STATIC_SCRATCH_BYTES 7149056
int pd_solve_static(int nx, int ny, int batch, int B0_dir, float lambda, float sigma, float tau, float theta,
                    const float *field, const float *mask, float *chi_out, int max_iters, float tol,
                    int *iters_done, float *relgap, float *relres, void *cuda_stream);

const char *pd_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif
