/*
 * pd_oracle.h -- C ABI of the CPU oracle for the primal-dual (PD) positive-contrast
 * susceptibility reconstruction of arXiv 2006.09808.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or constant generator with the CUDA path under
 * paper_2006_09808_b200/csrc/, and neither includes the other.
 *
 * Everything here is plain, slow, single-threaded C++ written from PAPER.md
 * (Eq. (1), pseudo-code PAPER.md:44-49) and the readings R1..R17 listed
 * in DESIGN.md.  Layout everywhere: one slice = ny rows of nx columns, x fastest,
 * a[b][y][x] at (b*ny + y)*nx + x.
 *
 * Pin status (tests/test_oracle_pins.py):
 *   FFT2 ............ pinned (brute-force O(N^4) DFT, numpy.fft)
 *   dipole D ........ pinned (closed-form values on the axes, symmetry, range)
 *   K, G, Gt ........ pinned (adjointness, zero-sum invariants, analytic field of a disc)
 *   prox steps ...... pinned (closed forms / optimality conditions)
 *   PD iteration .... pinned (closed-form first iterate, per-frequency recurrence at
 *                     alpha=0, dense-matrix brute force on 8x8, zero-mean invariant,
 *                     monotone proximal-point distance, convention A == rescaled B)
 *   l1-on-chi variant (PDO_REG_L1) and oblique in-plane B0 (PDO_B0_ANGLE): pinned (prox optimality,
 *                     closed-form first iterate, dense-matrix brute force, LASSO optimality at the fixed
 *                     point, alpha=0 reduction to the TV path; axis angles reduce to PDO_B0_X / PDO_B0_Y,
 *                     45 degree closed-form values, rotated analytic field of a disc)
 *   reconstruction QUALITY on real data: parity unpinned (the paper prints no number).
 */
#ifndef PD_ORACLE_H
#define PD_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

enum { PDO_B0_X = 0, PDO_B0_Y = 1,
       PDO_B0_ANGLE = 2 /* in-plane unit vector (cos a, sin a), a = b0_angle: k_b = kx cos a + ky sin a */ };
enum { PDO_REG_TV = 0,  /* the paper's regulariser ||M G chi||_1 with the dual q (reading R1) */
       PDO_REG_L1 = 1   /* plain l1 on chi, lambda ||M chi||_1: no q, the primal step ends in a soft shrinkage
                           (BASELINE.json north_star: "lambda ||chi||_1 ... the prox (clip onto the lambda-ball, or shrinkage)") */ };
enum { PDO_TV_ISO = 0, PDO_TV_ANISO = 1 };
enum { PDO_LAMBDA_REG = 0,  /* "convention B": 1/2||W(K chi - phi)||^2 + lambda ||M G chi||_1 (BASELINE.json north_star) */
       PDO_LAMBDA_DATA = 1  /* "convention A": lambda/2 ||...||^2 + ||M G chi||_1, literally PAPER.md:37,49 */ };

typedef struct {
    int nx, ny, batch;
    int b0_dir;        /* PDO_B0_X: k_b = kx ; PDO_B0_Y: k_b = ky (frequency along the slow/row axis) */
    double lambda;     /* regularisation parameter (meaning depends on lambda_conv) */
    double sigma, tau, theta;
    int max_iters;     /* N of "Until n >= N" */
    double tol;        /* <= 0: exactly max_iters iterations ; > 0: stop a slice when relgap < tol */
    int tv_mode;       /* PDO_TV_ISO / PDO_TV_ANISO (reading R4) */
    int lambda_conv;   /* PDO_LAMBDA_REG / PDO_LAMBDA_DATA (reading R2) */
    int check_every;   /* tolerance is tested when (n+1) % check_every == 0 */
    int regulariser;   /* PDO_REG_TV (default 0) / PDO_REG_L1 */
    double b0_angle;   /* radians from the x axis, used when b0_dir == PDO_B0_ANGLE (0 = PDO_B0_X, pi/2 = PDO_B0_Y) */
} pdo_params;

/* 2-D DFT, unnormalised forward, 1/(nx*ny)-scaled inverse.  Textbook iterative radix-2
 * along each axis when that length is a power of two, naive O(n^2) DFT per line otherwise. */
int pdo_fft2(int nx, int ny, const double *in_re, const double *in_im,
             double *out_re, double *out_im, int inverse);
/* The definition of the 2-D DFT written out as the quadruple loop, O((nx*ny)^2). */
int pdo_dft2_bruteforce(int nx, int ny, const double *in_re, const double *in_im,
                        double *out_re, double *out_im, int inverse);

/* D(kx,ky) = 1/3 - k_b^2/(kx^2+ky^2), D(0,0)=0 (BASELINE.json north_star; reading R6). */
int pdo_dipole(int nx, int ny, int b0_dir, double *D);
/* K(a) = Re(IFFT2(D .* FFT2(a))) ("dipole kernel convolution operator"). */
int pdo_apply_K(int nx, int ny, int b0_dir, const double *a, double *out);
/* The same two for an in-plane B0 direction at `angle` radians from the x axis: k_b = kx cos(angle) + ky sin(angle). */
int pdo_dipole_angle(int nx, int ny, double angle, double *D);
int pdo_apply_K_angle(int nx, int ny, double angle, const double *a, double *out);
/* Soft shrinkage, the prox of t*|.|: v <- sign(v) max(|v| - t[i], 0), per element (PDO_REG_L1). */
int pdo_shrink(int n, double *v, const double *t);
/* Forward differences with Neumann boundary, and the exact adjoint (reading R7). */
int pdo_grad(int nx, int ny, const double *a, double *gx, double *gy);
int pdo_gradT(int nx, int ny, const double *qx, const double *qy, double *out);
/* prox_sigma[F1*]: p <- (p + sigma*r)/(1+sigma)  [REG]  or /(1+sigma/lambda) [DATA]  (PAPER.md:49 line 1). */
int pdo_prox_p(int n, double *p, const double *r, double sigma, double lambda, int lambda_conv);
/* prox_sigma[F2*]: projection of t=(tx,ty) onto the radius ball, per pixel (PAPER.md:49 line 2). */
int pdo_prox_q(int n, double *tx, double *ty, double radius, int tv_mode);

/* The PD iteration, slice after slice ("a loop is added to the outside").
 * field, mask, weight: fp32 [batch][ny][nx]; mask/weight may be NULL (= all ones).
 * chi_out64 (may be NULL), chi_out32 (may be NULL): [batch][ny][nx].
 * iters_done: [batch].  relgap_hist, relres_hist (may be NULL): [batch][max_iters], entry n holds the
 * value computed in iteration n (0-based), i.e. relgap_{n+1}; unused entries are set to -1.
 * p_out, qx_out, qy_out, chibar_out (may be NULL): final dual / extrapolated state, [batch][ny][nx].
 * Arithmetic in double (pdo_solve_f64) or float (pdo_solve_f32, the one that is timed). */
int pdo_solve_f64(const pdo_params *prm, const float *field, const float *mask, const float *weight,
                  double *chi_out64, float *chi_out32, int *iters_done,
                  double *relgap_hist, double *relres_hist,
                  double *p_out, double *qx_out, double *qy_out, double *chibar_out);
int pdo_solve_f32(const pdo_params *prm, const float *field, const float *mask, const float *weight,
                  double *chi_out64, float *chi_out32, int *iters_done,
                  double *relgap_hist, double *relres_hist,
                  double *p_out, double *qx_out, double *qy_out, double *chibar_out);

/* Single slice, double, stores every iterate: trace[n][c][y][x] for n=0..max_iters,
 * c = 0:chi_n 1:p_n 2:qx_n 3:qy_n (n=0 is the zero initialisation). tol is ignored. */
int pdo_trace_f64(const pdo_params *prm, const float *field, const float *mask, const float *weight,
                  double *trace);

/* Off-path helper for the sphere pin (P11): 3-D forward model on an n^3 grid, B0 along z (slowest axis),
 * D3 = 1/3 - kz^2/|k|^2, D3(0)=0.  Never used by the PD iteration. */
int pdo_forward3d(int n, const double *chi, double *out);

#ifdef __cplusplus
}
#endif
#endif
