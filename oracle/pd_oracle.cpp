/*
 * pd_oracle.cpp -- plain single-threaded CPU oracle for the PD iteration of arXiv 2006.09808.
 *
 * TEST INFRASTRUCTURE ONLY (see pd_oracle.h).  No blocking, fusion or reordering beyond what
 * the paper's pseudo-code states: every operator is applied to a whole slice
 * as its own loop, in the paper's order and notation, so it can be checked against the paper
 * by eye.  Shares nothing with the CUDA path.
 *
 * Symbols follow the paper: chi (primal), chibar (extrapolated primal), p in Y (field space),
 * q in V (gradient vector space, two in-plane components), D dipole kernel, W weighting,
 * M mask, G gradient, phi = Delta B local field, sigma/tau/theta step parameters.
 */
#include "pd_oracle.h"

#include <cmath>
#include <cstddef>
#include <cstring>
#include <vector>

namespace {

const double kPi = 3.14159265358979323846264338327950288;

template <class T>
struct Cpx {
    T re, im;
};

inline bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

/* ---- 1-D DFT of a strided line ------------------------------------------------------------
 * X[k] = sum_n x[n] exp(-+ 2 pi i n k / len)   (minus: forward, plus: inverse; no scaling here).
 * Power of two: the textbook iterative radix-2 decimation-in-time FFT (bit reversal, then
 * butterflies of span 2,4,...,len).  Otherwise: the O(len^2) definition. */
template <class T>
void dft_line(Cpx<T> *a, int len, std::ptrdiff_t stride, bool inverse, std::vector<Cpx<T>> &tmp) {
    tmp.resize(len);
    for (int n = 0; n < len; ++n) tmp[n] = a[n * stride];
    const double sgn = inverse ? +1.0 : -1.0;
    if (is_pow2(len)) {
        for (int i = 1, j = 0; i < len; ++i) { /* bit-reversal permutation */
            int bit = len >> 1;
            for (; j & bit; bit >>= 1) j ^= bit;
            j ^= bit;
            if (i < j) {
                Cpx<T> t = tmp[i];
                tmp[i] = tmp[j];
                tmp[j] = t;
            }
        }
        for (int span = 2; span <= len; span <<= 1) {
            const int half = span >> 1;
            for (int base = 0; base < len; base += span) {
                for (int k = 0; k < half; ++k) {
                    const double ang = sgn * 2.0 * kPi * (double)k / (double)span;
                    const T wr = (T)std::cos(ang), wi = (T)std::sin(ang);
                    Cpx<T> &u = tmp[base + k];
                    Cpx<T> &v = tmp[base + k + half];
                    const T tr = v.re * wr - v.im * wi;
                    const T ti = v.re * wi + v.im * wr;
                    v.re = u.re - tr;
                    v.im = u.im - ti;
                    u.re = u.re + tr;
                    u.im = u.im + ti;
                }
            }
        }
        for (int n = 0; n < len; ++n) a[n * stride] = tmp[n];
    } else {
        std::vector<Cpx<T>> out(len);
        for (int k = 0; k < len; ++k) {
            T sr = 0, si = 0;
            for (int n = 0; n < len; ++n) {
                const long long nk = ((long long)n * k) % len;
                const double ang = sgn * 2.0 * kPi * (double)nk / (double)len;
                const T wr = (T)std::cos(ang), wi = (T)std::sin(ang);
                sr += tmp[n].re * wr - tmp[n].im * wi;
                si += tmp[n].re * wi + tmp[n].im * wr;
            }
            out[k].re = sr;
            out[k].im = si;
        }
        for (int n = 0; n < len; ++n) a[n * stride] = out[n];
    }
}

/* 2-D DFT in place: every row (along x), then every column (along y).  Inverse scaled by 1/(nx*ny). */
template <class T>
void fft2_inplace(Cpx<T> *a, int nx, int ny, bool inverse) {
    std::vector<Cpx<T>> tmp;
    for (int y = 0; y < ny; ++y) dft_line(a + (std::ptrdiff_t)y * nx, nx, 1, inverse, tmp);
    for (int x = 0; x < nx; ++x) dft_line(a + x, ny, nx, inverse, tmp);
    if (inverse) {
        const T s = (T)(1.0 / ((double)nx * (double)ny));
        for (std::ptrdiff_t i = 0; i < (std::ptrdiff_t)nx * ny; ++i) {
            a[i].re *= s;
            a[i].im *= s;
        }
    }
}

/* Signed DFT frequency index: 0,1,...,n/2-1,-n/2,...,-1 (reading R6: index n/2 maps to -n/2). */
inline int signed_index(int i, int n) { return (i < (n + 1) / 2) ? i : i - n; }

/* Dipole kernel in the in-plane form fixed by BASELINE.json north_star:
 * D(kx,ky) = 1/3 - k_b^2/(kx^2+ky^2), D(0,0) = 0, kx = fi/nx, ky = fj/ny cycles per pixel. */
template <class T>
void dipole_table(int nx, int ny, int b0_dir, T *D, double b0_angle = 0.0) {
    /* PDO_B0_ANGLE: B0 along the in-plane unit vector (cos a, sin a); a = 0 is PDO_B0_X, a = pi/2 is PDO_B0_Y */
    const double bx = std::cos(b0_angle), by = std::sin(b0_angle);
    for (int j = 0; j < ny; ++j) {
        for (int i = 0; i < nx; ++i) {
            const double kx = (double)signed_index(i, nx) / (double)nx;
            const double ky = (double)signed_index(j, ny) / (double)ny;
            const double k2 = kx * kx + ky * ky;
            const double kb = (b0_dir == PDO_B0_ANGLE) ? kx * bx + ky * by : (b0_dir == PDO_B0_Y) ? ky : kx;
            D[(std::ptrdiff_t)j * nx + i] = (i == 0 && j == 0) ? (T)0 : (T)(1.0 / 3.0 - kb * kb / k2);
        }
    }
}

/* K(a) = Re( IFFT2( D .* FFT2(a) ) ). */
template <class T>
void apply_K(int nx, int ny, const T *D, const T *a, T *out, std::vector<Cpx<T>> &work) {
    const std::ptrdiff_t P = (std::ptrdiff_t)nx * ny;
    work.resize(P);
    for (std::ptrdiff_t i = 0; i < P; ++i) {
        work[i].re = a[i];
        work[i].im = 0;
    }
    fft2_inplace(work.data(), nx, ny, false);
    for (std::ptrdiff_t i = 0; i < P; ++i) {
        work[i].re *= D[i];
        work[i].im *= D[i];
    }
    fft2_inplace(work.data(), nx, ny, true);
    for (std::ptrdiff_t i = 0; i < P; ++i) out[i] = work[i].re;
}

/* G: forward differences, Neumann boundary (difference across the last column / row is 0). */
template <class T>
void grad(int nx, int ny, const T *a, T *gx, T *gy) {
    for (int y = 0; y < ny; ++y)
        for (int x = 0; x < nx; ++x) {
            const std::ptrdiff_t i = (std::ptrdiff_t)y * nx + x;
            gx[i] = (x < nx - 1) ? a[i + 1] - a[i] : (T)0;
            gy[i] = (y < ny - 1) ? a[i + nx] - a[i] : (T)0;
        }
}

/* G^T (= -div): exact adjoint of grad above. */
template <class T>
void gradT(int nx, int ny, const T *qx, const T *qy, T *out) {
    for (int y = 0; y < ny; ++y)
        for (int x = 0; x < nx; ++x) {
            const std::ptrdiff_t i = (std::ptrdiff_t)y * nx + x;
            T s = 0;
            if (x > 0) s += qx[i - 1];
            if (x < nx - 1) s -= qx[i];
            if (y > 0) s += qy[i - nx];
            if (y < ny - 1) s -= qy[i];
            out[i] = s;
        }
}

/* prox_sigma[F1*] (PAPER.md:49 line 1).  DATA: literally /(1+sigma/lambda).  REG: /(1+sigma). */
template <class T>
void prox_p(std::ptrdiff_t n, T *p, const T *r, T sigma, T lambda, int lambda_conv) {
    const T denom = (lambda_conv == PDO_LAMBDA_DATA) ? (T)1 + sigma / lambda : (T)1 + sigma;
    for (std::ptrdiff_t i = 0; i < n; ++i) p[i] = (p[i] + sigma * r[i]) / denom;
}

/* prox_sigma[F2*] (PAPER.md:49 line 2): t / max(1, |t|/radius), written so that radius = 0 gives 0
 * without dividing by it (reading R13).  ISO: |t| is the Euclidean norm of the two components at a
 * pixel; ANISO: each component clamped to [-radius, radius] (reading R4). */
template <class T>
void prox_q(std::ptrdiff_t n, T *tx, T *ty, T radius, int tv_mode) {
    for (std::ptrdiff_t i = 0; i < n; ++i) {
        if (tv_mode == PDO_TV_ANISO) {
            tx[i] = tx[i] > radius ? radius : (tx[i] < -radius ? -radius : tx[i]);
            ty[i] = ty[i] > radius ? radius : (ty[i] < -radius ? -radius : ty[i]);
        } else {
            const T nrm = std::sqrt(tx[i] * tx[i] + ty[i] * ty[i]);
            const T s = (nrm > radius) ? radius / nrm : (T)1;
            tx[i] *= s;
            ty[i] *= s;
        }
    }
}

/* Soft shrinkage: the prox of t*|.| (PDO_REG_L1; BASELINE.json north_star "or shrinkage"). */
template <class T>
void shrink(std::ptrdiff_t n, T *v, const T *t) {
    for (std::ptrdiff_t i = 0; i < n; ++i) {
        const T a = std::fabs(v[i]) - t[i];
        v[i] = (a > 0) ? (v[i] > 0 ? a : -a) : (T)0;
    }
}

/* One slice of the PD iteration, steps in the paper's order. */
template <class T>
struct SliceSolver {
    int nx, ny;
    std::ptrdiff_t P;
    std::vector<T> D, phi, M, W;
    std::vector<T> chi, chibar, p, qx, qy;
    std::vector<T> u, r, gx, gy, wp, v, mqx, mqy, d, chinew;
    std::vector<Cpx<T>> work;
    T sigma, tau, theta, lambda;
    int tv_mode, lambda_conv, regulariser;
    std::vector<T> thr;   /* PDO_REG_L1: shrinkage threshold tau * radius * M per pixel */
    T radius;   /* ball of the q-projection: lambda (REG) or 1 (DATA) */
    double P0;  /* normaliser of relgap: primal objective at chi = 0 */

    void init(const pdo_params &prm, const float *field, const float *mask, const float *weight) {
        nx = prm.nx;
        ny = prm.ny;
        P = (std::ptrdiff_t)nx * ny;
        sigma = (T)prm.sigma;
        tau = (T)prm.tau;
        theta = (T)prm.theta;
        lambda = (T)prm.lambda;
        tv_mode = prm.tv_mode;
        lambda_conv = prm.lambda_conv;
        regulariser = prm.regulariser;
        radius = (lambda_conv == PDO_LAMBDA_DATA) ? (T)1 : lambda;
        D.resize(P);
        dipole_table(nx, ny, prm.b0_dir, D.data(), prm.b0_angle);
        phi.resize(P);
        M.resize(P);
        W.resize(P);
        for (std::ptrdiff_t i = 0; i < P; ++i) {
            phi[i] = (T)field[i];
            M[i] = mask ? (T)mask[i] : (T)1;
            W[i] = weight ? (T)weight[i] : (T)1;
        }
        /* step 2-3: chi_0 = p_0 = q_0 = 0, chibar_0 = chi_0 */
        chi.assign(P, 0);
        chibar.assign(P, 0);
        p.assign(P, 0);
        qx.assign(P, 0);
        qy.assign(P, 0);
        for (auto *vec : {&u, &r, &gx, &gy, &wp, &v, &mqx, &mqy, &d, &chinew}) vec->assign(P, 0);
        double s = 0;
        for (std::ptrdiff_t i = 0; i < P; ++i) {
            const double wphi = (double)(W[i] * phi[i]);
            s += wphi * wphi;
        }
        P0 = 0.5 * s * ((lambda_conv == PDO_LAMBDA_DATA) ? (double)lambda : 1.0);
        thr.resize(P);
        for (std::ptrdiff_t i = 0; i < P; ++i) thr[i] = tau * radius * M[i];
    }

    /* PDO_REG_L1: min 1/2||W(K chi - phi)||^2 + radius*||M chi||_1 (north_star's alternative regulariser).  The same
     * first-order primal-dual iteration with K_full = W K only: p as in PAPER.md:49 line 1, no q, and the primal step
     * chi_{n+1} = prox_{tau G}(chi_n - tau K W p_{n+1}) with G = radius*||M .||_1, whose prox is the soft shrinkage.
     * relgap: the Fenchel-Young gap of the data term alone (the q part of reading R9 does not exist here). */
    void iterate_l1(double *relgap, double *relres) {
        apply_K(nx, ny, D.data(), chibar.data(), u.data(), work);
        for (std::ptrdiff_t i = 0; i < P; ++i) r[i] = W[i] * (u[i] - phi[i]);
        prox_p(P, p.data(), r.data(), sigma, lambda, lambda_conv);
        double gap_p = 0;
        for (std::ptrdiff_t i = 0; i < P; ++i) {
            if (lambda_conv == PDO_LAMBDA_DATA) {
                const double e = (double)lambda * (double)r[i] - (double)p[i];
                gap_p += e * e / (2.0 * (double)lambda);
            } else {
                const double e = (double)r[i] - (double)p[i];
                gap_p += 0.5 * e * e;
            }
        }
        *relgap = (P0 > 0) ? gap_p / P0 : 0.0;
        for (std::ptrdiff_t i = 0; i < P; ++i) wp[i] = W[i] * p[i];
        apply_K(nx, ny, D.data(), wp.data(), v.data(), work);
        for (std::ptrdiff_t i = 0; i < P; ++i) chinew[i] = chi[i] - tau * v[i];
        shrink(P, chinew.data(), thr.data());
        double dn = 0, cn = 0;
        for (std::ptrdiff_t i = 0; i < P; ++i) {
            const double dd = (double)chinew[i] - (double)chi[i];
            dn += dd * dd;
            cn += (double)chinew[i] * (double)chinew[i];
        }
        const double cnorm = std::sqrt(cn);
        *relres = std::sqrt(dn) / (cnorm > 1e-300 ? cnorm : 1e-300);
        for (std::ptrdiff_t i = 0; i < P; ++i) {
            chibar[i] = chinew[i] + theta * (chinew[i] - chi[i]);
            chi[i] = chinew[i];
        }
    }

    /* One pass of the Repeat body.  Returns relgap_{n+1} and relres_{n+1} (readings R9). */
    void iterate(double *relgap, double *relres) {
        if (regulariser == PDO_REG_L1) { iterate_l1(relgap, relres); return; }
        /* p_{n+1} = (p_n + sigma*(W(D chibar_n - Delta B))) / (1 + sigma[/lambda])   (residual per Eq.(1), reading R3) */
        apply_K(nx, ny, D.data(), chibar.data(), u.data(), work);
        for (std::ptrdiff_t i = 0; i < P; ++i) r[i] = W[i] * (u[i] - phi[i]);
        prox_p(P, p.data(), r.data(), sigma, lambda, lambda_conv);

        /* q_{n+1} = (q_n + sigma*M G chibar_n) / max(1, |q_n + sigma*M G chibar_n|) */
        grad(nx, ny, chibar.data(), gx.data(), gy.data());
        for (std::ptrdiff_t i = 0; i < P; ++i) {
            gx[i] *= M[i];
            gy[i] *= M[i];
            qx[i] += sigma * gx[i];
            qy[i] += sigma * gy[i];
        }
        prox_q(P, qx.data(), qy.data(), radius, tv_mode);

        /* Fenchel-Young gap of F at (K_full chibar_n, y_{n+1}), normalised by P0 (reading R9), new p and q. */
        double gap_p = 0, gap_q = 0;
        for (std::ptrdiff_t i = 0; i < P; ++i) {
            if (lambda_conv == PDO_LAMBDA_DATA) {
                const double e = (double)lambda * (double)r[i] - (double)p[i];
                gap_p += e * e / (2.0 * (double)lambda);
            } else {
                const double e = (double)r[i] - (double)p[i];
                gap_p += 0.5 * e * e;
            }
            const double gxi = gx[i], gyi = gy[i];
            const double gn = (tv_mode == PDO_TV_ANISO) ? std::fabs(gxi) + std::fabs(gyi)
                                                        : std::sqrt(gxi * gxi + gyi * gyi);
            gap_q += (double)radius * gn - gxi * (double)qx[i] - gyi * (double)qy[i];
        }
        *relgap = (P0 > 0) ? (gap_p + gap_q) / P0 : 0.0;

        /* chi_{n+1} = chi_n - tau*(D* W* p_{n+1}) - tau*(G* M* q_{n+1}) */
        for (std::ptrdiff_t i = 0; i < P; ++i) wp[i] = W[i] * p[i];
        apply_K(nx, ny, D.data(), wp.data(), v.data(), work);
        for (std::ptrdiff_t i = 0; i < P; ++i) {
            mqx[i] = M[i] * qx[i];
            mqy[i] = M[i] * qy[i];
        }
        gradT(nx, ny, mqx.data(), mqy.data(), d.data());
        double dn = 0, cn = 0;
        for (std::ptrdiff_t i = 0; i < P; ++i) {
            chinew[i] = chi[i] - tau * v[i] - tau * d[i];
            const double dd = (double)chinew[i] - (double)chi[i];
            dn += dd * dd;
            cn += (double)chinew[i] * (double)chinew[i];
        }
        const double cnorm = std::sqrt(cn);
        *relres = std::sqrt(dn) / (cnorm > 1e-300 ? cnorm : 1e-300);

        /* chibar_{n+1} = chi_{n+1} + theta*(chi_{n+1} - chi_n) ; n = n + 1 */
        for (std::ptrdiff_t i = 0; i < P; ++i) {
            chibar[i] = chinew[i] + theta * (chinew[i] - chi[i]);
            chi[i] = chinew[i];
        }
    }
};

template <class T>
int solve_impl(const pdo_params *prm, const float *field, const float *mask, const float *weight,
               double *chi_out64, float *chi_out32, int *iters_done, double *relgap_hist,
               double *relres_hist, double *p_out, double *qx_out, double *qy_out, double *chibar_out) {
    if (!prm || !field || prm->nx < 1 || prm->ny < 1 || prm->batch < 1 || prm->max_iters < 0) return -1;
    const std::ptrdiff_t P = (std::ptrdiff_t)prm->nx * prm->ny;
    const int check_every = prm->check_every > 0 ? prm->check_every : 1;
    SliceSolver<T> s;
    /* "a loop is added to the outside of the iterative calculation": slice after slice */
    for (int b = 0; b < prm->batch; ++b) {
        s.init(*prm, field + b * P, mask ? mask + b * P : nullptr, weight ? weight + b * P : nullptr);
        if (relgap_hist)
            for (int n = 0; n < prm->max_iters; ++n) relgap_hist[(std::ptrdiff_t)b * prm->max_iters + n] = -1.0;
        if (relres_hist)
            for (int n = 0; n < prm->max_iters; ++n) relres_hist[(std::ptrdiff_t)b * prm->max_iters + n] = -1.0;
        int n = 0;
        if (!(prm->tol > 0 && s.P0 == 0)) { /* reading R13b: an all-zero slice stops at once when a tolerance is set */
            while (n < prm->max_iters) {
                double relgap, relres;
                s.iterate(&relgap, &relres);
                if (relgap_hist) relgap_hist[(std::ptrdiff_t)b * prm->max_iters + n] = relgap;
                if (relres_hist) relres_hist[(std::ptrdiff_t)b * prm->max_iters + n] = relres;
                ++n;
                if (prm->tol > 0 && (n % check_every) == 0 && relgap < prm->tol) break;
            }
        }
        if (iters_done) iters_done[b] = n;
        for (std::ptrdiff_t i = 0; i < P; ++i) {
            if (chi_out64) chi_out64[b * P + i] = (double)s.chi[i];
            if (chi_out32) chi_out32[b * P + i] = (float)s.chi[i];
            if (p_out) p_out[b * P + i] = (double)s.p[i];
            if (qx_out) qx_out[b * P + i] = (double)s.qx[i];
            if (qy_out) qy_out[b * P + i] = (double)s.qy[i];
            if (chibar_out) chibar_out[b * P + i] = (double)s.chibar[i];
        }
    }
    return 0;
}

}  // namespace

extern "C" {

int pdo_fft2(int nx, int ny, const double *in_re, const double *in_im, double *out_re, double *out_im,
             int inverse) {
    if (nx < 1 || ny < 1 || !in_re || !out_re || !out_im) return -1;
    const std::ptrdiff_t P = (std::ptrdiff_t)nx * ny;
    std::vector<Cpx<double>> a(P);
    for (std::ptrdiff_t i = 0; i < P; ++i) {
        a[i].re = in_re[i];
        a[i].im = in_im ? in_im[i] : 0.0;
    }
    fft2_inplace(a.data(), nx, ny, inverse != 0);
    for (std::ptrdiff_t i = 0; i < P; ++i) {
        out_re[i] = a[i].re;
        out_im[i] = a[i].im;
    }
    return 0;
}

int pdo_dft2_bruteforce(int nx, int ny, const double *in_re, const double *in_im, double *out_re,
                        double *out_im, int inverse) {
    if (nx < 1 || ny < 1 || !in_re || !out_re || !out_im) return -1;
    const double sgn = inverse ? +1.0 : -1.0;
    const double scale = inverse ? 1.0 / ((double)nx * ny) : 1.0;
    for (int ky = 0; ky < ny; ++ky)
        for (int kx = 0; kx < nx; ++kx) {
            double sr = 0, si = 0;
            for (int y = 0; y < ny; ++y)
                for (int x = 0; x < nx; ++x) {
                    const double ang =
                        sgn * 2.0 * kPi * ((double)((long long)x * kx % nx) / nx + (double)((long long)y * ky % ny) / ny);
                    const double wr = std::cos(ang), wi = std::sin(ang);
                    const double ar = in_re[(std::ptrdiff_t)y * nx + x];
                    const double ai = in_im ? in_im[(std::ptrdiff_t)y * nx + x] : 0.0;
                    sr += ar * wr - ai * wi;
                    si += ar * wi + ai * wr;
                }
            out_re[(std::ptrdiff_t)ky * nx + kx] = sr * scale;
            out_im[(std::ptrdiff_t)ky * nx + kx] = si * scale;
        }
    return 0;
}

int pdo_dipole(int nx, int ny, int b0_dir, double *D) {
    if (nx < 1 || ny < 1 || !D) return -1;
    dipole_table(nx, ny, b0_dir, D);
    return 0;
}

int pdo_apply_K(int nx, int ny, int b0_dir, const double *a, double *out) {
    if (nx < 1 || ny < 1 || !a || !out) return -1;
    std::vector<double> D((std::ptrdiff_t)nx * ny);
    dipole_table(nx, ny, b0_dir, D.data());
    std::vector<Cpx<double>> work;
    apply_K(nx, ny, D.data(), a, out, work);
    return 0;
}

int pdo_dipole_angle(int nx, int ny, double angle, double *D) {
    if (nx < 1 || ny < 1 || !D) return -1;
    dipole_table(nx, ny, PDO_B0_ANGLE, D, angle);
    return 0;
}

int pdo_apply_K_angle(int nx, int ny, double angle, const double *a, double *out) {
    if (nx < 1 || ny < 1 || !a || !out) return -1;
    std::vector<double> D((std::ptrdiff_t)nx * ny);
    dipole_table(nx, ny, PDO_B0_ANGLE, D.data(), angle);
    std::vector<Cpx<double>> work;
    apply_K(nx, ny, D.data(), a, out, work);
    return 0;
}

int pdo_shrink(int n, double *v, const double *t) {
    if (n < 0 || !v || !t) return -1;
    shrink<double>(n, v, t);
    return 0;
}

int pdo_grad(int nx, int ny, const double *a, double *gx, double *gy) {
    if (nx < 1 || ny < 1 || !a || !gx || !gy) return -1;
    grad(nx, ny, a, gx, gy);
    return 0;
}

int pdo_gradT(int nx, int ny, const double *qx, const double *qy, double *out) {
    if (nx < 1 || ny < 1 || !qx || !qy || !out) return -1;
    gradT(nx, ny, qx, qy, out);
    return 0;
}

int pdo_prox_p(int n, double *p, const double *r, double sigma, double lambda, int lambda_conv) {
    if (n < 0 || !p || !r) return -1;
    prox_p<double>(n, p, r, sigma, lambda, lambda_conv);
    return 0;
}

int pdo_prox_q(int n, double *tx, double *ty, double radius, int tv_mode) {
    if (n < 0 || !tx || !ty) return -1;
    prox_q<double>(n, tx, ty, radius, tv_mode);
    return 0;
}

int pdo_solve_f64(const pdo_params *prm, const float *field, const float *mask, const float *weight,
                  double *chi_out64, float *chi_out32, int *iters_done, double *relgap_hist,
                  double *relres_hist, double *p_out, double *qx_out, double *qy_out, double *chibar_out) {
    return solve_impl<double>(prm, field, mask, weight, chi_out64, chi_out32, iters_done, relgap_hist,
                              relres_hist, p_out, qx_out, qy_out, chibar_out);
}

int pdo_solve_f32(const pdo_params *prm, const float *field, const float *mask, const float *weight,
                  double *chi_out64, float *chi_out32, int *iters_done, double *relgap_hist,
                  double *relres_hist, double *p_out, double *qx_out, double *qy_out, double *chibar_out) {
    return solve_impl<float>(prm, field, mask, weight, chi_out64, chi_out32, iters_done, relgap_hist,
                             relres_hist, p_out, qx_out, qy_out, chibar_out);
}

int pdo_trace_f64(const pdo_params *prm, const float *field, const float *mask, const float *weight,
                  double *trace) {
    if (!prm || !field || !trace || prm->nx < 1 || prm->ny < 1 || prm->max_iters < 0) return -1;
    const std::ptrdiff_t P = (std::ptrdiff_t)prm->nx * prm->ny;
    SliceSolver<double> s;
    s.init(*prm, field, mask, weight);
    for (int n = 0; n <= prm->max_iters; ++n) {
        double *t = trace + (std::ptrdiff_t)n * 4 * P;
        std::memcpy(t + 0 * P, s.chi.data(), P * sizeof(double));
        std::memcpy(t + 1 * P, s.p.data(), P * sizeof(double));
        std::memcpy(t + 2 * P, s.qx.data(), P * sizeof(double));
        std::memcpy(t + 3 * P, s.qy.data(), P * sizeof(double));
        if (n < prm->max_iters) {
            double relgap, relres;
            s.iterate(&relgap, &relres);
        }
    }
    return 0;
}

int pdo_forward3d(int n, const double *chi, double *out) {
    if (n < 1 || !chi || !out) return -1;
    const std::ptrdiff_t n2 = (std::ptrdiff_t)n * n, n3 = n2 * n;
    std::vector<Cpx<double>> a(n3);
    std::vector<Cpx<double>> tmp;
    for (std::ptrdiff_t i = 0; i < n3; ++i) {
        a[i].re = chi[i];
        a[i].im = 0;
    }
    for (int pass = 0; pass < 2; ++pass) {
        const bool inv = pass == 1;
        for (std::ptrdiff_t l = 0; l < n2; ++l) dft_line(a.data() + l * n, n, 1, inv, tmp);                      /* x */
        for (int z = 0; z < n; ++z)
            for (int x = 0; x < n; ++x) dft_line(a.data() + z * n2 + x, n, n, inv, tmp);                         /* y */
        for (std::ptrdiff_t l = 0; l < n2; ++l) dft_line(a.data() + l, n, n2, inv, tmp);                         /* z */
        if (!inv) {
            for (int kz = 0; kz < n; ++kz)
                for (int ky = 0; ky < n; ++ky)
                    for (int kx = 0; kx < n; ++kx) {
                        const double fx = (double)signed_index(kx, n) / n, fy = (double)signed_index(ky, n) / n,
                                     fz = (double)signed_index(kz, n) / n;
                        const double k2 = fx * fx + fy * fy + fz * fz;
                        const double D3 = (k2 == 0) ? 0.0 : 1.0 / 3.0 - fz * fz / k2;
                        Cpx<double> &c = a[kz * n2 + (std::ptrdiff_t)ky * n + kx];
                        c.re *= D3;
                        c.im *= D3;
                    }
        }
    }
    for (std::ptrdiff_t i = 0; i < n3; ++i) out[i] = a[i].re / (double)n3;
    return 0;
}

}  // extern "C"
