"""Pins of the CPU oracle (oracle/pd_oracle.cpp) to facts the paper and the mathematics fix.

The paper prints no worked numeric example, so every pin is a closed form, an invariant,
a special case that reduces to a library routine (numpy.fft / numpy.linalg), or brute force on a
tiny input.  Pin numbers P1..P14 follow DESIGN.md "Pins".  None of these
tests touches the CUDA path.
"""
import numpy as np
import pytest

from paper_2006_09808_b200 import synth

SIG = 0.25


def rel(a, b):
    return float(np.linalg.norm(np.ravel(a) - np.ravel(b)) / max(np.linalg.norm(np.ravel(b)), 1e-300))


def np_dipole(nx, ny, b0="y"):
    """Closed form typed independently of the oracle (signed integer frequencies, ratio form)."""
    fi = np.array([i if i < nx / 2 else i - nx for i in range(nx)], float)[None, :]
    fj = np.array([j if j < ny / 2 else j - ny for j in range(ny)], float)[:, None]
    a, b = fi * ny, fj * nx  # kx : ky = fi/nx : fj/ny = fi*ny : fj*nx
    den = a * a + b * b
    num = (b * b if b0 == "y" else a * a) + 0 * den
    out = np.zeros((ny, nx))
    out[den > 0] = 1.0 / 3.0 - num[den > 0] / den[den > 0]
    return out


def np_K(a, b0="y"):
    ny, nx = a.shape
    return np.real(np.fft.ifft2(np_dipole(nx, ny, b0) * np.fft.fft2(a)))


def rng(seed):
    return np.random.default_rng(seed)


# ---------------------------------------------------------------- P1: FFT
@pytest.mark.parametrize("ny,nx", [(8, 8), (8, 16), (16, 8), (4, 32), (6, 10)])
def test_P1_fft2_vs_bruteforce_dft(oracle, ny, nx):
    r = rng(1)
    a = r.standard_normal((ny, nx)) + 1j * r.standard_normal((ny, nx))
    # the definition, typed here as dense DFT matrices (axis order matters: catches axis swaps)
    Fy = np.exp(-2j * np.pi * np.outer(np.arange(ny), np.arange(ny)) / ny)
    Fx = np.exp(-2j * np.pi * np.outer(np.arange(nx), np.arange(nx)) / nx)
    ref = Fy @ a @ Fx.T
    assert rel(oracle.fft2(a), ref) < 1e-12
    assert rel(oracle.fft2(a, bruteforce=True), ref) < 1e-12
    assert rel(oracle.fft2(a), np.fft.fft2(a)) < 1e-12
    assert rel(oracle.fft2(a, inverse=True), np.fft.ifft2(a)) < 1e-12
    assert rel(oracle.fft2(a, inverse=True, bruteforce=True), np.fft.ifft2(a)) < 1e-12
    assert rel(oracle.fft2(oracle.fft2(a), inverse=True), a) < 1e-12


def test_P1_fft2_large_pow2_vs_numpy(oracle):
    a = rng(2).standard_normal((128, 256))
    assert rel(oracle.fft2(a), np.fft.fft2(a)) < 1e-12


# ---------------------------------------------------------------- P2: dipole kernel
@pytest.mark.parametrize("ny,nx", [(16, 16), (64, 64), (32, 64), (12, 20)])
def test_P2_dipole_closed_form(oracle, ny, nx):
    Dy = oracle.dipole(nx, ny, oracle.B0_Y)
    Dx = oracle.dipole(nx, ny, oracle.B0_X)
    assert Dy[0, 0] == 0.0 and Dx[0, 0] == 0.0
    assert Dy.min() >= -2.0 / 3.0 - 1e-15 and Dy.max() <= 1.0 / 3.0 + 1e-15
    # on the axis perpendicular to B0 (k_b = 0): 1/3 ; on the B0 axis: 1/3 - 1 = -2/3
    assert np.allclose(Dy[0, 1:], 1.0 / 3.0, atol=1e-15) and np.allclose(Dy[1:, 0], -2.0 / 3.0, atol=1e-15)
    assert np.allclose(Dx[1:, 0], 1.0 / 3.0, atol=1e-15) and np.allclose(Dx[0, 1:], -2.0 / 3.0, atol=1e-15)
    # even: D(k) = D(-k)
    idx_y = (-np.arange(ny)) % ny
    idx_x = (-np.arange(nx)) % nx
    assert np.array_equal(Dy, Dy[idx_y][:, idx_x])
    # the two in-plane directions share 1/3 - kb^2/k^2: Dx + Dy = 2/3 - 1 = -1/3 away from DC
    s = Dx + Dy
    s[0, 0] = -1.0 / 3.0
    assert np.allclose(s, -1.0 / 3.0, atol=1e-15)
    assert np.allclose(Dy, np_dipole(nx, ny, "y"), atol=1e-15)
    if nx == ny:  # swapping B0_dir transposes D
        assert np.array_equal(Dx, Dy.T)
        # on the diagonal kx = ky: 1/3 - 1/2
        assert np.allclose(np.diag(Dy)[1:], -1.0 / 6.0, atol=1e-15)


def test_P2_dipole_only_zero_is_dc(oracle):
    D = oracle.dipole(16, 16, oracle.B0_Y)
    assert np.count_nonzero(D == 0) == 1


# ---------------------------------------------------------------- P3: operators
@pytest.mark.parametrize("ny,nx", [(16, 16), (24, 40), (7, 9)])
def test_P3_adjointness_and_zero_sums(oracle, ny, nx):
    r = rng(3)
    a, b = r.standard_normal((ny, nx)), r.standard_normal((ny, nx))
    qx, qy = r.standard_normal((ny, nx)), r.standard_normal((ny, nx))
    gx, gy = oracle.grad(a)
    lhs = np.sum(gx * qx) + np.sum(gy * qy)
    rhs = np.sum(a * oracle.gradT(qx, qy))
    assert abs(lhs - rhs) < 1e-12 * (abs(lhs) + 1)
    assert abs(np.sum(oracle.gradT(qx, qy))) < 1e-11           # G^T q sums to zero (G kills constants)
    for b0 in (oracle.B0_X, oracle.B0_Y):
        Ka, Kb = oracle.apply_K(a, b0), oracle.apply_K(b, b0)
        assert abs(np.sum(Ka * b) - np.sum(a * Kb)) < 1e-12 * (abs(np.sum(Ka * b)) + 1)   # K symmetric
        assert abs(np.sum(Ka)) < 1e-11                          # D(0,0)=0 removes the mean
    assert rel(oracle.apply_K(a, oracle.B0_Y), np_K(a, "y")) < 1e-12
    assert rel(oracle.apply_K(a, oracle.B0_X), np_K(a, "x")) < 1e-12


def test_P3_grad_explicit_small(oracle):
    a = np.array([[1.0, 4.0, 9.0], [2.0, 3.0, 5.0]])
    gx, gy = oracle.grad(a)
    assert np.array_equal(gx, [[3.0, 5.0, 0.0], [1.0, 2.0, 0.0]])       # Neumann: last column 0
    assert np.array_equal(gy, [[1.0, -1.0, -4.0], [0.0, 0.0, 0.0]])     # last row 0
    # G^T as the transposed dense matrix
    ny, nx = 3, 4
    n = ny * nx
    G = np.zeros((2 * n, n))
    for j in range(n):
        e = np.zeros(n)
        e[j] = 1
        ex, ey = oracle.grad(e.reshape(ny, nx))
        G[:n, j], G[n:, j] = ex.ravel(), ey.ravel()
    q = rng(4).standard_normal(2 * n)
    assert np.allclose(oracle.gradT(q[:n].reshape(ny, nx), q[n:].reshape(ny, nx)).ravel(), G.T @ q, atol=1e-14)
    # ||G||^2 = largest eigenvalue of G^T G = 4 cos^2(pi/2nx) + 4 cos^2(pi/2ny) < 8 (bound used for the steps)
    lam = np.linalg.eigvalsh(G.T @ G).max()
    assert abs(lam - (4 * np.cos(np.pi / (2 * nx)) ** 2 + 4 * np.cos(np.pi / (2 * ny)) ** 2)) < 1e-12


# ---------------------------------------------------------------- P4: prox operators
def test_P4_prox_p_optimality(oracle):
    r = rng(5)
    p, res = r.standard_normal(50), r.standard_normal(50)
    # REG: p+ = argmin_y 1/(2 sigma)||y - p~||^2 + 1/2||y||^2 + <y, W phi>, p~ = p + sigma*W K chibar
    # first-order condition with res = W K chibar - W phi :  (y - p - sigma*res)/sigma + y = 0
    y = oracle.prox_p(p, res, SIG)
    assert np.allclose((y - p - SIG * res) / SIG + y, 0, atol=1e-14)
    # DATA (paper's literal form), F1*(y) = ||y||^2/(2 lambda) + <y, W phi>: (y - p - sigma*res)/sigma + y/lambda = 0
    lam = 0.37
    y = oracle.prox_p(p, res, SIG, lam, oracle.LAMBDA_DATA)
    assert np.allclose((y - p - SIG * res) / SIG + y / lam, 0, atol=1e-13)


def test_P4_prox_q_projection(oracle):
    r = rng(6)
    tx, ty = 3 * r.standard_normal(200), 3 * r.standard_normal(200)
    rad = 1.3
    qx, qy = oracle.prox_q(tx, ty, rad, oracle.TV_ISO)
    nt, nq = np.hypot(tx, ty), np.hypot(qx, qy)
    assert np.all(nq <= rad * (1 + 1e-15))
    inside = nt <= rad
    assert inside.any() and (~inside).any()
    assert np.array_equal(qx[inside], tx[inside]) and np.array_equal(qy[inside], ty[inside])
    assert np.allclose(nq[~inside], rad, rtol=1e-14)
    assert np.allclose(qx * ty, qy * tx, atol=1e-12)           # parallel to t
    assert np.all(qx * tx >= 0)                                  # same direction
    q2x, q2y = oracle.prox_q(qx, qy, rad, oracle.TV_ISO)        # idempotent
    assert np.allclose(q2x, qx, rtol=1e-15) and np.allclose(q2y, qy, rtol=1e-15)
    ax, ay = oracle.prox_q(tx, ty, rad, oracle.TV_ANISO)
    assert np.array_equal(ax, np.clip(tx, -rad, rad)) and np.array_equal(ay, np.clip(ty, -rad, rad))
    zx, zy = oracle.prox_q(tx, ty, 0.0, oracle.TV_ISO)          # radius 0 -> 0, no NaN (R13)
    assert np.array_equal(zx, np.zeros(200)) and np.array_equal(zy, np.zeros(200))
    zx, zy = oracle.prox_q(np.zeros(4), np.zeros(4), 0.0, oracle.TV_ISO)
    assert np.array_equal(zx, np.zeros(4))


# ---------------------------------------------------------------- P5: closed-form first iterate
@pytest.mark.parametrize("with_w", [False, True])
def test_P5_first_iterate_closed_form(oracle, with_w):
    case = synth.random_case(32, 16, 2, seed=1, with_mask=True, with_weight=with_w)
    tau = 0.2
    out = oracle.solve(case["field"], case["mask"], case["weight"], lambda_=0.01, sigma=SIG, tau=tau,
                       max_iters=1, want_state=True)
    for b in range(2):
        phi = case["field"][b].astype(np.float64)
        W = case["weight"][b].astype(np.float64) if with_w else np.ones_like(phi)
        assert rel(out["p"][b], -SIG * W * phi / (1 + SIG)) < 1e-14
        assert np.all(out["qx"][b] == 0) and np.all(out["qy"][b] == 0)
        assert rel(out["chi"][b], SIG * tau / (1 + SIG) * np_K(W * W * phi)) < 1e-12
        assert rel(out["chibar"][b], 2 * out["chi"][b]) < 1e-15      # theta=1, chi_0=0
        assert abs(out["relgap"][b, 0] - 1 / (1 + SIG) ** 2) < 1e-14  # = 0.64 for any phi, W, M
        assert abs(out["relres"][b, 0] - 1.0) < 1e-15


# ---------------------------------------------------------------- P6: alpha = 0 limit
def freq_recurrence(phi, d, sigma, tau, iters):
    """alpha = 0: per frequency, p^ <- (p^ + sigma (d (2c^ - c^prev) - phi^))/(1+sigma), c^ <- c^ - tau d p^."""
    ph = np.fft.fft2(phi)
    c = np.zeros_like(ph)
    cprev = np.zeros_like(ph)
    p = np.zeros_like(ph)
    for _ in range(iters):
        p = (p + sigma * (d * (2 * c - cprev) - ph)) / (1 + sigma)
        cprev, c = c, c - tau * d * p
    return c


@pytest.mark.parametrize("iters", [1, 10, 200])
def test_P6_alpha0_matches_per_frequency_recurrence(oracle, iters):
    n = 16
    phi = synth.random_case(n, n, 1, seed=2, with_mask=False)["field"][0]
    out = oracle.solve(phi, lambda_=0.0, sigma=SIG, tau=SIG, max_iters=iters)
    c = freq_recurrence(phi.astype(np.float64), np_dipole(n, n), SIG, SIG, iters)
    assert rel(out["chi"][0], np.real(np.fft.ifft2(c))) < 1e-12
    assert np.abs(np.imag(np.fft.ifft2(c))).max() < 1e-12


def test_P6_alpha0_limit_is_kspace_least_squares(oracle):
    """lambda=0: the iterate converges to phi^/D where D != 0 (north_star's "lambda=0 limit"); slow near the cone,
    so compare on |D| > 0.3 after 2000 iterations."""
    n = 16
    phi = synth.random_case(n, n, 1, seed=3, with_mask=False)["field"][0]
    out = oracle.solve(phi, lambda_=0.0, sigma=SIG, tau=SIG, max_iters=2000, want_hist=False)
    D = np_dipole(n, n)
    sel = np.abs(D) > 0.3
    ch = np.fft.fft2(out["chi"][0])
    ls = np.fft.fft2(phi.astype(np.float64))[sel] / D[sel]
    assert rel(ch[sel], ls) < 1e-10
    assert abs(ch[0, 0]) < 1e-10                                  # DC stays 0


# ---------------------------------------------------------------- P7: zero-mean invariant
def test_P7_zero_mean_every_iterate(oracle):
    case = synth.random_case(24, 20, 1, seed=4, with_mask=True, with_weight=True)
    tr = oracle.trace(case["field"][0], case["mask"][0], case["weight"][0], lambda_=0.5, sigma=SIG, tau=SIG,
                      max_iters=40)
    sums = tr[:, 0].sum(axis=(1, 2))
    scale = np.abs(tr[:, 0]).sum(axis=(1, 2)).max()
    assert np.abs(sums).max() < 1e-12 * scale


# ---------------------------------------------------------------- P8: monotone proximal-point distance
@pytest.mark.parametrize("tv,sig", [("iso", 0.25), ("aniso", 0.25), ("iso", 0.3441)])
def test_P8_proximal_point_distance_nonincreasing(oracle, tv, sig):
    """theta=1, sigma*tau*||K_full||^2 < 1: PDHG is a proximal-point method in the metric
    [[I/tau, -K^T], [-K, I/sigma]] on u_n = (chi_n, y_{n+1}); ||u_{n+1}-u_n||_M^2 never increases [7]."""
    data = synth.generate(0)
    phi = data["field"][0]
    N = 120
    tvm = oracle.TV_ISO if tv == "iso" else oracle.TV_ANISO
    tr = oracle.trace(phi, None, None, lambda_=0.01, sigma=sig, tau=sig, max_iters=N + 1, tv_mode=tvm)
    chi, p, qx, qy = tr[:, 0], tr[:, 1], tr[:, 2], tr[:, 3]
    d = []
    for n in range(1, N):      # u_n = (chi_n, y_{n+1})
        dchi = chi[n + 1] - chi[n]
        dp, dqx, dqy = p[n + 2] - p[n + 1], qx[n + 2] - qx[n + 1], qy[n + 2] - qy[n + 1]
        gx, gy = oracle.grad(dchi)
        Kd = np_K(dchi)
        cross = np.sum(Kd * dp) + np.sum(gx * dqx) + np.sum(gy * dqy)
        d.append(np.sum(dchi ** 2) / sig - 2 * cross + (np.sum(dp ** 2) + np.sum(dqx ** 2) + np.sum(dqy ** 2)) / sig)
    d = np.array(d)
    assert np.all(d > 0)
    assert np.all(d[1:] <= d[:-1] * (1 + 1e-9))


def test_P8_relgap_nonnegative_and_eventually_decreasing(oracle):
    data = synth.generate(0)
    out = oracle.solve(data["field"], data["mask"], lambda_=0.01, sigma=SIG, tau=SIG, max_iters=100)
    g = out["relgap"][0]
    assert np.all(g >= 0)
    assert abs(g[0] - 0.64) < 1e-12
    assert np.all(g[31:] <= g[30:-1] * (1 + 1e-6))
    assert g[99] < 1e-3 * g[0]
    r = out["relres"][0]
    assert r[0] == 1.0 and np.all(r[1:] < r[:-1])


# ---------------------------------------------------------------- P9: lambda convention
def test_P9_paper_convention_equals_rescaled_default(oracle):
    """A(lambda, sigma, tau) == B(alpha = 1/lambda, sigma/lambda, tau*lambda): identical chi sequence, p and q / lambda."""
    case = synth.random_case(16, 24, 1, seed=5, with_mask=True, with_weight=True)
    lam, sig, tau = 50.0, 0.25, 0.25
    for tvm in (oracle.TV_ISO, oracle.TV_ANISO):
        a = oracle.solve(case["field"], case["mask"], case["weight"], lambda_=lam, sigma=sig, tau=tau, max_iters=60,
                         lambda_conv=oracle.LAMBDA_DATA, tv_mode=tvm, want_state=True)
        b = oracle.solve(case["field"], case["mask"], case["weight"], lambda_=1 / lam, sigma=sig / lam, tau=tau * lam,
                         max_iters=60, lambda_conv=oracle.LAMBDA_REG, tv_mode=tvm, want_state=True)
        assert rel(a["chi"], b["chi"]) < 1e-12
        assert rel(a["p"] / lam, b["p"]) < 1e-12
        assert rel(a["qx"] / lam, b["qx"]) < 1e-12
        assert rel(a["relgap"], b["relgap"]) < 1e-10


# ---------------------------------------------------------------- P10: analytic field of a cylinder
@pytest.mark.parametrize("n,R", [(64, 3.0), (256, 16.0), (256, 5.0)])
def test_P10_forward_model_cylinder(oracle, n, R):
    """Infinite cylinder perpendicular to the slice, B0 in-plane along y: field/chi = -1/6 inside,
    (R^2 / 2 r^2) cos(2 theta) outside, theta measured from the B0 axis."""
    yy, xx = np.mgrid[0:n, 0:n]
    c = n / 2.0
    disc = ((xx - c) ** 2 + (yy - c) ** 2 <= R * R).astype(np.float64)
    f = oracle.apply_K(disc, oracle.B0_Y)
    f = f - f[0, 0] + 0.0  # far corner ~ 0 up to periodic images / removed DC
    inside = (xx - c) ** 2 + (yy - c) ** 2 <= (0.6 * R) ** 2
    assert abs(f[inside].mean() - (-1.0 / 6.0)) < 0.02 * (1.0 / 6.0) * 3  # pixelation: within a few percent
    r2 = (xx - c) ** 2 + (yy - c) ** 2
    ring = (r2 > (1.5 * R) ** 2) & (r2 < (4 * R) ** 2)
    cos2t = ((yy - c) ** 2 - (xx - c) ** 2) / np.maximum(r2, 1e-30)   # theta from the y (B0) axis
    ana = R * R / (2 * np.maximum(r2, 1e-30)) * cos2t
    assert np.corrcoef(f[ring], ana[ring])[0, 1] > 0.995
    assert rel(f[ring], ana[ring]) < 0.12
    # signs: positive along B0, negative across
    k = int(round(2 * R))
    assert f[int(c) + k, int(c)] > 0 and f[int(c), int(c) + k] < 0
    # B0 along x is the transposed picture
    fx = oracle.apply_K(disc, oracle.B0_X)
    assert rel(fx, oracle.apply_K(disc.T.copy(), oracle.B0_Y).T) < 1e-12


# ---------------------------------------------------------------- P11: sphere (3-D helper, off path)
def test_P11_forward_model_sphere_3d(oracle):
    """Sphere in the 3-D kernel 1/3 - kz^2/|k|^2: 0 inside (Lorentz sphere), (R^3/3r^3)(3cos^2 theta - 1) outside."""
    n, R = 32, 5.0
    zz, yy, xx = np.mgrid[0:n, 0:n, 0:n]
    c = n / 2.0
    r2 = (xx - c) ** 2 + (yy - c) ** 2 + (zz - c) ** 2
    f = oracle.forward3d((r2 <= R * R).astype(np.float64))
    f = f - f[0, 0, 0]
    assert abs(f[r2 <= (0.5 * R) ** 2].mean()) < 0.02
    shell = (r2 > (1.6 * R) ** 2) & (r2 < (2.6 * R) ** 2)
    ana = R ** 3 / (3 * np.maximum(r2, 1e-30) ** 1.5) * (3 * (zz - c) ** 2 / np.maximum(r2, 1e-30) - 1)
    assert np.corrcoef(f[shell], ana[shell])[0, 1] > 0.99
    assert rel(f[shell], ana[shell]) < 0.2


# ---------------------------------------------------------------- P12: round trip (sanity, loose)
def test_P12_round_trip_recovers_needle(oracle):
    data = synth.generate(0, want_truth=True)
    out = oracle.solve(data["field"], data["mask"], lambda_=0.01, sigma=SIG, tau=SIG, max_iters=100, want_hist=False)
    truth = data["chi_true"][0] - data["chi_true"][0].mean()
    chi = out["chi"][0]
    assert abs(chi.max() - 200.0) < 0.25 * 200.0
    assert np.unravel_index(chi.argmax(), chi.shape) == np.unravel_index(truth.argmax(), truth.shape) or \
        truth[np.unravel_index(chi.argmax(), chi.shape)] > 100
    assert np.corrcoef(chi.ravel(), truth.ravel())[0, 1] > 0.85


# ---------------------------------------------------------------- P14: dense-matrix brute force
@pytest.mark.parametrize("tv", ["iso", "aniso"])
def test_P14_dense_matrix_bruteforce_8x8(oracle, tv):
    """8x8 slice, 5 iterations: K_full = [W K; M G] built as dense matrices (K from DFT matrices, G by stencils),
    the iteration done with mat-vecs."""
    n = 8
    P = n * n
    case = synth.random_case(n, n, 1, seed=6, with_mask=True, with_weight=True)
    phi = case["field"][0].astype(np.float64).ravel()
    M = case["mask"][0].astype(np.float64).ravel()
    M[::7] = 0.0   # make the mask non-trivial on this tiny grid
    W = case["weight"][0].astype(np.float64).ravel()
    F1 = np.exp(-2j * np.pi * np.outer(np.arange(n), np.arange(n)) / n)
    F2 = np.kron(F1, F1)                                # row-major (y,x) flattening: FFT2 as one matrix
    Kmat = np.real(np.conj(F2).T @ np.diag(np_dipole(n, n).ravel()) @ F2) / P
    Gx = np.zeros((P, P))
    Gy = np.zeros((P, P))
    for y in range(n):
        for x in range(n):
            i = y * n + x
            if x < n - 1:
                Gx[i, i + 1], Gx[i, i] = 1, -1
            if y < n - 1:
                Gy[i, i + n], Gy[i, i] = 1, -1
    A = np.vstack([np.diag(W) @ Kmat, np.diag(M) @ Gx, np.diag(M) @ Gy])      # 192 x 64
    alpha, sig, tau, theta = 0.7, 0.25, 0.25, 1.0
    chi = np.zeros(P)
    chib = np.zeros(P)
    y_ = np.zeros(3 * P)
    for _ in range(5):
        t = y_ + sig * (A @ chib)
        pn = (t[:P] - sig * W * phi) / (1 + sig)
        tx, ty = t[P:2 * P], t[2 * P:]
        if tv == "iso":
            s = np.maximum(1.0, np.hypot(tx, ty) / alpha)
            qn = np.concatenate([tx / s, ty / s])
        else:
            qn = np.clip(np.concatenate([tx, ty]), -alpha, alpha)
        y_ = np.concatenate([pn, qn])
        chin = chi - tau * (A.T @ y_)
        chib = chin + theta * (chin - chi)
        chi = chin
    mask_in = M.reshape(1, n, n).astype(np.float32)
    out = oracle.solve(case["field"], mask_in, case["weight"], lambda_=alpha, sigma=sig, tau=tau, theta=theta,
                       max_iters=5, tv_mode=oracle.TV_ISO if tv == "iso" else oracle.TV_ANISO, want_state=True)
    assert rel(out["chi"][0].ravel(), chi) < 1e-12
    assert rel(out["p"][0].ravel(), y_[:P]) < 1e-12
    assert rel(np.concatenate([out["qx"][0].ravel(), out["qy"][0].ravel()]), y_[P:]) < 1e-12
    assert rel(out["chibar"][0].ravel(), chib) < 1e-12


def test_P14_relgap_is_fenchel_young_gap(oracle):
    """relgap_{n+1} = [F(K chibar_n) + F*(y_{n+1}) - <K chibar_n, y_{n+1}>]/P0 with F = 1/2||. - W phi||^2 + alpha||.||_{2,1}
    (reading R9): recompute it from the traced iterates with numpy operators."""
    case = synth.random_case(16, 16, 1, seed=7, with_mask=True, with_weight=True)
    phi = case["field"][0].astype(np.float64)
    M = case["mask"][0].astype(np.float64)
    W = case["weight"][0].astype(np.float64)
    alpha, N = 0.4, 12
    tr = oracle.trace(phi, M, W, lambda_=alpha, sigma=SIG, tau=SIG, max_iters=N)
    out = oracle.solve(phi, M, W, lambda_=alpha, sigma=SIG, tau=SIG, max_iters=N)
    P0 = 0.5 * np.sum((W * phi) ** 2)
    for n in range(N):
        chib = 2 * tr[n, 0] - (tr[n - 1, 0] if n > 0 else 0)
        y1 = W * np_K(chib)
        gx = np.zeros_like(chib)
        gy = np.zeros_like(chib)
        gx[:, :-1] = chib[:, 1:] - chib[:, :-1]
        gy[:-1, :] = chib[1:, :] - chib[:-1, :]
        gx, gy = M * gx, M * gy
        p, qx, qy = tr[n + 1, 1], tr[n + 1, 2], tr[n + 1, 3]
        F = 0.5 * np.sum((y1 - W * phi) ** 2) + alpha * np.sum(np.hypot(gx, gy))
        Fstar = 0.5 * np.sum(p ** 2) + np.sum(p * W * phi)          # + indicator(|q| <= alpha) = 0
        assert np.hypot(qx, qy).max() <= alpha * (1 + 1e-12)
        gap = F + Fstar - np.sum(y1 * p) - np.sum(gx * qx) - np.sum(gy * qy)
        assert abs(gap / P0 - out["relgap"][0, n]) < 1e-12 * max(1.0, gap / P0)
        chi_new, chi_old = tr[n + 1, 0], tr[n, 0]
        assert abs(np.linalg.norm(chi_new - chi_old) / np.linalg.norm(chi_new) - out["relres"][0, n]) < 1e-12


# ---------------------------------------------------------------- stopping rule, corner cases, precision
def test_tolerance_stop_is_first_crossing(oracle):
    data = synth.generate(0)
    full = oracle.solve(data["field"], data["mask"], lambda_=0.01, sigma=SIG, tau=SIG, max_iters=150)
    g = full["relgap"][0]
    tol = 1e-4
    first = int(np.argmax(g < tol)) + 1
    assert 40 < first < 120
    st = oracle.solve(data["field"], data["mask"], lambda_=0.01, sigma=SIG, tau=SIG, max_iters=150, tol=tol)
    assert st["iters_done"][0] == first
    assert np.all(st["relgap"][0, first:] == -1)
    ref = oracle.solve(data["field"], data["mask"], lambda_=0.01, sigma=SIG, tau=SIG, max_iters=first, want_hist=False)
    assert np.array_equal(st["chi"], ref["chi"])
    st8 = oracle.solve(data["field"], data["mask"], lambda_=0.01, sigma=SIG, tau=SIG, max_iters=150, tol=tol,
                       check_every=8)
    assert st8["iters_done"][0] == -(-first // 8) * 8
    capped = oracle.solve(data["field"], data["mask"], lambda_=0.01, sigma=SIG, tau=SIG, max_iters=20, tol=tol)
    assert capped["iters_done"][0] == 20


def test_zero_field_slice(oracle):
    f = np.zeros((2, 8, 8), np.float32)
    f[1] = synth.random_case(8, 8, 1, seed=8)["field"][0]
    a = oracle.solve(f, lambda_=0.1, sigma=SIG, tau=SIG, max_iters=7, tol=1e-3)
    assert a["iters_done"][0] == 0 and np.all(a["chi"][0] == 0)
    b = oracle.solve(f, lambda_=0.1, sigma=SIG, tau=SIG, max_iters=7)
    assert b["iters_done"][0] == 7 and np.all(b["chi"][0] == 0) and np.all(b["relgap"][0] == 0)
    assert b["iters_done"][1] == 7 and np.abs(b["chi"][1]).max() > 0


def test_slices_are_independent_and_batch_order(oracle):
    case = synth.random_case(16, 8, 3, seed=9)
    allb = oracle.solve(case["field"], case["mask"], lambda_=0.3, sigma=SIG, tau=SIG, max_iters=9)
    for b in range(3):
        one = oracle.solve(case["field"][b], case["mask"][b], lambda_=0.3, sigma=SIG, tau=SIG, max_iters=9)
        assert np.array_equal(one["chi"][0], allb["chi"][b])


def test_float_instantiation_tracks_double(oracle):
    data = synth.generate(0)
    d = oracle.solve(data["field"], data["mask"], lambda_=0.01, sigma=SIG, tau=SIG, max_iters=100, want_hist=False)
    f = oracle.solve(data["field"], data["mask"], lambda_=0.01, sigma=SIG, tau=SIG, max_iters=100, want_hist=False,
                     precision="f32")
    assert rel(f["chi"], d["chi"]) < 1e-5
    assert rel(d["chi32"], d["chi"]) < 1e-7


def test_theta_zero_and_b0x_variants_run(oracle):
    """theta = 0 (Arrow-Hurwicz) and B0 along x: chibar = chi ; solving the transposed problem transposes chi."""
    case = synth.random_case(16, 16, 1, seed=10, with_mask=False)
    a = oracle.solve(case["field"], lambda_=0.2, sigma=0.2, tau=0.2, theta=0.0, max_iters=6, want_state=True)
    assert np.array_equal(a["chibar"], a["chi"])
    fx = np.ascontiguousarray(case["field"][0].T)[None]
    x = oracle.solve(fx, lambda_=0.2, sigma=SIG, tau=SIG, max_iters=6, b0_dir=oracle.B0_X)
    y = oracle.solve(case["field"], lambda_=0.2, sigma=SIG, tau=SIG, max_iters=6, b0_dir=oracle.B0_Y)
    assert rel(x["chi"][0].T, y["chi"][0]) < 1e-12


# ---------------------------------------------------------------- P15: oblique in-plane B0
def np_dipole_angle(nx, ny, ang):
    """Closed form typed independently: k_b = k . (cos a, sin a), standard fftfreq."""
    kx = np.fft.fftfreq(nx)[None, :]
    ky = np.fft.fftfreq(ny)[:, None]
    k2 = kx * kx + ky * ky
    kb = kx * np.cos(ang) + ky * np.sin(ang)
    out = np.zeros((ny, nx))
    nz = k2 > 0
    out[nz] = 1.0 / 3.0 - (kb * kb + 0 * k2)[nz] / k2[nz]
    return out


@pytest.mark.parametrize("ny,nx", [(16, 16), (8, 32), (12, 10)])
def test_P15_dipole_angle_reduces_to_axes_and_closed_form(oracle, ny, nx):
    assert rel(oracle.dipole_angle(nx, ny, 0.0), oracle.dipole(nx, ny, oracle.B0_X)) < 1e-15
    assert rel(oracle.dipole_angle(nx, ny, np.pi / 2), oracle.dipole(nx, ny, oracle.B0_Y)) < 1e-15
    for ang in (0.3, np.pi / 4, 2.0, -0.7):
        D = oracle.dipole_angle(nx, ny, ang)
        assert rel(D, np_dipole_angle(nx, ny, ang)) < 1e-13
        assert D[0, 0] == 0.0 and D.min() >= -2.0 / 3.0 - 1e-12 and D.max() <= 1.0 / 3.0 + 1e-12
        # B0 and -B0 are the same axis
        assert rel(oracle.dipole_angle(nx, ny, ang + np.pi), D) < 1e-12
    # 45 degrees on a square grid: -2/3 on the diagonal kx = ky, +1/3 on the anti-diagonal, transpose-symmetric
    if nx == ny:
        D = oracle.dipole_angle(nx, ny, np.pi / 4)
        for i in range(1, nx // 2):
            assert abs(D[i, i] + 2.0 / 3.0) < 1e-12 and abs(D[nx - i, i] - 1.0 / 3.0) < 1e-12
        assert rel(D, D.T) < 1e-12
    # the sum over two perpendicular in-plane directions is 2/3 - 1 = -1/3 away from DC
    S = oracle.dipole_angle(nx, ny, 0.4) + oracle.dipole_angle(nx, ny, 0.4 + np.pi / 2)
    S[0, 0] = -1.0 / 3.0
    assert np.abs(S + 1.0 / 3.0).max() < 1e-12


def test_P15_forward_model_cylinder_rotated(oracle):
    """The analytic field of a cylinder, (R^2/2r^2) cos 2(theta - a) outside and -1/6 inside, turns with B0; and
    K(a) stays real and symmetric (the oracle takes the real part: only the even part of D acts)."""
    n, R, ang = 256, 16.0, 0.6
    yy, xx = np.mgrid[0:n, 0:n]
    c = n / 2.0
    disc = ((xx - c) ** 2 + (yy - c) ** 2 <= R * R).astype(np.float64)
    f = oracle.apply_K_angle(disc, ang)
    f = f - f[0, 0]
    r2 = (xx - c) ** 2 + (yy - c) ** 2
    inside = r2 <= (0.6 * R) ** 2
    assert abs(f[inside].mean() + 1.0 / 6.0) < 0.02
    ring = (r2 > (1.5 * R) ** 2) & (r2 < (4 * R) ** 2)
    th = np.arctan2(yy - c, xx - c)
    ana = R * R / (2 * np.maximum(r2, 1e-30)) * np.cos(2 * (th - ang))
    assert np.corrcoef(f[ring], ana[ring])[0, 1] > 0.995
    assert rel(f[ring], ana[ring]) < 0.12
    # independent numpy evaluation of Re(IFFT(D FFT(a)))
    a = rng(31).standard_normal((24, 40))
    ref = np.real(np.fft.ifft2(np_dipole_angle(40, 24, ang) * np.fft.fft2(a)))
    assert rel(oracle.apply_K_angle(a, ang), ref) < 1e-12
    b = rng(32).standard_normal((24, 40))
    assert abs(np.vdot(oracle.apply_K_angle(a, ang), b) - np.vdot(a, oracle.apply_K_angle(b, ang))) < 1e-10


def test_P15_angle_iteration_matches_axis_iteration(oracle):
    case = synth.random_case(32, 16, 2, seed=15, with_mask=True, with_weight=True)
    kw = dict(lambda_=0.3, sigma=SIG, tau=SIG, max_iters=7)
    a = oracle.solve(case["field"], case["mask"], case["weight"], b0_dir=oracle.B0_X, **kw)
    b = oracle.solve(case["field"], case["mask"], case["weight"], b0_angle=0.0, **kw)
    assert rel(b["chi"], a["chi"]) < 1e-14
    c = oracle.solve(case["field"], case["mask"], case["weight"], b0_angle=np.pi / 2, **kw)
    d = oracle.solve(case["field"], case["mask"], case["weight"], b0_dir=oracle.B0_Y, **kw)
    assert rel(c["chi"], d["chi"]) < 1e-12


# ---------------------------------------------------------------- P16: l1 on chi with a shrinkage prox (north_star's alternative)
def test_P16_shrink_is_the_prox_of_the_l1_norm(oracle):
    r = rng(16)
    v = np.concatenate([r.standard_normal(200) * 2, [0.0, 1.0, -1.0, 0.5, -0.5]])
    t = np.abs(r.standard_normal(v.size)) + 0.0
    t[-5:] = [1.0, 1.0, 1.0, 1.0, 1.0]
    x = oracle.shrink(v, t)
    # first-order optimality of argmin_x 1/2 (x - v)^2 + t |x| : v - x = t sign(x) where x != 0, |v - x| <= t where x = 0
    nz = x != 0
    assert np.allclose((v - x)[nz], (t * np.sign(x))[nz], atol=1e-15)
    assert np.all(np.abs(v - x)[~nz] <= t[~nz] + 1e-15)
    assert np.all(np.sign(x[nz]) == np.sign(v[nz]))
    assert np.array_equal(x[-5:], [0.0, 0.0, 0.0, 0.0, 0.0])
    # brute force: the minimiser on a fine grid
    for vi, ti in ((1.7, 0.4), (-0.9, 0.25), (0.1, 0.3)):
        g = np.linspace(-3, 3, 600001)
        xb = g[np.argmin(0.5 * (g - vi) ** 2 + ti * np.abs(g))]
        assert abs(oracle.shrink(np.array([vi]), ti)[0] - xb) < 2e-5
    # threshold 0 is the identity
    assert np.array_equal(oracle.shrink(v, 0.0), v)


@pytest.mark.parametrize("with_w", [False, True])
def test_P16_l1_first_iterate_closed_form(oracle, with_w):
    """chi_1 = shrink((sigma tau/(1+sigma)) K(W^2 phi), tau alpha M), p_1 = -sigma W phi/(1+sigma), relgap_1 = 1/(1+sigma)^2."""
    case = synth.random_case(32, 16, 1, seed=160, with_mask=True, with_weight=with_w)
    phi = case["field"][0].astype(np.float64)
    W = case["weight"][0].astype(np.float64) if with_w else np.ones_like(phi)
    M = case["mask"][0].astype(np.float64)
    alpha, tau = 0.02, 0.3
    out = oracle.solve(case["field"], case["mask"], case["weight"] if with_w else None, lambda_=alpha, sigma=SIG, tau=tau,
                       max_iters=1, regulariser=oracle.REG_L1, want_state=True)
    v = SIG * tau / (1 + SIG) * np_K(W * W * phi)
    chi1 = np.sign(v) * np.maximum(np.abs(v) - tau * alpha * M, 0.0)
    assert rel(out["chi"][0], chi1) < 1e-12
    assert rel(out["p"][0], -SIG * W * phi / (1 + SIG)) < 1e-12
    assert abs(out["relgap"][0, 0] - 1.0 / (1 + SIG) ** 2) < 1e-12
    assert np.all(out["qx"] == 0) and np.all(out["qy"] == 0)
    assert (out["chi"][0] == 0).sum() > 0 and (out["chi"][0] != 0).sum() > 0     # the threshold bites on part of the image


def test_P16_l1_dense_matrix_bruteforce_8x8(oracle):
    """8x8, 6 iterations, K as a dense matrix from DFT matrices, the iteration written with mat-vecs."""
    n = 8
    P = n * n
    case = synth.random_case(n, n, 1, seed=161, with_mask=True, with_weight=True)
    phi = case["field"][0].astype(np.float64).ravel()
    M = case["mask"][0].astype(np.float64).ravel()
    M[::5] = 0.0
    W = case["weight"][0].astype(np.float64).ravel()
    F1 = np.exp(-2j * np.pi * np.outer(np.arange(n), np.arange(n)) / n)
    F2 = np.kron(F1, F1)
    Kmat = np.real(np.conj(F2).T @ np.diag(np_dipole(n, n).ravel()) @ F2) / P
    A = np.diag(W) @ Kmat
    alpha, sig, tau, theta = 0.05, 0.4, 0.5, 0.8
    chi, chib, p = np.zeros(P), np.zeros(P), np.zeros(P)
    for _ in range(6):
        p = (p + sig * (A @ chib - W * phi)) / (1 + sig)
        v = chi - tau * (A.T @ p)
        chin = np.sign(v) * np.maximum(np.abs(v) - tau * alpha * M, 0.0)
        chib = chin + theta * (chin - chi)
        chi = chin
    out = oracle.solve(case["field"], M.reshape(1, n, n).astype(np.float32), case["weight"], lambda_=alpha, sigma=sig, tau=tau,
                       theta=theta, max_iters=6, regulariser=oracle.REG_L1, want_state=True)
    assert rel(out["chi"][0].ravel(), chi) < 1e-12
    assert rel(out["p"][0].ravel(), p) < 1e-12
    assert rel(out["chibar"][0].ravel(), chib) < 1e-12


def test_P16_l1_fixed_point_is_the_lasso_optimum(oracle):
    """After many iterations chi satisfies the optimality condition of min 1/2||K chi - phi||^2 + alpha||chi||_1:
    g = K(K chi - phi) has |g| <= alpha everywhere and g = -alpha sign(chi) on the support."""
    n = 16
    case = synth.random_case(n, n, 1, seed=162, with_mask=False)
    phi = case["field"][0].astype(np.float64)
    alpha = 0.05 * np.abs(np_K(phi)).max()
    out = oracle.solve(case["field"], None, lambda_=alpha, sigma=1.0, tau=1.0, max_iters=6000, regulariser=oracle.REG_L1,
                       want_hist=False)
    chi = out["chi"][0]
    g = np_K(np_K(chi) - phi)
    assert np.abs(g).max() <= alpha * (1 + 1e-6)
    sup = np.abs(chi) > 1e-9 * np.abs(chi).max()
    assert sup.sum() > 0 and (~sup).sum() > 0
    assert np.abs(g[sup] + alpha * np.sign(chi[sup])).max() < 1e-6 * alpha


def test_P16_l1_with_alpha_zero_equals_tv_with_alpha_zero(oracle):
    case = synth.random_case(16, 16, 2, seed=163, with_mask=True, with_weight=True)
    kw = dict(lambda_=0.0, sigma=SIG, tau=SIG, max_iters=9)
    a = oracle.solve(case["field"], case["mask"], case["weight"], **kw)
    b = oracle.solve(case["field"], case["mask"], case["weight"], regulariser=oracle.REG_L1, **kw)
    assert rel(b["chi"], a["chi"]) < 1e-14
    assert np.allclose(b["relgap"], a["relgap"], rtol=1e-12)
