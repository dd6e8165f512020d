"""Pins of oracle/pd3_oracle.py (NEXT-2, the true 3-D variant; reading R23) against things other than itself.  No GPU."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, os.path.join(ROOT, "oracle"))
import pd3_oracle as o3  # noqa: E402


def rel(a, b):
    return np.linalg.norm(np.asarray(a) - np.asarray(b)) / max(np.linalg.norm(b), 1e-300)


def test_P20_forward_model_against_the_independent_dft(oracle):
    """apply_K3 (numpy.fft) == pdo_forward3d (the C++ oracle's own O(n^2) line DFT, pinned to the analytic sphere by P11)."""
    rng = np.random.default_rng(20)
    for n in (4, 8, 12):
        a = rng.normal(size=(n, n, n))
        assert rel(o3.apply_K3(a, o3.B0_Z), oracle.forward3d(a)) < 1e-12
    # axis values of the kernel: 1/3 across B0, -2/3 along it; the three directions sum to 0 off the origin (1 - 1)
    D = o3.dipole3(8, 4, 16, o3.B0_Z)
    assert D.shape == (16, 4, 8) and D[0, 0, 0] == 0.0
    assert D[0, 0, 3] == pytest.approx(1 / 3) and D[0, 2, 0] == pytest.approx(1 / 3) and D[5, 0, 0] == pytest.approx(-2 / 3)
    tot = o3.dipole3(8, 4, 16, 0) + o3.dipole3(8, 4, 16, 1) + o3.dipole3(8, 4, 16, 2)
    tot[0, 0, 0] = 0.0
    assert np.abs(tot).max() < 1e-15
    assert D[3, 1, 2] == pytest.approx(1 / 3 - (3 / 16) ** 2 / ((2 / 8) ** 2 + (1 / 4) ** 2 + (3 / 16) ** 2))


@pytest.mark.parametrize("b0", [0, 1])
def test_P21_one_slice_volume_is_the_2d_problem(oracle, b0):
    """nz = 1: kz = 0 and the z-difference vanishes, so the 3-D iteration IS the 2-D one (C++ oracle, pinned by P1-P16)."""
    rng = np.random.default_rng(21 + b0)
    f = rng.normal(size=(12, 16))
    m = (rng.uniform(size=f.shape) > 0.3).astype(np.float64)
    w = rng.uniform(0.2, 1.0, size=f.shape).astype(np.float32)
    got = o3.solve3(f.astype(np.float32)[None], m[None], w[None], lambda_=0.3, sigma=0.25, tau=0.25, max_iters=6, b0_dir=b0)
    ref = oracle.solve(f.astype(np.float32), m.astype(np.float32), w, lambda_=0.3, sigma=0.25, tau=0.25, max_iters=6, b0_dir=b0)["chi"][0]
    assert rel(got[0], ref) < 1e-12                                       # with a data weighting W as well
    for iters, theta in [(1, 1.0), (7, 1.0), (5, 0.5)]:
        got = o3.solve3(f[None], m[None], lambda_=0.3, sigma=0.25, tau=0.25, theta=theta, max_iters=iters, b0_dir=b0)
        ref = oracle.solve(f.astype(np.float32), m.astype(np.float32), lambda_=0.3, sigma=0.25, tau=0.25, theta=theta,
                           max_iters=iters, b0_dir=b0)["chi"][0]
        want = o3.solve3(f.astype(np.float32)[None], m[None], lambda_=0.3, sigma=0.25, tau=0.25, theta=theta, max_iters=iters, b0_dir=b0)
        assert rel(want[0], ref) < 1e-12 and rel(got[0], ref) < 1e-6     # (the 2-D oracle takes float32 inputs)


def test_P22_gradient_hand_values_and_adjoint():
    a = np.arange(8, dtype=np.float64).reshape(2, 2, 2) ** 2           # a[z][y][x] = (4z + 2y + x)^2
    gx, gy, gz = o3.grad3(a)
    assert gx[:, :, 0].tolist() == [[1.0, 5.0], [9.0, 13.0]] and not gx[:, :, 1].any()
    assert gy[:, 0, :].tolist() == [[4.0, 8.0], [20.0, 24.0]] and not gy[:, 1, :].any()
    assert gz[0].tolist() == [[16.0, 24.0], [32.0, 40.0]] and not gz[1].any()
    rng = np.random.default_rng(22)
    a = rng.normal(size=(5, 6, 7))
    q = rng.normal(size=(3, 5, 6, 7))
    lhs = sum((g * qq).sum() for g, qq in zip(o3.grad3(a), q))
    assert lhs == pytest.approx((a * o3.grad3T(*q)).sum(), rel=1e-12)
    # ||G||^2 <= 12: the Rayleigh quotient of the checkerboard approaches it from below
    cb = (-1.0) ** np.add.outer(np.add.outer(np.arange(16), np.arange(16)), np.arange(16))
    ray = sum((g * g).sum() for g in o3.grad3(cb)) / (cb * cb).sum()
    assert 10.0 < ray < 12.0


def dense_ops(nx, ny, nz, b0):
    n = nx * ny * nz
    def dft(m):
        k = np.arange(m)
        return np.exp(-2j * np.pi * np.outer(k, k) / m)
    F = np.kron(dft(nz), np.kron(dft(ny), dft(nx)))
    fz, fy, fx = [np.where(np.arange(m) < (m + 1) // 2, np.arange(m), np.arange(m) - m) / m for m in (nz, ny, nx)]
    K2 = fz[:, None, None] ** 2 + fy[None, :, None] ** 2 + fx[None, None, :] ** 2
    kb = [fx[None, None, :], fy[None, :, None], fz[:, None, None]][b0] * np.ones((nz, ny, nx))
    D = np.where(K2 == 0, 0.0, 1 / 3 - kb ** 2 / np.where(K2 == 0, 1, K2)).ravel()
    K = np.real(np.conj(F).T @ (D[:, None] * F)) / n
    idx = np.arange(n).reshape(nz, ny, nx)
    G = np.zeros((3, n, n))
    for z in range(nz):
        for y in range(ny):
            for x in range(nx):
                i = idx[z, y, x]
                if x + 1 < nx: G[0, i, idx[z, y, x + 1]] += 1; G[0, i, i] -= 1
                if y + 1 < ny: G[1, i, idx[z, y + 1, x]] += 1; G[1, i, i] -= 1
                if z + 1 < nz: G[2, i, idx[z + 1, y, x]] += 1; G[2, i, i] -= 1
    return K, G


@pytest.mark.parametrize("b0,theta,weighted", [(2, 1.0, False), (0, 0.7, False), (1, 0.9, True)])
def test_P23_dense_matrix_bruteforce_4x4x4(b0, theta, weighted):
    """K from Kronecker DFT matrices, G from stencils, the iteration with mat-vecs (non-cubic 4x3x5 volume, mask)."""
    nx, ny, nz = 4, 3, 5
    K, G = dense_ops(nx, ny, nz, b0)
    rng = np.random.default_rng(23)
    f = rng.normal(size=(nz, ny, nx))
    m = (rng.uniform(size=f.shape) > 0.25).astype(np.float64)
    w = rng.uniform(0.2, 1.0, size=f.shape) if weighted else np.ones_like(f)
    lam, sig, tau = 0.2, 0.25, 0.25
    chi = np.zeros(f.size); bar = chi.copy(); p = chi.copy(); q = np.zeros((3, f.size))
    Kw = w.ravel()[:, None] * K                                          # K_full's data block is W K; its transpose K^T W
    for _ in range(6):
        p = (p + sig * (Kw @ bar - w.ravel() * f.ravel())) / (1 + sig)
        t = q + sig * m.ravel() * (G @ bar)
        nrm = np.sqrt((t * t).sum(0))
        q = t * np.where(nrm > lam, lam / np.maximum(nrm, 1e-300), 1.0)
        new = chi - tau * (Kw.T @ p) - tau * sum(G[c].T @ (m.ravel() * q[c]) for c in range(3))
        bar = new + theta * (new - chi)
        chi = new
    got = o3.solve3(f, m, w if weighted else None, lambda_=lam, sigma=sig, tau=tau, theta=theta, max_iters=6, b0_dir=b0)
    assert rel(got.ravel(), chi) < 1e-12


def test_P24_closed_form_first_iterate():
    """From zero: p1 = -sigma phi/(1+sigma), q1 = 0, chi1 = tau sigma/(1+sigma) K phi (K symmetric)."""
    rng = np.random.default_rng(24)
    f = rng.normal(size=(8, 4, 16))
    got = o3.solve3(f, None, lambda_=0.1, sigma=0.3, tau=0.2, max_iters=1, b0_dir=1)
    assert rel(got, 0.2 * 0.3 / 1.3 * o3.apply_K3(f, 1)) < 1e-13
    assert abs(got.mean()) < 1e-15                                     # D3(0) = 0: zero mean


def test_P25_axis_permutation_symmetry():
    """Transposing the volume and moving B0 with it transposes the solution (no axis is special in the code)."""
    rng = np.random.default_rng(25)
    f = rng.normal(size=(4, 6, 8))
    m = (rng.uniform(size=f.shape) > 0.3).astype(np.float64)
    a = o3.solve3(f, m, lambda_=0.2, sigma=0.25, tau=0.25, max_iters=4, b0_dir=o3.B0_Z)
    b = o3.solve3(f.transpose(2, 1, 0).copy(), m.transpose(2, 1, 0).copy(), lambda_=0.2, sigma=0.25, tau=0.25, max_iters=4, b0_dir=o3.B0_X)
    assert rel(b.transpose(2, 1, 0), a) < 1e-12
    c = o3.solve3(f.transpose(1, 0, 2).copy(), m.transpose(1, 0, 2).copy(), lambda_=0.2, sigma=0.25, tau=0.25, max_iters=4, b0_dir=o3.B0_Y)
    assert rel(c.transpose(1, 0, 2), a) < 1e-12
    # a stack of volumes is solved volume by volume
    st = o3.solve3(np.stack([f, 2 * f]), np.stack([m, m]), lambda_=0.2, sigma=0.25, tau=0.25, max_iters=4)
    assert rel(st[0], a) < 1e-15 and st.shape == (2, 4, 6, 8)
