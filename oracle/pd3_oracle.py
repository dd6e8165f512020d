"""CPU oracle of the true 3-D variant: Eq.(1) as the paper literally states it, "G is the gradient
operator in all three dimensions", with the 3-D dipole kernel, on a whole volume at once.

TEST INFRASTRUCTURE ONLY: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  Plain numpy, float64, the Repeat body of PAPER.md:49 line by line in the paper's order, every
operator a whole-volume statement; numpy.fft.fftn is the library primitive behind F.  Pinned by
tests/test_oracle3d_pins.py (P20-P25): the independent C++ O(n^2)-per-line DFT forward model of pd_oracle.cpp, the exact
reduction to the 2-D oracle for nz = 1, hand values and adjointness of the gradient, a dense-matrix restatement on
4x4x4, the closed-form first iterate, axis-permutation symmetry.

Readings (R23): volume [nz][ny][nx], isotropic voxels ("isotropy"): k = (fi/nx, fj/ny, fk/nz)
with signed fftfreq indices; D3 = 1/3 - k_b^2/|k|^2, D3(0) = 0, B0 along x, y or z; G: forward differences with Neumann
boundary on all three axes, G^T its exact adjoint; the q-projection is the pointwise Euclidean norm over the three
components; lambda on the regulariser (R2), r = W (K chi_bar - phi) (R3; W optional), zero start, chi_N returned (R11).
"""
import numpy as np

B0_X, B0_Y, B0_Z = 0, 1, 2


def dipole3(nx, ny, nz, b0_dir=B0_Z):
    kz, ky, kx = np.meshgrid(np.fft.fftfreq(nz), np.fft.fftfreq(ny), np.fft.fftfreq(nx), indexing="ij")
    k2 = kx * kx + ky * ky + kz * kz
    kb = (kx, ky, kz)[b0_dir]
    D = 1.0 / 3.0 - kb * kb / np.where(k2 == 0, 1.0, k2)
    D[0, 0, 0] = 0.0
    return D


def apply_K3(a, b0_dir=B0_Z):
    a = np.asarray(a, np.float64)
    nz, ny, nx = a.shape
    return np.real(np.fft.ifftn(dipole3(nx, ny, nz, b0_dir) * np.fft.fftn(a)))


def grad3(a):
    """Forward differences, Neumann: the last difference along every axis is 0.  Returns (gx, gy, gz)."""
    gx, gy, gz = np.zeros_like(a), np.zeros_like(a), np.zeros_like(a)
    gx[:, :, :-1] = a[:, :, 1:] - a[:, :, :-1]
    gy[:, :-1, :] = a[:, 1:, :] - a[:, :-1, :]
    gz[:-1, :, :] = a[1:, :, :] - a[:-1, :, :]
    return gx, gy, gz


def grad3T(qx, qy, qz):
    """Exact adjoint of grad3."""
    out = np.zeros_like(qx)
    out[:, :, :-1] -= qx[:, :, :-1]
    out[:, :, 1:] += qx[:, :, :-1]
    out[:, :-1, :] -= qy[:, :-1, :]
    out[:, 1:, :] += qy[:, :-1, :]
    out[:-1, :, :] -= qz[:-1, :, :]
    out[1:, :, :] += qz[:-1, :, :]
    return out


def solve3(field, mask=None, weight=None, *, lambda_, sigma, tau, theta=1.0, max_iters=10, b0_dir=B0_Z):
    """PAPER.md:45-49 on one volume [nz][ny][nx] (or a stack of independent volumes [nvol][nz][ny][nx]).  Returns chi_N.
    weight: the data weighting W of Eq.(1) (None = identity): r = W (K chi_bar - phi) (R3), chi-update with K (W p)."""
    field = np.asarray(field, np.float64)
    if field.ndim == 4:
        return np.stack([solve3(field[v], None if mask is None else np.asarray(mask)[v],
                                None if weight is None else np.asarray(weight)[v], lambda_=lambda_, sigma=sigma, tau=tau,
                                theta=theta, max_iters=max_iters, b0_dir=b0_dir) for v in range(field.shape[0])])
    M = np.ones_like(field) if mask is None else np.asarray(mask, np.float64)
    W = np.ones_like(field) if weight is None else np.asarray(weight, np.float64)
    chi = np.zeros_like(field)
    chibar = np.zeros_like(field)
    p = np.zeros_like(field)
    qx, qy, qz = np.zeros_like(field), np.zeros_like(field), np.zeros_like(field)
    for _ in range(max_iters):
        p = (p + sigma * W * (apply_K3(chibar, b0_dir) - field)) / (1.0 + sigma)        # PAPER.md:49 line 1
        gx, gy, gz = grad3(chibar)
        tx, ty, tz = qx + sigma * M * gx, qy + sigma * M * gy, qz + sigma * M * gz      # PAPER.md:49 line 2
        nrm = np.sqrt(tx * tx + ty * ty + tz * tz)
        scale = np.where(nrm > lambda_, lambda_ / np.where(nrm > lambda_, nrm, 1.0), 1.0)   # onto the lambda-ball (R13)
        qx, qy, qz = tx * scale, ty * scale, tz * scale
        new = chi - tau * apply_K3(W * p, b0_dir) - tau * grad3T(M * qx, M * qy, M * qz)   # PAPER.md:49 line 3
        chibar = new + theta * (new - chi)                                              # PAPER.md:49 line 4
        chi = new
    return chi
