"""GPU-vs-oracle parity of the true 3-D variant (NEXT-2) through the C ABI: pd_plan3d / pd_solve3d against
oracle/pd3_oracle.py (numpy float64, the paper's iteration literally).  Gates as for the 2-D path (north_star): per-volume
relative L2 of chi <= 1e-5 after one iteration, <= 1e-3 after the full count."""
import os
import sys

import numpy as np
import pytest

from paper_2006_09808_b200 import synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def pd(torch):
    from paper_2006_09808_b200 import binding
    binding.lib()   # fails loudly if the extension is missing: there is no fallback
    return binding


@pytest.fixture(scope="module")
def o3():
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import pd3_oracle
    return pd3_oracle


def vol_rel(a, b):
    a = a.reshape(a.shape[0], -1).astype(np.float64)
    b = b.reshape(b.shape[0], -1).astype(np.float64)
    return np.linalg.norm(a - b, axis=1) / np.maximum(np.linalg.norm(b, axis=1), 1e-300)


def gpu_solve3(torch, pd, field, mask, iters, *, lam, b0, sigma=0.25, tau=0.25, theta=1.0, weight=None):
    nvol, nz, ny, nx = field.shape
    plan = pd.Plan3D(nx, ny, nz, nvol, b0, lam, sigma, tau, theta)
    if weight is not None:
        plan.set_weight(torch.from_numpy(weight).cuda())
    f = torch.from_numpy(field).cuda()
    m = None if mask is None else torch.from_numpy(mask).cuda()
    out = torch.full_like(f, float("nan"))
    plan.solve(f, m, out, iters)
    torch.cuda.synchronize()
    n = plan.last_launch_count
    plan.destroy()
    return out.cpu().numpy(), n


@pytest.mark.parametrize("nx,ny,nz,b0", [(16, 8, 8, 2), (64, 32, 16, 0), (32, 128, 64, 1), (256, 16, 8, 2), (128, 256, 32, 2)])
def test_one_iteration_all_axes(torch, pd, o3, nx, ny, nz, b0):
    rng = np.random.default_rng(nx + ny + nz)
    f = rng.normal(size=(2, nz, ny, nx)).astype(np.float32)          # unstructured: every frequency is exercised
    m = (rng.uniform(size=f.shape) > 0.3).astype(np.float32)
    g, launches = gpu_solve3(torch, pd, f, m, 1, lam=0.05, b0=b0)
    o = o3.solve3(f, m, lambda_=0.05, sigma=0.25, tau=0.25, max_iters=1, b0_dir=b0)
    assert vol_rel(g, o).max() < 1e-5
    # normalisation, phi^, one iteration, un-normalisation; nx >= 64: the chi-update rides the x passes (one launch less)
    assert launches == 2 + 3 + (6 if nx >= 64 else 7) + 1


@pytest.mark.parametrize("iters,theta,masked", [(2, 1.0, True), (3, 0.5, True), (25, 1.0, True), (25, 1.0, False)])
def test_iterations_exercise_q_and_divergence(torch, pd, o3, iters, theta, masked):
    case = synth.volume_case(64, 32, 16, nvol=3, seed=iters, b0_axis=2)
    lam = 0.02 * float(np.abs(case["field"]).max())                  # the ball is active on part of the volume
    m = case["mask"] if masked else None
    g, _ = gpu_solve3(torch, pd, case["field"], m, iters, lam=lam, b0=2, theta=theta)
    o = o3.solve3(case["field"], m, lambda_=lam, sigma=0.25, tau=0.25, theta=theta, max_iters=iters, b0_dir=2)
    assert vol_rel(g, o).max() < (1e-5 if iters <= 3 else 1e-3)
    assert vol_rel(g, o).max() < 2e-5                                  # what fp32 actually achieves
    assert np.abs(g.reshape(3, -1).mean(1)).max() < 1e-5 * np.abs(g).max()   # D3(0) = 0 and sum(G^T v) = 0: zero mean


@pytest.mark.parametrize("nx,ny,nz,b0,iters", [(16, 8, 8, 2, 1), (64, 32, 16, 0, 1), (128, 64, 64, 1, 1), (64, 32, 16, 2, 12)])
def test_data_weighting(torch, pd, o3, nx, ny, nz, b0, iters):
    """W set: the literal iteration (p in the image domain, K applied twice), three volumes (the last rides alone)."""
    case = synth.volume_case(nx, ny, nz, nvol=3, seed=nx + iters, b0_axis=b0)
    rng = np.random.default_rng(nx * nz)
    w = rng.uniform(0.2, 1.0, size=case["field"].shape).astype(np.float32)
    lam = 0.02 * float(np.abs(case["field"]).max())
    g, launches = gpu_solve3(torch, pd, case["field"], case["mask"], iters, lam=lam, b0=b0, weight=w)
    o = o3.solve3(case["field"], case["mask"], w, lambda_=lam, sigma=0.25, tau=0.25, max_iters=iters, b0_dir=b0)
    assert vol_rel(g, o).max() < (1e-5 if iters == 1 else 2e-5)
    assert launches == 2 + 3 + 12 * iters + 1
    # W = 1 everywhere through the literal path equals the Fourier-domain path up to rounding
    one = np.ones_like(w)
    g1, _ = gpu_solve3(torch, pd, case["field"], case["mask"], iters, lam=lam, b0=b0, weight=one)
    g0, _ = gpu_solve3(torch, pd, case["field"], case["mask"], iters, lam=lam, b0=b0)
    assert vol_rel(g1, g0).max() < 2e-5


@pytest.mark.parametrize("nx,ny,nz", [(64, 32, 25), (128, 64, 12), (64, 64, 42), (16, 8, 3), (32, 16, 64)])
def test_slice_counts_of_the_paper(torch, pd, o3, nx, ny, nz):
    """Any slice count up to 64 (25, 12 and 42 slices): dense z-line transform; two volumes + one alone."""
    case = synth.volume_case(nx, ny, nz, nvol=3, seed=nz, b0_axis=2)
    lam = 0.02 * float(np.abs(case["field"]).max())
    for iters, gate in [(1, 1e-5), (10, 2e-5)]:
        g, _ = gpu_solve3(torch, pd, case["field"], case["mask"], iters, lam=lam, b0=2)
        o = o3.solve3(case["field"], case["mask"], lambda_=lam, sigma=0.25, tau=0.25, max_iters=iters, b0_dir=2)
        assert vol_rel(g, o).max() < gate
    w = np.random.default_rng(nz).uniform(0.2, 1.0, size=case["field"].shape).astype(np.float32)
    g, _ = gpu_solve3(torch, pd, case["field"], case["mask"], 4, lam=lam, b0=0, weight=w)      # literal path, B0 along x
    o = o3.solve3(case["field"], case["mask"], w, lambda_=lam, sigma=0.25, tau=0.25, max_iters=4, b0_dir=0)
    assert vol_rel(g, o).max() < 2e-5


def test_automatic_steps_alpha_zero_and_max_iters_zero(torch, pd, o3):
    case = synth.volume_case(32, 16, 8, nvol=1, seed=3, b0_axis=0)
    s = 1.0 / np.sqrt(4.0 / 9.0 + 12.0)
    g, _ = gpu_solve3(torch, pd, case["field"], case["mask"], 6, lam=0.0, b0=0, sigma=0.0, tau=0.0)   # alpha = 0: q = 0 (R13)
    o = o3.solve3(case["field"], case["mask"], lambda_=0.0, sigma=s, tau=s, max_iters=6, b0_dir=0)
    assert vol_rel(g, o).max() < 1e-5
    g, n = gpu_solve3(torch, pd, case["field"], None, 0, lam=0.1, b0=0)
    assert not g.any() and n == 5


@pytest.mark.parametrize("ratio", [1e-2, 1e-3, 1e4])
def test_pair_partners_of_unequal_magnitude(torch, pd, o3, ratio):
    """Volumes 2k and 2k+1 share one complex transform; every volume is iterated in its own power-of-two normalisation
    (the iteration is invariant under (phi, alpha) -> (c phi, c alpha)), so a weak partner does not inherit the absolute
    rounding error of a strong one: the one-iteration gate holds for both."""
    case = synth.volume_case(64, 32, 16, nvol=3, seed=5, b0_axis=2)
    f = case["field"].copy()
    f[1] *= np.float32(ratio)
    lam = 0.02 * float(np.abs(case["field"]).max()) * min(1.0, ratio)    # active on the weak volume too
    for iters, gate in [(1, 1e-5), (10, 2e-5)]:
        g, _ = gpu_solve3(torch, pd, f, case["mask"], iters, lam=lam, b0=2)
        o = o3.solve3(f, case["mask"], lambda_=lam, sigma=0.25, tau=0.25, max_iters=iters, b0_dir=2)
        assert vol_rel(g, o).max() < gate, vol_rel(g, o)
    z = f.copy()
    z[0] = 0.0                                                           # a zero volume beside an active partner stays zero
    g, _ = gpu_solve3(torch, pd, z, case["mask"], 3, lam=lam, b0=2)
    assert not g[0].any() and g[1].any()


def test_chain_preprocess_solve3d_combine(torch, pd, o3):
    """Flow steps (1)-(5) on volumes: the two echo acquisitions of 3 coils -> field map, W, Mask (pd_preprocess) -> one
    weighted, masked 3-D solve per coil volume (pd_set_weight3d, pd_solve3d) -> pd_combine_coils; the CUDA chain against
    the oracle chain, every stage fed by its own side's previous stage."""
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import pd_prepost_oracle as po
    nx, ny, nz, nc, iters, thr = 64, 32, 16, 3, 10, 0.3
    e = synth.echo_volumes(nx, ny, nz, nc, seed=4)
    a, b = torch.from_numpy(e["s0"]).cuda(), torch.from_numpy(e["s1"]).cuda()
    f = torch.empty((nc, nz, ny, nx), device="cuda")
    w, m, chi = torch.empty_like(f), torch.empty_like(f), torch.empty_like(f)
    wmax = torch.zeros(1, device="cuda")
    pd.preprocess(a.view(nc * nz, ny, nx), b.view(nc * nz, ny, nx), e["fscale"], thr, field=f.view(nc * nz, ny, nx),
                  weight=w.view(nc * nz, ny, nx), mask=m.view(nc * nz, ny, nx), wmax=wmax)
    lam = 0.02 * float(np.abs(e["field"]).max())
    plan = pd.Plan3D(nx, ny, nz, nc, 2, lam, 0.25, 0.25, 1.0)
    plan.set_weight(w)
    plan.solve(f, m, chi, iters)
    out = torch.empty((1, nz * ny, nx), device="cuda")
    pd.combine_coils(chi.view(nc, nz * ny, nx), w.view(nc, nz * ny, nx), nc, out)      # one "slice" of nz*ny rows, nc coils
    torch.cuda.synchronize()
    plan.destroy()
    of = po.field_map(e["s0"], e["s1"], e["fscale"]).astype(np.float32)
    ow = po.weight(e["s0"], e["s1"], float(po.wscale_f32(e["s0"], e["s1"])))
    om = po.mask_f32(e["s0"], e["s1"], thr)
    assert np.array_equal(m.cpu().numpy(), om) and 0.05 < om.mean() < 0.95
    ochi = o3.solve3(of, om, ow.astype(np.float32), lambda_=lam, sigma=0.25, tau=0.25, max_iters=iters, b0_dir=2)
    assert vol_rel(chi.cpu().numpy(), ochi).max() < 1e-3
    ocomb = po.combine_coils(ochi.reshape(nc, nz * ny, nx), ow.reshape(nc, nz * ny, nx), nc)
    assert vol_rel(out.cpu().numpy(), ocomb).max() < 1e-3


def test_full_size_volume(torch, pd, o3):
    """The size bench.py --volume times per coil: 256 x 256 x 64, 10 iterations against the oracle."""
    case = synth.volume_case(256, 256, 64, nvol=1, seed=9, b0_axis=2)
    lam = 0.02 * float(np.abs(case["field"]).max())
    g, _ = gpu_solve3(torch, pd, case["field"], case["mask"], 10, lam=lam, b0=2)
    o = o3.solve3(case["field"], case["mask"], lambda_=lam, sigma=0.25, tau=0.25, max_iters=10, b0_dir=2)
    assert vol_rel(g, o).max() < 2e-5


def test_plan3d_errors(pd):
    import ctypes as C
    L, h = pd.lib(), C.c_void_p()
    assert L.pd_plan3d(C.byref(h), 8, 16, 16, 1, 2, 0.01, 0.25, 0.25, 1.0) == pd.ESIZE       # nx < 16
    assert L.pd_plan3d(C.byref(h), 64, 48, 16, 1, 2, 0.01, 0.25, 0.25, 1.0) == pd.ESIZE      # ny not a power of two
    assert L.pd_plan3d(C.byref(h), 64, 32, 100, 1, 2, 0.01, 0.25, 0.25, 1.0) == pd.ESIZE     # nz: a power of two, or <= 64
    assert L.pd_plan3d(C.byref(h), 512, 16, 16, 1, 2, 0.01, 0.25, 0.25, 1.0) == pd.ESIZE
    assert L.pd_plan3d(C.byref(h), 16, 8, 256, 600, 2, 0.01, 0.25, 0.25, 1.0) == pd.ESIZE     # 300 pairs x 256 planes > 65535
    assert L.pd_plan3d(C.byref(h), 64, 16, 16, 1, 3, 0.01, 0.25, 0.25, 1.0) == pd.EINVAL     # B0 axis
    assert L.pd_plan3d(C.byref(h), 64, 16, 16, 0, 2, 0.01, 0.25, 0.25, 1.0) == pd.EINVAL
    assert L.pd_plan3d(C.byref(h), 64, 16, 16, 1, 2, 0.01, 0.3, 0.3, 1.0) == pd.ESTEP        # 0.09 * 12.44 > 1
    assert h.value is None
    assert L.pd_solve3d(None, None, None, None, 1, None) == pd.EINVAL and L.pd_destroy3d(None) == pd.EINVAL
