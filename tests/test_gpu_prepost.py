"""GPU-vs-oracle parity of the steps either side of the iteration (NEXT-4): pd_preprocess and pd_combine_coils through
the C ABI, and the whole chain pre-processing -> per-coil solves with W and Mask -> coil combination.

Tolerances: field map 2e-6 rad x fscale (fp32 products of the complex multiply + atan2f, compared modulo
the 2 pi wrap); weight bitwise against the oracle's fp32 sequence and 1e-6 against its double definition; mask and stack
maximum bitwise (integer decisions, taken in fp32 on both sides); combined map 2e-6 relative (+ 1e-7 max|chi|)."""
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


def slice_rel(a, b):
    a = a.reshape(a.shape[0], -1).astype(np.float64)
    b = b.reshape(b.shape[0], -1).astype(np.float64)
    return np.linalg.norm(a - b, axis=1) / np.maximum(np.linalg.norm(b, axis=1), 1e-300)


@pytest.fixture(scope="module")
def po():
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import pd_prepost_oracle
    return pd_prepost_oracle


def gpu_preprocess(torch, pd, s0, s1, fscale, thr, wscale=0.0):
    a, b = torch.from_numpy(s0).cuda(), torch.from_numpy(s1).cuda()
    f = torch.full(s0.shape, float("nan"), device="cuda")
    w, m = torch.full_like(f, float("nan")), torch.full_like(f, float("nan"))
    wmax = torch.full((4,), float("nan"), device="cuda")
    pd.preprocess(a, b, fscale, thr, wscale=wscale, field=f, weight=w, mask=m, wmax=wmax)
    torch.cuda.synchronize()
    return f.cpu().numpy(), w.cpu().numpy(), m.cpu().numpy(), wmax.cpu().numpy()


def check_preprocess(po, s0, s1, fscale, thr, got, wscale=None):
    f, w, m, wmax = got
    ref = po.field_map(s0, s1, fscale)
    d = (f.astype(np.float64) - ref) / fscale
    d = (d + np.pi) % (2 * np.pi) - np.pi                      # +pi and -pi are the same phase
    assert np.abs(d).max() < 2e-6
    assert np.array_equal(w, po.weight_f32(s0, s1, wscale))    # the same fp32 sequence: bit for bit
    scale64 = None if wscale is None else float(np.float32(wscale))
    assert np.abs(w - po.weight(s0, s1, scale64)).max() < 1e-6 * max(1.0, float(w.max()))
    assert np.array_equal(m, po.mask_f32(s0, s1, thr, wscale))
    if wscale is None:
        assert wmax[0] == po.magnitude_f32(s0, s1).max() and np.isnan(wmax[1:]).all()


@pytest.mark.parametrize("cid,nslices", [(0, 3), (3, 1)])
def test_preprocess_matches_oracle(torch, pd, po, cid, nslices):
    e = synth.echo_pair(cid, nslices=nslices)                  # C0: 64x64 single coil ; C3: 8 coil maps of 256x256
    got = gpu_preprocess(torch, pd, e["s0"], e["s1"], e["fscale"], 0.3)
    check_preprocess(po, e["s0"], e["s1"], e["fscale"], 0.3, got)
    assert 0.05 < got[2].mean() < 0.95
    # and the field the pair was built from comes back (noise 0.01 on magnitudes >= 0.03: a loose sanity bound)
    inside = got[1] > 0.5
    assert np.abs(got[0] - e["field"])[inside].mean() < 0.05 * e["fscale"]
    # a given scale instead of the automatic one
    got = gpu_preprocess(torch, pd, e["s0"], e["s1"], e["fscale"], 0.5, wscale=0.75)
    check_preprocess(po, e["s0"], e["s1"], e["fscale"], 0.5, got, wscale=0.75)


@pytest.mark.parametrize("shape", [(1, 5, 7), (3, 1, 2), (1, 1, 1), (2, 33, 66)])
def test_preprocess_ragged_sizes_and_special_pixels(torch, pd, po, shape):
    rng = np.random.default_rng(sum(shape))
    s0 = (rng.normal(size=shape) + 1j * rng.normal(size=shape)).astype(np.complex64)
    s1 = (rng.normal(size=shape) + 1j * rng.normal(size=shape)).astype(np.complex64)
    s0.flat[0] = 0                                             # zero product: field 0, weight 0
    if s0.size > 2:
        s1.flat[2] = 0
        s1.flat[1] = s0.flat[1] * np.complex64(2.0)            # zero phase difference
    got = gpu_preprocess(torch, pd, s0, s1, 0.5, 0.4)
    check_preprocess(po, s0, s1, 0.5, 0.4, got)
    assert got[0].flat[0] == 0.0 and got[1].flat[0] == 0.0 and got[2].flat[0] == 0.0


def test_preprocess_optional_outputs_and_errors(torch, pd, po):
    e = synth.echo_pair(0, nslices=1)
    a, b = torch.from_numpy(e["s0"]).cuda(), torch.from_numpy(e["s1"]).cuda()
    m = torch.full(e["s0"].shape, float("nan"), device="cuda")
    wmax = torch.zeros(1, device="cuda")
    pd.preprocess(a, b, 1.0, 0.3, mask=m, wmax=wmax)          # only the mask
    torch.cuda.synchronize()
    assert np.array_equal(m.cpu().numpy(), po.mask_f32(e["s0"], e["s1"], 0.3))
    L = pd.lib()
    assert L.pd_preprocess(a.data_ptr(), b.data_ptr(), a.numel(), 1.0, 0.0, 0.3, None, None, m.data_ptr(), None, None) == pd.EINVAL
    assert L.pd_preprocess(None, b.data_ptr(), a.numel(), 1.0, 1.0, 0.3, None, None, m.data_ptr(), None, None) == pd.EINVAL
    assert L.pd_preprocess(a.data_ptr() + 8, b.data_ptr(), 4, 1.0, 1.0, 0.3, None, None, m.data_ptr(), None, None) == pd.EINVAL
    assert L.pd_preprocess(a.data_ptr(), b.data_ptr(), 0, 1.0, 1.0, 0.3, None, None, None, None, None) == pd.OK
    assert L.pd_combine_coils(None, None, 1, 1, 4, 4, None, None) == pd.EINVAL
    assert L.pd_combine_coils(m.data_ptr(), m.data_ptr(), 1, 0, 4, 4, m.data_ptr(), None) == pd.EINVAL


@pytest.mark.parametrize("ns,nc,ny,nx", [(3, 8, 128, 128), (2, 3, 5, 7), (4, 1, 64, 64), (1, 32, 2, 2)])
def test_combine_coils_matches_oracle(torch, pd, po, ns, nc, ny, nx):
    rng = np.random.default_rng(ns * 1000 + nc)
    chi = rng.normal(size=(ns * nc, ny, nx)).astype(np.float32)
    W = rng.uniform(0, 1, size=chi.shape).astype(np.float32)
    W[rng.uniform(size=W.shape) < 0.2] = 0.0
    W[0:nc, 0, 0] = 0.0                                        # a pixel no coil sees
    out = torch.full((ns, ny, nx), float("nan"), device="cuda")
    pd.combine_coils(torch.from_numpy(chi).cuda(), torch.from_numpy(W).cuda(), nc, out)
    torch.cuda.synchronize()
    g, o = out.cpu().numpy(), po.combine_coils(chi, W, nc)
    assert g[0, 0, 0] == 0.0
    assert np.allclose(g, o, rtol=2e-6, atol=1e-7 * float(np.abs(chi).max()))


def test_chain_preprocess_solve_combine(torch, pd, po, oracle):
    """Flow steps (1)-(5) and the coil combination on 2 slices x 8 coils of 256x256 (the shape of C3): the CUDA chain
    against the oracle chain, every stage fed by its own side's previous stage."""
    e = synth.echo_pair(3, nslices=2)
    cfg, iters, thr, lam = e["cfg"], 12, 0.3, 0.02
    batch, ny, nx = e["s0"].shape
    a, b = torch.from_numpy(e["s0"]).cuda(), torch.from_numpy(e["s1"]).cuda()
    f = torch.empty((batch, ny, nx), device="cuda")
    w, m, chi = torch.empty_like(f), torch.empty_like(f), torch.empty_like(f)
    wmax = torch.zeros(1, device="cuda")
    out = torch.empty((batch // cfg.ncoils, ny, nx), device="cuda")
    pd.preprocess(a, b, e["fscale"], thr, field=f, weight=w, mask=m, wmax=wmax)
    plan = pd.Plan(nx, ny, batch, pd.B0_Y, lam, 0.25, 0.25, 1.0)
    plan.set_weight(w)
    plan.solve(f, m, chi, iters, 0.0)
    pd.combine_coils(chi, w, cfg.ncoils, out)
    torch.cuda.synchronize()
    plan.destroy()
    # the oracle chain (double precision values, fp32 mask decision)
    of = po.field_map(e["s0"], e["s1"], e["fscale"]).astype(np.float32)
    ow = po.weight(e["s0"], e["s1"], float(po.wscale_f32(e["s0"], e["s1"])))
    om = po.mask_f32(e["s0"], e["s1"], thr)
    assert np.array_equal(m.cpu().numpy(), om)
    ow32 = ow.astype(np.float32)
    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(max_workers=os.cpu_count() or 1) as ex:
        res = list(ex.map(lambda k: oracle.solve(of[k], om[k], ow32[k], lambda_=lam, sigma=0.25, tau=0.25, max_iters=iters)["chi"][0],
                          range(batch)))
    ochi = np.stack(res)
    assert slice_rel(chi.cpu().numpy(), ochi).max() < 1e-3
    ocomb = po.combine_coils(ochi, ow, cfg.ncoils)
    assert slice_rel(out.cpu().numpy(), ocomb).max() < 1e-3
