"""GPU-vs-oracle parity through the C ABI (run on the B200 box: pytest -m gpu).

Gates (BASELINE.json north_star): per-slice relative L2 of chi <= 1e-5 after 1 iteration, <= 1e-3 after the full
iteration count; relgap within 1e-3 relative; |iters_done difference| <= 1 under tolerance stopping (R16).
Inputs come from paper_2006_09808_b200/synth.py; expected values only from oracle/ (double precision).
"""
import os

import numpy as np
import pytest

from paper_2006_09808_b200 import synth

pytestmark = pytest.mark.gpu

TOL_1IT = 1e-5
TOL_FULL = 1e-3


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def pd(torch):
    from paper_2006_09808_b200 import binding
    binding.lib()  # fails loudly if the extension is missing: there is no fallback
    return binding


def slice_rel(a, b):
    a = a.reshape(a.shape[0], -1).astype(np.float64)
    b = b.reshape(b.shape[0], -1).astype(np.float64)
    den = np.maximum(np.linalg.norm(b, axis=1), 1e-300)
    return np.linalg.norm(a - b, axis=1) / den


@pytest.fixture(params=["auto", "streaming"])
def variant(request):
    """auto = the resident cluster kernel where the size has one (square, <= 256), else streaming."""
    return request.param


def gpu_solve(torch, pd, field, mask, iters, *, lam, sigma=0.25, tau=0.25, theta=1.0, tol=0.0, weight=None, b0=1,
              options=(), host=False, variant="auto", b0_angle=None):
    batch, ny, nx = field.shape
    plan = pd.Plan(nx, ny, batch, b0, lam, sigma, tau, theta)
    if b0_angle is not None:
        plan.set_b0_angle(b0_angle)
    if variant == "streaming":
        plan.set_option(pd.OPT_VARIANT, pd.VARIANT_STREAMING)
    for k, v in options:
        plan.set_option(k, v)
    if host:
        chi = np.empty_like(field)
        plan.solve_host(field, mask, chi, iters, tol)
    else:
        f = torch.from_numpy(field).cuda()
        m = None if mask is None else torch.from_numpy(np.ascontiguousarray(mask)).cuda()
        w = None if weight is None else torch.from_numpy(weight).cuda()
        plan.set_weight(w)
        out = torch.full_like(f, float("nan"))
        plan.solve(f, m, out, iters, tol)
        torch.cuda.synchronize()
        chi = out.cpu().numpy()
    it, gap, res = plan.stats()
    launches = plan.last_launch_count
    tail = plan.hybrid_tail()
    plan.destroy()
    return {"chi": chi, "iters_done": it, "relgap": gap, "relres": res, "launches": launches, "hybrid_tail": tail}


def oracle_many(oracle, fields, masks, jobs, **kw):
    """The (single-threaded) oracle on several batch entries at once: a parallel-for over slices OUTSIDE the oracle, one
    call per entry on a thread pool over the host cores (the ctypes call releases the GIL).  jobs: [(b, max_iters)]."""
    import os
    from concurrent.futures import ThreadPoolExecutor

    def one(job):
        b, iters = job
        return oracle.solve(fields[b], None if masks is None else masks[b], max_iters=iters, **kw)
    with ThreadPoolExecutor(max_workers=os.cpu_count() or 1) as ex:
        return list(ex.map(one, jobs))


@pytest.mark.parametrize("ny,nx", [(64, 64), (128, 128), (256, 256), (512, 512), (64, 256), (512, 128), (128, 64)])
def test_one_iteration_all_sizes(torch, pd, oracle, ny, nx, variant):
    case = synth.random_case(nx, ny, 3, seed=nx + ny, with_mask=True, with_weight=True)   # odd batch: ragged last pair
    g = gpu_solve(torch, pd, case["field"], case["mask"], 1, lam=0.05, weight=case["weight"], variant=variant)
    o = oracle.solve(case["field"], case["mask"], case["weight"], lambda_=0.05, sigma=0.25, tau=0.25, max_iters=1)
    assert slice_rel(g["chi"], o["chi"]).max() < TOL_1IT
    assert np.allclose(g["relgap"], o["relgap"][:, 0], rtol=1e-4)
    assert np.all(g["iters_done"] == 1)


@pytest.mark.parametrize("n", [64, 128, 256])
@pytest.mark.parametrize("iters", [1, 2, 5])
def test_identity_weight_fourier_domain_dual(torch, pd, oracle, n, iters):
    """W = I: the resident kernel keeps p in the Fourier domain (one FFT round trip per iteration, gap by Parseval
    over mirror-paired columns).  Same gates as the literal path, and agreement with it (PD_OPT_FOURIER_DUAL = 0)."""
    case = synth.random_case(n, n, 5, seed=3 * n + iters, with_mask=True)        # odd batch: ragged last pair
    g = gpu_solve(torch, pd, case["field"], case["mask"], iters, lam=0.2)
    o = oracle.solve(case["field"], case["mask"], lambda_=0.2, sigma=0.25, tau=0.25, max_iters=iters)
    assert slice_rel(g["chi"], o["chi"]).max() < TOL_1IT
    assert np.allclose(g["relgap"], o["relgap"][:, iters - 1], rtol=1e-4)
    assert np.allclose(g["relres"], o["relres"][:, iters - 1], rtol=1e-3)
    lit = gpu_solve(torch, pd, case["field"], case["mask"], iters, lam=0.2, options=[(pd.OPT_FOURIER_DUAL, 0)])
    assert slice_rel(g["chi"], lit["chi"]).max() < TOL_1IT
    assert np.allclose(g["relgap"], lit["relgap"], rtol=1e-4)


@pytest.mark.parametrize("ny,nx", [(64, 64), (256, 256), (128, 64), (512, 512)])
@pytest.mark.parametrize("angle", [0.6, -1.1, np.pi / 4])
def test_oblique_in_plane_b0(torch, pd, oracle, variant, ny, nx, angle):
    """pd_set_b0_angle: B0 along (cos a, sin a); the table is the even part of D (the oracle's
    K takes the real part), so pairs of slices still ride one transform.  Same gates as the axis-aligned kernel."""
    case = synth.random_case(nx, ny, 3, seed=int(1000 * abs(angle)) + nx, with_mask=True)
    for iters in (1, 6):
        g = gpu_solve(torch, pd, case["field"], case["mask"], iters, lam=0.2, variant=variant, b0_angle=angle)
        o = oracle.solve(case["field"], case["mask"], lambda_=0.2, sigma=0.25, tau=0.25, max_iters=iters, b0_angle=angle)
        assert slice_rel(g["chi"], o["chi"]).max() < TOL_1IT
        assert np.allclose(g["relgap"], o["relgap"][:, iters - 1], rtol=1e-4)
    # the angle is not a no-op: the axis-aligned result differs
    ax = oracle.solve(case["field"], case["mask"], lambda_=0.2, sigma=0.25, tau=0.25, max_iters=6)
    assert slice_rel(g["chi"], ax["chi"]).min() > 1e-2


@pytest.mark.parametrize("ny,nx", [(64, 64), (128, 128), (256, 256), (512, 256), (64, 128)])
@pytest.mark.parametrize("weighted", [False, True])
def test_l1_regulariser_with_shrinkage(torch, pd, oracle, variant, ny, nx, weighted):
    """PD_REG_L1 (north_star's alternative regulariser): lambda ||M chi||_1, no q, soft shrinkage in
    the primal step.  Resident kernel (W = I, square <= 256), streaming two-launch path (W = I) and streaming literal
    path (W set) against the oracle's PDO_REG_L1; odd batch; the threshold is chosen so that it bites on part of the image."""
    case = synth.random_case(nx, ny, 5, seed=nx + 7 * ny, with_mask=True, with_weight=weighted)
    w = case["weight"] if weighted else None
    lam = 0.4
    for iters in (1, 2, 7):
        g = gpu_solve(torch, pd, case["field"], case["mask"], iters, lam=lam, weight=w, variant=variant,
                      options=[(pd.OPT_REGULARISER, pd.REG_L1)])
        o = oracle.solve(case["field"], case["mask"], w, lambda_=lam, sigma=0.25, tau=0.25, max_iters=iters,
                         regulariser=oracle.REG_L1)
        assert slice_rel(g["chi"], o["chi"]).max() < TOL_1IT, iters
        assert np.allclose(g["relgap"], o["relgap"][:, iters - 1], rtol=1e-4)
        assert np.allclose(g["relres"], o["relres"][:, iters - 1], rtol=1e-3)
    nzero = (o["chi"] == 0).mean()
    assert 0.01 < nzero < 0.98, nzero


def test_l1_regulariser_full_run_and_tolerance_stop(torch, pd, oracle, variant):
    """C1-sized phantoms, 200 iterations with the l1 regulariser, then a tolerance stop (relgap = data term of the
    Fenchel-Young gap): full-count gate, relgap and |iters_done difference| <= 1 (R16)."""
    d = synth.generate(1, nslices=5)
    cfg = d["cfg"]
    lam = 0.05
    opts = [(pd.OPT_REGULARISER, pd.REG_L1)]
    g = gpu_solve(torch, pd, d["field"], d["mask"], cfg.iters, lam=lam, variant=variant, options=opts)
    o = oracle.solve(d["field"], d["mask"], lambda_=lam, sigma=cfg.sigma, tau=cfg.tau, max_iters=cfg.iters, regulariser=oracle.REG_L1)
    assert slice_rel(g["chi"], o["chi"]).max() < TOL_FULL
    assert np.allclose(g["relgap"], o["relgap"][:, -1], rtol=1e-3)
    tol = float(np.sqrt(o["relgap"][:, 20].max() * o["relgap"][:, 60].min()))   # crossed somewhere between iterations 20 and 60
    gt = gpu_solve(torch, pd, d["field"], d["mask"], cfg.iters, lam=lam, tol=tol, variant=variant, options=opts)
    ot = oracle.solve(d["field"], d["mask"], lambda_=lam, sigma=cfg.sigma, tau=cfg.tau, max_iters=cfg.iters, tol=tol,
                      regulariser=oracle.REG_L1, want_hist=False)
    assert np.abs(gt["iters_done"].astype(int) - ot["iters_done"].astype(int)).max() <= 1
    assert np.all(gt["iters_done"] < cfg.iters)


@pytest.mark.parametrize("ny,nx", [(256, 258), (128, 132), (132, 128), (20, 12), (36, 66), (100, 6), (46, 94)])
def test_general_lengths_few_iterations(torch, pd, oracle, ny, nx):
    """Sizes that are not powers of two (the paper's matrices are 256x258 and 128x132):
    the general-length streaming kernels (two dense DFT stages per line, literal iteration) against the oracle, whose
    lines of such lengths are the O(n^2) definition.  Mask, weight, odd batch; 1, 2 and 5 iterations; then the l1
    regulariser, the anisotropic projection, an oblique B0 and a tolerance stop on the same kernels."""
    case = synth.random_case(nx, ny, 3, seed=nx + 5 * ny, with_mask=True, with_weight=True)
    kw = dict(lambda_=0.3, sigma=0.25, tau=0.25)
    for iters in (1, 2, 5):
        g = gpu_solve(torch, pd, case["field"], case["mask"], iters, lam=0.3, weight=case["weight"])
        o = _oracle_batch(oracle, case, iters, **kw)
        assert slice_rel(g["chi"], o["chi"]).max() < TOL_1IT, iters
        assert np.allclose(g["relgap"], o["relgap"], rtol=1e-4)
        assert np.allclose(g["relres"], o["relres"], rtol=1e-3)
        assert np.all(g["iters_done"] == iters)
    if nx * ny <= 132 * 128:
        g = gpu_solve(torch, pd, case["field"], case["mask"], 4, lam=0.3, weight=case["weight"], options=[(pd.OPT_REGULARISER, pd.REG_L1)])
        o = _oracle_batch(oracle, case, 4, regulariser=oracle.REG_L1, **kw)
        assert slice_rel(g["chi"], o["chi"]).max() < TOL_1IT
        g = gpu_solve(torch, pd, case["field"], case["mask"], 4, lam=0.3, weight=case["weight"], options=[(pd.OPT_TV_MODE, pd.TV_ANISO)], b0_angle=0.5)
        o = _oracle_batch(oracle, case, 4, tv_mode=oracle.TV_ANISO, b0_angle=0.5, **kw)
        assert slice_rel(g["chi"], o["chi"]).max() < TOL_1IT
        assert np.allclose(g["relgap"], o["relgap"], rtol=1e-4)


def _oracle_batch(oracle, case, iters, **kw):
    """oracle.solve over the slices of a small case in parallel threads; relgap / relres of the last iteration."""
    n = case["field"].shape[0]

    def one(b):
        w = None if case.get("weight") is None else case["weight"][b]
        return oracle.solve(case["field"][b], None if case["mask"] is None else case["mask"][b], w, max_iters=iters, **kw)
    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(max_workers=os.cpu_count() or 1) as ex:
        outs = list(ex.map(one, range(n)))
    return {"chi": np.concatenate([o["chi"] for o in outs]), "relgap": np.array([o["relgap"][0, iters - 1] for o in outs]),
            "relres": np.array([o["relres"][0, iters - 1] for o in outs]), "iters_done": np.array([o["iters_done"][0] for o in outs])}


def test_paper_matrix_sizes_full_runs(torch, pd, oracle):
    """Seeded stand-ins in the paper's own matrix sizes (synth configs 6-8).  E2/E3 (128x132): the full 200
    iterations on four slices, and a tolerance stop.  E1 (256x258): 100 iterations on two slices -- the oracle's O(n^2)
    line DFT costs 1-2 s per iteration of one such slice, so 200 iterations would take 4-8 minutes per slice."""
    from concurrent.futures import ThreadPoolExecutor
    d2, d1 = synth.generate(7, nslices=4), synth.generate(6, nslices=2)
    c2, c1 = d2["cfg"], d1["cfg"]
    kw2, kw1 = dict(lambda_=c2.lam, sigma=c2.sigma, tau=c2.tau), dict(lambda_=c1.lam, sigma=c1.sigma, tau=c1.tau)
    it1 = 100
    with ThreadPoolExecutor(max_workers=os.cpu_count() or 1) as ex:
        f1 = [ex.submit(oracle.solve, d1["field"][b], d1["mask"][b], max_iters=it1, **kw1) for b in range(2)]
        f2 = [ex.submit(oracle.solve, d2["field"][b], d2["mask"][b], max_iters=c2.iters, **kw2) for b in range(4)]
        g2 = gpu_solve(torch, pd, d2["field"], d2["mask"], c2.iters, lam=c2.lam)
        g1 = gpu_solve(torch, pd, d1["field"], d1["mask"], it1, lam=c1.lam)
        o1, o2 = [f.result() for f in f1], [f.result() for f in f2]
    for b, o in enumerate(o2):
        assert slice_rel(g2["chi"][b:b + 1], o["chi"]).max() < TOL_FULL
        assert abs(g2["relgap"][b] / o["relgap"][0, -1] - 1) < 1e-3
    for b, o in enumerate(o1):
        assert slice_rel(g1["chi"][b:b + 1], o["chi"]).max() < TOL_FULL
        assert abs(g1["relgap"][b] / o["relgap"][0, -1] - 1) < 1e-3
    assert np.all(g2["iters_done"] == c2.iters) and np.all(g1["iters_done"] == it1)
    # tolerance stop on E2: the oracle's trajectory gives the crossing (R16: +-1)
    tol = float(np.sqrt(max(o["relgap"][0, 40] for o in o2) * min(o["relgap"][0, 90] for o in o2)))
    gt = gpu_solve(torch, pd, d2["field"], d2["mask"], c2.iters, lam=c2.lam, tol=tol)
    for b, o in enumerate(o2):
        cross = int(np.argmax(o["relgap"][0] < tol)) + 1
        assert abs(int(gt["iters_done"][b]) - cross) <= 1, (b, gt["iters_done"][b], cross)
    assert gt["launches"] == 5 * (int(gt["iters_done"].max()) + 1) + 4


@pytest.mark.parametrize("ratio", [1e-2, 1e-3, 1e4])
@pytest.mark.parametrize("weighted", [False, True])
def test_pair_partners_of_unequal_magnitude(torch, pd, oracle, variant, ratio, weighted):
    """Two real slices ride one complex transform, whose twiddle multiplications mix the lanes'
    rounding errors.  Every slice is therefore iterated in its own power-of-two normalisation (pair_scale), and the data
    term of the gap is accumulated per lane: a slice 100 to 10000 times weaker (or stronger) than its partner still meets
    the ONE-iteration gate and the relgap gate.  lambda is scaled with the slice so that the projection is active."""
    n = 128
    case = synth.random_case(n, n, 4, seed=4242, with_mask=True, with_weight=weighted)
    field = case["field"].copy()
    field[1] *= np.float32(ratio)            # pair (0, 1): partner weaker / stronger ; pair (2, 3): equal
    w = case["weight"] if weighted else None
    for iters in (1, 6):
        g = gpu_solve(torch, pd, field, case["mask"], iters, lam=0.05, weight=w, variant=variant)
        o = oracle.solve(field, case["mask"], w, lambda_=0.05, sigma=0.25, tau=0.25, max_iters=iters)
        assert slice_rel(g["chi"], o["chi"]).max() < TOL_1IT, (iters, slice_rel(g["chi"], o["chi"]))
        assert np.allclose(g["relgap"], o["relgap"][:, iters - 1], rtol=1e-4)
    # the weak slice with a projection that matters at ITS scale: lambda scaled by the ratio, slices 0 and 1 swapped in
    lam = 0.05 * min(ratio, 1.0)
    g = gpu_solve(torch, pd, field[[1, 0, 2, 3]], case["mask"][[1, 0, 2, 3]], 6, lam=lam, variant=variant)
    o = oracle.solve(field[[1, 0, 2, 3]], case["mask"][[1, 0, 2, 3]], lambda_=lam, sigma=0.25, tau=0.25, max_iters=6)
    assert slice_rel(g["chi"], o["chi"]).max() < TOL_1IT
    assert np.allclose(g["relgap"], o["relgap"][:, 5], rtol=1e-4)


@pytest.mark.parametrize("ny,nx", [(64, 64), (128, 128), (256, 256), (512, 512), (64, 256), (512, 128), (128, 64)])
@pytest.mark.parametrize("iters", [1, 2, 5])
def test_streaming_fourier_domain_dual(torch, pd, oracle, ny, nx, iters):
    """W = I, streaming variant: two launches per iteration (pd_streaming_fd.cuh), every size including non-square.
    Same gates as the literal four-launch path (PD_OPT_FOURIER_DUAL = 0), and agreement with it."""
    case = synth.random_case(nx, ny, 5, seed=nx + 3 * ny + iters, with_mask=True)   # odd batch: ragged last pair
    g = gpu_solve(torch, pd, case["field"], case["mask"], iters, lam=0.2, variant="streaming")
    assert g["launches"] == 3 * iters + 4          # graphed loop: scale, init x2, per iteration cols + rows + loop control, finish
    o = oracle.solve(case["field"], case["mask"], lambda_=0.2, sigma=0.25, tau=0.25, max_iters=iters)
    assert slice_rel(g["chi"], o["chi"]).max() < TOL_1IT
    assert np.allclose(g["relgap"], o["relgap"][:, iters - 1], rtol=1e-4)
    assert np.allclose(g["relres"], o["relres"][:, iters - 1], rtol=1e-3)
    assert np.all(g["iters_done"] == iters)
    lit = gpu_solve(torch, pd, case["field"], case["mask"], iters, lam=0.2, variant="streaming",
                    options=[(pd.OPT_FOURIER_DUAL, 0)])
    assert lit["launches"] == 5 * iters + 4        # cols (returns at once in iteration 0), dual rows, cols, rows, loop control
    assert slice_rel(g["chi"], lit["chi"]).max() < TOL_1IT
    assert np.allclose(g["relgap"], lit["relgap"], rtol=1e-4)
    # the same solves with one stream launch per kernel (PD_OPT_GRAPH_LOOP = 0): bit-identical results
    for opts, count in (([(pd.OPT_GRAPH_LOOP, 0)], 2 * iters + 4), ([(pd.OPT_GRAPH_LOOP, 0), (pd.OPT_FOURIER_DUAL, 0)], 4 * iters + 3)):
        h = gpu_solve(torch, pd, case["field"], case["mask"], iters, lam=0.2, variant="streaming", options=opts)
        assert h["launches"] == count
        ref = g if len(opts) == 1 else lit
        assert np.array_equal(h["chi"], ref["chi"]) and np.array_equal(h["relgap"], ref["relgap"])


@pytest.mark.parametrize("tail", [1, 2, 4])
def test_hybrid_schedule_tail_through_streaming(torch, pd, oracle, tail):
    """256x256, W = I: the last `tail` slice pairs run through the streaming kernels on the plan's second stream while
    the resident clusters take the rest (PD_OPT_HYBRID_TAIL).  Same gates; stats of both parts land in one array."""
    case = synth.random_case(256, 256, 9, seed=900 + tail, with_mask=True)        # odd batch: ragged last pair
    iters = 4
    plan_opts = [(pd.OPT_HYBRID_TAIL, tail)]
    g = gpu_solve(torch, pd, case["field"], case["mask"], iters, lam=0.2, options=plan_opts)
    assert g["launches"] == 1 + 3 * iters + 4      # resident kernel + the graphed streaming loop of the tail
    o = oracle.solve(case["field"], case["mask"], lambda_=0.2, sigma=0.25, tau=0.25, max_iters=iters)
    assert slice_rel(g["chi"], o["chi"]).max() < TOL_1IT
    assert np.allclose(g["relgap"], o["relgap"][:, iters - 1], rtol=1e-4)
    assert np.allclose(g["relres"], o["relres"][:, iters - 1], rtol=1e-3)
    assert np.all(g["iters_done"] == iters)
    off = gpu_solve(torch, pd, case["field"], case["mask"], iters, lam=0.2, options=[(pd.OPT_HYBRID_TAIL, 0)])
    assert off["launches"] == 1
    assert slice_rel(g["chi"], off["chi"]).max() < TOL_1IT


def test_hybrid_schedule_with_l1_regulariser_and_oblique_b0(torch, pd, oracle):
    """The two halves of the hybrid schedule run different kernels (resident MODE = l1 / streaming sfd_rows_l1) and read
    two layouts of the same dipole table (thread-private order / [ny][nx]): both must follow PD_REG_L1 and pd_set_b0_angle."""
    case = synth.random_case(256, 256, 7, seed=77, with_mask=True)
    kw = dict(lambda_=0.4, sigma=0.25, tau=0.25, max_iters=5)
    g = gpu_solve(torch, pd, case["field"], case["mask"], 5, lam=0.4, b0_angle=0.9,
                  options=[(pd.OPT_HYBRID_TAIL, 2), (pd.OPT_REGULARISER, pd.REG_L1)])
    assert g["hybrid_tail"] == 2
    o = _oracle_batch(oracle, case, 5, regulariser=oracle.REG_L1, b0_angle=0.9, **{k: v for k, v in kw.items() if k != "max_iters"})
    assert slice_rel(g["chi"], o["chi"]).max() < TOL_1IT
    assert np.allclose(g["relgap"], o["relgap"], rtol=1e-4)
    g = gpu_solve(torch, pd, case["field"], case["mask"], 5, lam=0.4, b0_angle=0.9, options=[(pd.OPT_HYBRID_TAIL, 2)])
    o = _oracle_batch(oracle, case, 5, b0_angle=0.9, **{k: v for k, v in kw.items() if k != "max_iters"})
    assert slice_rel(g["chi"], o["chi"]).max() < TOL_1IT
    assert np.allclose(g["relgap"], o["relgap"], rtol=1e-4)


def test_hybrid_schedule_tolerance_stop(torch, pd, oracle):
    """Per-slice stopping under the hybrid schedule: the resident clusters and the streaming tail each stop their own
    slices on the device; both parts agree with the hybrid-off run and with the oracle's stop iteration (R16)."""
    d = synth.generate(2, nslices=7)          # C2 phantoms, 256x256
    tol = 2e-3
    g = gpu_solve(torch, pd, d["field"], d["mask"], 120, lam=0.005, tol=tol, options=[(pd.OPT_HYBRID_TAIL, 2)])
    off = gpu_solve(torch, pd, d["field"], d["mask"], 120, lam=0.005, tol=tol, options=[(pd.OPT_HYBRID_TAIL, 0)])
    assert np.abs(g["iters_done"].astype(int) - off["iters_done"].astype(int)).max() <= 1
    assert np.all(g["iters_done"] < 120) and np.all(g["iters_done"] > 0)
    for b in (0, 3, 4, 6):                    # two from the resident part, two from the tail (slices 3..6)
        ob = oracle.solve(d["field"][b], d["mask"][b], lambda_=0.005, sigma=0.25, tau=0.25,
                          max_iters=int(g["iters_done"][b]), want_hist=True)
        assert slice_rel(g["chi"][b:b + 1], ob["chi"]).max() < TOL_FULL
        assert abs(g["relgap"][b] / ob["relgap"][0, -1] - 1) < 1e-3
        assert g["relgap"][b] < tol


@pytest.mark.parametrize("ny,nx", [(64, 128), (256, 256), (512, 512)])
def test_streaming_without_mask(torch, pd, oracle, ny, nx):
    """mask = NULL (M = 1): the streaming row kernel neither builds nor reads the mask plane; 3 iterations also pass
    through all three chi buffers (chibar is recomputed from chi_n and chi_{n-1})."""
    case = synth.random_case(nx, ny, 3, seed=5 * nx + ny, with_mask=False)
    for iters in (1, 4):
        g = gpu_solve(torch, pd, case["field"], None, iters, lam=0.2, variant="streaming")
        o = oracle.solve(case["field"], None, lambda_=0.2, sigma=0.25, tau=0.25, max_iters=iters)
        assert slice_rel(g["chi"], o["chi"]).max() < TOL_1IT
        assert np.allclose(g["relgap"], o["relgap"][:, iters - 1], rtol=1e-4)
        assert np.allclose(g["relres"], o["relres"][:, iters - 1], rtol=1e-3)


@pytest.mark.parametrize("iters", [2, 3, 7])
def test_few_iterations_exercise_q_and_divergence(torch, pd, oracle, iters, variant):
    case = synth.random_case(128, 64, 4, seed=77, with_mask=True, with_weight=True)
    g = gpu_solve(torch, pd, case["field"], case["mask"], iters, lam=0.5, weight=case["weight"], variant=variant)
    o = oracle.solve(case["field"], case["mask"], case["weight"], lambda_=0.5, sigma=0.25, tau=0.25, max_iters=iters)
    assert slice_rel(g["chi"], o["chi"]).max() < TOL_1IT
    assert np.allclose(g["relgap"], o["relgap"][:, iters - 1], rtol=1e-3)
    assert np.allclose(g["relres"], o["relres"][:, iters - 1], rtol=1e-3)


def test_config0_full(torch, pd, oracle, variant):
    d = synth.generate(0)
    cfg = d["cfg"]
    g = gpu_solve(torch, pd, d["field"], d["mask"], cfg.iters, lam=cfg.lam, variant=variant)
    o = oracle.solve(d["field"], d["mask"], lambda_=cfg.lam, sigma=cfg.sigma, tau=cfg.tau, max_iters=cfg.iters)
    assert slice_rel(g["chi"], o["chi"]).max() < TOL_FULL
    assert slice_rel(g["chi"], o["chi"]).max() < 2e-5   # what fp32 actually achieves
    assert np.allclose(g["relgap"], o["relgap"][:, -1], rtol=1e-3)
    assert np.allclose(g["relres"], o["relres"][:, -1], rtol=1e-3)
    assert g["iters_done"][0] == 100


def test_config1_full(torch, pd, oracle, variant):
    d = synth.generate(1)
    cfg = d["cfg"]
    g = gpu_solve(torch, pd, d["field"], d["mask"], cfg.iters, lam=cfg.lam, variant=variant)
    o = oracle.solve(d["field"], d["mask"], lambda_=cfg.lam, sigma=cfg.sigma, tau=cfg.tau, max_iters=cfg.iters,
                     want_hist=True)
    r = slice_rel(g["chi"], o["chi"])
    assert r.max() < TOL_FULL and r.max() < 5e-5
    assert np.allclose(g["relgap"], o["relgap"][:, -1], rtol=1e-3)


def _sampled_full_config(torch, pd, oracle, cid, sample, host=False, variant="auto"):
    """Run the GPU on the FULL config (the launch configuration bench.py times); oracle on sampled batch entries."""
    d = synth.generate(cid)
    cfg = d["cfg"]
    # as bench.py: a config whose mask is all ones passes mask = NULL (M = 1)
    gmask = None if bool((d["mask"] == 1.0).all()) else d["mask"]
    g = gpu_solve(torch, pd, d["field"], gmask, cfg.iters, lam=cfg.lam, tol=cfg.tol, host=host, variant=variant)
    assert np.all(np.isfinite(g["chi"]))
    # property that holds at any size: every iterate has zero mean (DESIGN.md pin P7)
    means = np.abs(g["chi"].reshape(cfg.batch, -1).astype(np.float64).mean(axis=1))
    assert means.max() < 1e-3
    if callable(sample):   # sample chosen from what the plan did (e.g. both sides of the resident / streaming-tail split)
        sample = sample(g)
    sample = sorted(set(int(b) for b in sample if 0 <= b < cfg.batch))
    kw = dict(lambda_=cfg.lam, sigma=cfg.sigma, tau=cfg.tau)
    ors = oracle_many(oracle, d["field"], d["mask"], [(b, int(g["iters_done"][b]) if cfg.tol > 0 else cfg.iters) for b in sample], **kw)
    worst = 0.0
    for b, o in zip(sample, ors):
        rel = slice_rel(g["chi"][b:b + 1], o["chi"]).max()
        worst = max(worst, rel)
        assert rel < TOL_FULL, b
        assert abs(g["relgap"][b] / o["relgap"][0, -1] - 1) < 1e-3
    if cfg.tol > 0:   # the oracle's own stopping point may differ by one iteration at most (R16)
        from concurrent.futures import ThreadPoolExecutor
        with ThreadPoolExecutor(max_workers=os.cpu_count() or 1) as ex:
            osts = list(ex.map(lambda b: oracle.solve(d["field"][b], d["mask"][b], max_iters=cfg.iters, tol=cfg.tol, want_hist=False, **kw), sample))
        for b, ost in zip(sample, osts):
            assert abs(int(ost["iters_done"][0]) - int(g["iters_done"][b])) <= 1
    print("config %d: %d entries against the oracle, worst rel-L2 %.2e" % (cid, len(sample), worst))
    return d, g


def _split_sample(g, base):
    """base + both slices of the pair on each side of the resident / streaming-tail split + two more inside the tail."""
    batch = g["chi"].shape[0]
    tail = g["hybrid_tail"]
    s = list(base)
    if tail > 0:
        first_tail = 2 * ((batch + 1) // 2 - tail)
        s += [first_tail - 2, first_tail - 1, first_tail, first_tail + 1, first_tail + 2 * (tail // 2), batch - 2]
    return s


def test_config2_full_sampled(torch, pd, oracle):
    _sampled_full_config(torch, pd, oracle, 2, lambda g: _split_sample(g, [0, 1, 17, 30, 37, 44, 62, 63]))


def test_config3_full_sampled(torch, pd, oracle):
    """C3 as bench.py times it (pd_solve on device buffers, automatic hybrid tail): >= 16 entries against the oracle; then
    the whole batch against the same plan with the hybrid tail off and through the streaming kernels only."""
    d, g = _sampled_full_config(torch, pd, oracle, 3, lambda g: _split_sample(g, [0, 1, 5, 8, 255, 256, 511, 512, 777, 1022, 1023]))
    assert np.all(g["iters_done"] == 200)
    cfg = d["cfg"]
    assert g["hybrid_tail"] > 0
    off = gpu_solve(torch, pd, d["field"], d["mask"], cfg.iters, lam=cfg.lam, options=[(pd.OPT_HYBRID_TAIL, 0)])
    st = gpu_solve(torch, pd, d["field"], d["mask"], cfg.iters, lam=cfg.lam, variant="streaming")
    r_off, r_st = slice_rel(g["chi"], off["chi"]), slice_rel(g["chi"], st["chi"])
    print("C3 whole batch: hybrid vs hybrid-off %.2e, hybrid vs streaming-only %.2e (max per-slice rel-L2)" % (r_off.max(), r_st.max()))
    assert r_off.max() < 5e-5 and r_st.max() < 5e-5      # three schedules of the same arithmetic: fp32 rounding order only
    assert np.allclose(g["relgap"], off["relgap"], rtol=1e-3) and np.allclose(g["relgap"], st["relgap"], rtol=1e-3)


def test_config3_full_sampled_through_host_entry(torch, pd, oracle):
    d, g = _sampled_full_config(torch, pd, oracle, 3, [5, 30, 31, 150, 151, 600, 1023], host=True)
    assert np.all(g["iters_done"] == 200)


def test_northstar_stack_sampled(torch, pd, oracle, variant):
    _sampled_full_config(torch, pd, oracle, 5, lambda g: _split_sample(g, [0, 1, 31, 64, 90, 127]), variant=variant)


def test_config4_full_tolerance_stop_sampled(torch, pd, oracle):
    d, g = _sampled_full_config(torch, pd, oracle, 4, [0, 3, 64, 101, 128, 200, 254, 255])
    assert g["iters_done"].min() > 40 and g["iters_done"].max() < 140
    assert np.all(g["relgap"] < 1e-4)
    # the graphed loop stops launching one iteration after the last slice has stopped (not at max_iters = 500)
    assert g["launches"] == 3 * (int(g["iters_done"].max()) + 1) + 4


@pytest.mark.parametrize("ny,nx,batch,variant_", [(64, 64, 901, "auto"), (64, 128, 51, "streaming"), (256, 256, 61, "auto")])
def test_host_entry_pipeline_chunks(torch, pd, oracle, ny, nx, batch, variant_):
    """pd_solve_host cuts a large batch into chunks (upload k+1 || solve k || download k-1 on plan-owned streams): same
    chi and statistics as pd_solve on device buffers -- bit for bit where every slice runs through the same kernels
    (64x64: five chunks of resident waves; 64x128: three chunks of graphed streaming loops, odd batch), within the
    one-iteration gate where the hybrid tail may land elsewhere (256x256) -- and as the oracle on sampled slices."""
    case = synth.random_case(nx, ny, batch, seed=batch + nx, with_mask=True)
    iters, tol = (12, 0.0) if variant_ == "auto" else (40, 5e-2)
    dev = gpu_solve(torch, pd, case["field"], case["mask"], iters, lam=0.2, tol=tol, variant=variant_)
    host = gpu_solve(torch, pd, case["field"], case["mask"], iters, lam=0.2, tol=tol, variant=variant_, host=True,
                     options=[(pd.OPT_HOST_CHUNKING, 1)])   # small streaming batches are not chunked automatically
    assert np.array_equal(host["iters_done"], dev["iters_done"])
    if nx == 256:
        assert slice_rel(host["chi"], dev["chi"]).max() < TOL_1IT
    else:
        assert np.array_equal(host["chi"], dev["chi"]) and np.array_equal(host["relgap"], dev["relgap"])
    for b in (0, batch // 2, batch - 1):
        o = oracle.solve(case["field"][b], case["mask"][b], lambda_=0.2, sigma=0.25, tau=0.25, max_iters=int(host["iters_done"][b]))
        assert slice_rel(host["chi"][b:b + 1], o["chi"]).max() < TOL_1IT


def test_options_aniso_dataconv_sharedmask_b0x_theta(torch, pd, oracle, variant):
    case = synth.random_case(64, 128, 2, seed=5, with_mask=True)
    f, m = case["field"], case["mask"]
    g = gpu_solve(torch, pd, f, m, 20, lam=0.3, options=[(pd.OPT_TV_MODE, pd.TV_ANISO)], variant=variant)
    o = oracle.solve(f, m, lambda_=0.3, sigma=0.25, tau=0.25, max_iters=20, tv_mode=oracle.TV_ANISO)
    assert slice_rel(g["chi"], o["chi"]).max() < 2e-5
    assert np.allclose(g["relgap"], o["relgap"][:, -1], rtol=1e-3)
    g = gpu_solve(torch, pd, f, m, 20, lam=40.0, options=[(pd.OPT_LAMBDA_CONV, pd.LAMBDA_DATA)], variant=variant)
    o = oracle.solve(f, m, lambda_=40.0, sigma=0.25, tau=0.25, max_iters=20, lambda_conv=oracle.LAMBDA_DATA)
    assert slice_rel(g["chi"], o["chi"]).max() < 2e-5
    assert np.allclose(g["relgap"], o["relgap"][:, -1], rtol=1e-3)
    g = gpu_solve(torch, pd, f, m[0], 20, lam=0.3, options=[(pd.OPT_MASK_SHARED, 1)], variant=variant)
    o = oracle.solve(f, np.stack([m[0], m[0]]), lambda_=0.3, sigma=0.25, tau=0.25, max_iters=20)
    assert slice_rel(g["chi"], o["chi"]).max() < 2e-5
    g = gpu_solve(torch, pd, f, None, 20, lam=0.3, b0=0, theta=0.5, variant=variant)
    o = oracle.solve(f, None, lambda_=0.3, sigma=0.25, tau=0.25, theta=0.5, max_iters=20, b0_dir=oracle.B0_X)
    assert slice_rel(g["chi"], o["chi"]).max() < 2e-5
    g = gpu_solve(torch, pd, f, m, 20, lam=0.3, sigma=-1.0, tau=-1.0, variant=variant)   # automatic steps
    s = 1.0 / np.sqrt(8 + 4 / 9)
    o = oracle.solve(f, m, lambda_=0.3, sigma=np.float32(s), tau=np.float32(s), max_iters=20)
    assert slice_rel(g["chi"], o["chi"]).max() < 2e-5
    g = gpu_solve(torch, pd, f, m, 20, lam=0.0, variant=variant)                 # alpha = 0: q stays 0 (R13)
    o = oracle.solve(f, m, lambda_=0.0, sigma=0.25, tau=0.25, max_iters=20)
    assert slice_rel(g["chi"], o["chi"]).max() < 2e-5


def test_degenerate_cases(torch, pd, oracle, variant):
    f = synth.random_case(64, 64, 3, seed=9)["field"]
    f[1] = 0.0                                                                # an all-zero slice inside an active pair
    g = gpu_solve(torch, pd, f, None, 15, lam=0.1, tol=1e-9, variant=variant)
    assert g["iters_done"].tolist() == [15, 0, 15] and np.all(g["chi"][1] == 0)
    o = oracle.solve(f, None, lambda_=0.1, sigma=0.25, tau=0.25, max_iters=15)
    assert slice_rel(g["chi"][[0, 2]], o["chi"][[0, 2]]).max() < 2e-5
    g = gpu_solve(torch, pd, f, None, 15, lam=0.1, variant=variant)           # tol <= 0: runs N no-op iterations
    assert g["iters_done"].tolist() == [15, 15, 15] and np.all(g["chi"][1] == 0) and g["relgap"][1] == 0
    g = gpu_solve(torch, pd, f, None, 0, lam=0.1, variant=variant)            # max_iters = 0: chi_0 = 0
    assert np.all(g["chi"] == 0) and np.all(g["iters_done"] == 0)
    one = gpu_solve(torch, pd, f[:1], None, 15, lam=0.1, variant=variant)     # batch 1: half-empty pair
    assert slice_rel(one["chi"], o["chi"][:1]).max() < 2e-5


def test_per_slice_stop_mixed_batch(torch, pd, oracle, variant):
    """Slices of one batch stop at different iterations; a stopped slice is frozen while its pair partner goes on."""
    d = synth.generate(1, nslices=5)
    f = d["field"].copy()
    f[1] *= 1e-3          # different noise-to-signal ratios do not matter; different phantoms already differ
    tol = 3e-4
    g = gpu_solve(torch, pd, f, d["mask"], 300, lam=0.01, tol=tol, variant=variant)
    o = oracle.solve(f, d["mask"], lambda_=0.01, sigma=0.25, tau=0.25, max_iters=300, tol=tol)
    assert np.abs(g["iters_done"].astype(int) - o["iters_done"].astype(int)).max() <= 1
    assert len(set(g["iters_done"].tolist())) > 1
    for b in range(5):
        ob = oracle.solve(f[b], d["mask"][b], lambda_=0.01, sigma=0.25, tau=0.25, max_iters=int(g["iters_done"][b]),
                          want_hist=True)
        assert slice_rel(g["chi"][b:b + 1], ob["chi"]).max() < TOL_FULL
        assert abs(g["relgap"][b] / ob["relgap"][0, -1] - 1) < 1e-3
    ge = gpu_solve(torch, pd, f, d["mask"], 300, lam=0.01, tol=tol, options=[(pd.OPT_CHECK_EVERY, 8)], variant=variant)
    oe = oracle.solve(f, d["mask"], lambda_=0.01, sigma=0.25, tau=0.25, max_iters=300, tol=tol, check_every=8,
                      want_hist=False)
    assert np.all((ge["iters_done"] % 8 == 0) | (ge["iters_done"] == 300))
    assert np.abs(ge["iters_done"].astype(int) - oe["iters_done"].astype(int)).max() <= 8


def test_repeatable_and_plan_reuse(torch, pd):
    d = synth.generate(1, nslices=4)
    f = torch.from_numpy(d["field"]).cuda()
    m = torch.from_numpy(d["mask"]).cuda()
    plan = pd.Plan(128, 128, 4, 1, 0.01, 0.25, 0.25, 1.0)
    a, b = torch.empty_like(f), torch.empty_like(f)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        plan.solve(f, m, a, 50, 1e-3)
        plan.solve(f, m, b, 50, 1e-3)
    s.synchronize()
    assert torch.equal(a, b)                                                  # bitwise deterministic, stream honoured
    it, _, _ = plan.stats(s)
    assert it.max() <= 50
    plan.destroy()


@pytest.mark.parametrize("seed", range(24))
def test_seeded_random_option_combinations(torch, pd, oracle, seed):
    """A seeded differential sweep over combinations no other test pairs up: size (tuned, non-square, general length),
    variant, regulariser, projection mode, lambda convention, theta, B0 (axis or oblique), weight, shared mask, batch parity,
    iteration count, explicit or automatic steps -- each combination against the oracle with the same settings."""
    r = np.random.default_rng(1000 + seed)
    ny, nx = [(64, 64), (128, 128), (64, 128), (128, 64), (256, 256), (36, 66), (20, 12), (132, 128), (64, 66), (512, 64)][int(r.integers(10))]
    batch = int(r.integers(1, 6))
    iters = int(r.integers(1, 9))
    variant = ["auto", "streaming"][int(r.integers(2))]
    l1 = bool(r.integers(2))
    aniso = bool(r.integers(2)) and not l1
    conv_a = bool(r.integers(4) == 0)
    theta = [1.0, 1.0, 0.5, 0.0][int(r.integers(4))]
    angle = [None, None, float(r.uniform(-3, 3))][int(r.integers(3))]
    b0 = int(r.integers(2))
    weighted = bool(r.integers(3) == 0)
    shared = bool(r.integers(4) == 0)
    auto_steps = bool(r.integers(4) == 0)
    fd = bool(r.integers(4) != 0)
    lam = float([0.05, 0.3, 1.0][int(r.integers(3))])
    if conv_a:
        lam = 1.0 / lam
    sig = tau = 0.25
    case = synth.random_case(nx, ny, batch, seed=500 + seed, with_mask=True, with_weight=weighted)
    mask = case["mask"]
    if shared:
        mask = np.repeat(mask[:1], batch, axis=0)
    opts = []
    if l1:
        opts.append((pd.OPT_REGULARISER, pd.REG_L1))
    if aniso:
        opts.append((pd.OPT_TV_MODE, pd.TV_ANISO))
    if conv_a:
        opts.append((pd.OPT_LAMBDA_CONV, pd.LAMBDA_DATA))
    if shared:
        opts.append((pd.OPT_MASK_SHARED, 1))
    if not fd:
        opts.append((pd.OPT_FOURIER_DUAL, 0))
    gs = 0.0 if auto_steps else sig
    g = gpu_solve(torch, pd, case["field"], mask[0] if shared else mask, iters, lam=lam, sigma=gs, tau=gs, theta=theta,
                  weight=case["weight"] if weighted else None, b0=b0, options=opts, variant=variant, b0_angle=angle)
    if auto_steps:
        sig = tau = 1.0 / np.sqrt(4.0 / 9.0 + 8.0)
    kw = dict(lambda_=lam, sigma=sig, tau=tau, theta=theta, tv_mode=oracle.TV_ANISO if aniso else oracle.TV_ISO,
              lambda_conv=oracle.LAMBDA_DATA if conv_a else oracle.LAMBDA_REG, regulariser=oracle.REG_L1 if l1 else oracle.REG_TV)
    if angle is not None:
        kw["b0_angle"] = angle
    else:
        kw["b0_dir"] = b0
    o = _oracle_batch(oracle, dict(field=case["field"], mask=mask, weight=case["weight"] if weighted else None), iters, **kw)
    what = dict(size=(ny, nx), batch=batch, iters=iters, variant=variant, l1=l1, aniso=aniso, conv_a=conv_a, theta=theta, angle=angle,
                b0=b0, weighted=weighted, shared=shared, auto_steps=auto_steps, fd=fd, lam=lam)
    assert slice_rel(g["chi"], o["chi"]).max() < TOL_1IT, what
    assert np.allclose(g["relgap"], o["relgap"], rtol=1e-3), what
    assert np.all(g["iters_done"] == iters), what


def test_norm_bounds_for_automatic_steps(torch, pd, oracle, variant):
    """pd_set_norm_bounds (R14): mask values up to 2 and weights up to 1.5 with the automatic steps
    sigma = tau = 1/sqrt(4/9 max|W|^2 + 8 max|M|^2); PD_ESTEP follows the same bound."""
    case = synth.random_case(64, 64, 3, seed=14, with_mask=True, with_weight=True)
    m, w = 2.0 * case["mask"], 1.5 * case["weight"]
    step = 1.0 / np.sqrt(4.0 / 9.0 * 1.5 ** 2 + 8.0 * 2.0 ** 2)
    batch, ny, nx = case["field"].shape
    plan = pd.Plan(nx, ny, batch, pd.B0_Y, 0.3, 0.0, 0.0, 1.0)       # sigma = tau = 0: automatic
    if variant == "streaming":
        plan.set_option(pd.OPT_VARIANT, pd.VARIANT_STREAMING)
    plan.set_norm_bounds(1.5, 2.0)
    f, mm, ww = (torch.from_numpy(a).cuda() for a in (case["field"], m, w))
    plan.set_weight(ww)
    out = torch.empty_like(f)
    plan.solve(f, mm, out, 25, 0.0)
    torch.cuda.synchronize()
    o = oracle.solve(case["field"], m, w, lambda_=0.3, sigma=step, tau=step, max_iters=25)
    assert slice_rel(out.cpu().numpy(), o["chi"]).max() < 2e-5
    with pytest.raises(pd.PdError) as e:     # 0.25 * 0.25 * (1 + 32) > 1 under the stated bounds
        plan.set_steps(0.3, 0.25, 0.25)
    assert e.value.code == pd.ESTEP
    with pytest.raises(pd.PdError) as e:
        plan.set_norm_bounds(0.0, 1.0)
    assert e.value.code == pd.EINVAL
    plan.destroy()


def test_runtime_errors(torch, pd):
    plan = pd.Plan(64, 64, 2)
    f = torch.zeros(2, 64, 64, device="cuda")
    with pytest.raises(pd.PdError) as e:
        plan.solve(f, None, f.clone(), -1)
    assert e.value.code == pd.EINVAL
    with pytest.raises(pd.PdError) as e:
        plan.set_option(pd.OPT_VARIANT, 99)
    assert e.value.code == pd.EINVAL
    with pytest.raises(pd.PdError) as e:
        plan.set_steps(0.01, 0.5, 0.5)
    assert e.value.code == pd.ESTEP
    plan.destroy()
