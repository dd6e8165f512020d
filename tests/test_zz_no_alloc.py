"""pd_solve_static -- the allocation-free entry point (workspace in a file-scope static device array, include/pd.h) --
against the existing path: pd_plan + pd_solve through the streaming kernels, which it must reproduce (same kernels, same
launch order, same tables: the comparison is within the tests' tolerances and, in fact, bitwise), and against the
oracle.  Two calls in a row, with DIFFERENT inputs and shapes, share the array: the second must not see the first.
Collected last (pytest -x): a failure here hides nothing.  Passes alone in a fresh process as well.
"""
import numpy as np
import pytest

from paper_2006_09808_b200 import synth

pytestmark = pytest.mark.gpu

TOL_FULL = 1e-3   # tests/test_gpu_parity.py: per-slice relative L2 of chi after the full iteration count


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


def existing_path(torch, pd, f, m, iters, tol, lam, b0):
    """pd_plan + pd_solve, streaming variant, plain launches: what pd_solve_static restates without a plan."""
    batch, ny, nx = f.shape
    plan = pd.Plan(nx, ny, batch, b0, lam, 0.25, 0.25, 1.0)
    plan.set_option(pd.OPT_VARIANT, pd.VARIANT_STREAMING)
    plan.set_option(pd.OPT_GRAPH_LOOP, 0)
    out = torch.full_like(f, float("nan"))
    plan.solve(f, m, out, iters, tol)
    torch.cuda.synchronize()
    it, gap, res = plan.stats()
    plan.destroy()
    return out, it, gap, res


def static_outputs(torch, f):
    batch = f.shape[0]
    return (torch.full_like(f, float("nan")), torch.full((batch,), -1, dtype=torch.int32, device="cuda"),
            torch.full((batch,), float("nan"), device="cuda"), torch.full((batch,), float("nan"), device="cuda"))


def test_static_workspace_matches_existing_path_twice_in_a_row(torch, pd, oracle):
    # call 1: 5 slices of 128x128 (ragged last pair), mask, B0 along y; call 2, right after it on the same array: 7
    # slices of 64 rows x 128 columns (other tables, other plane offsets), B0 along x, tolerance stopping; call 3 repeats
    # call 1 (tables rebuilt once more, the stale state of call 2 in the array)
    cases = [(128, 128, 5, pd.B0_Y, 12, 0.0, 11), (128, 64, 7, pd.B0_X, 40, 5e-2, 12), (128, 128, 5, pd.B0_Y, 12, 0.0, 11)]
    for nx, ny, batch, b0, iters, tol, seed in cases:
        case = synth.random_case(nx, ny, batch, seed=seed, with_mask=True)
        f = torch.from_numpy(case["field"]).cuda()
        m = torch.from_numpy(np.ascontiguousarray(case["mask"])).cuda()
        ref, rit, rgap, rres = existing_path(torch, pd, f, m, iters, tol, 0.05, b0)
        # set-up call for this (nx, ny, B0): address of the array, tables; it also loads every kernel the next call uses
        warm = static_outputs(torch, f)
        pd.solve_static(f, m, warm[0], 1, 0.0, b0_dir=b0, lambda_=0.05, iters_done=warm[1], relgap=warm[2], relres=warm[3])
        got, it, gap, res = static_outputs(torch, f)
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        pd.solve_static(f, m, got, iters, tol, b0_dir=b0, lambda_=0.05, iters_done=it, relgap=gap, relres=res)
        torch.cuda.synchronize()
        # the driver's free-memory figure around the call: the equivalent cudaMalloc'ed workspace would be >= 4 MB
        assert free0 - torch.cuda.mem_get_info()[0] < (1 << 20)
        g, r = got.cpu().numpy(), ref.cpu().numpy()
        it, gap, res = it.cpu().numpy(), gap.cpu().numpy(), res.cpu().numpy()
        assert np.isfinite(g).all()
        assert slice_rel(g, r).max() < TOL_FULL
        assert np.array_equal(g, r), "same kernels, same order, same tables: expected bitwise agreement"
        assert np.array_equal(it, rit)
        assert np.allclose(gap, rgap, rtol=1e-3) and np.allclose(res, rres, rtol=1e-3)
        # and the oracle, on two slices (the first, and the unpaired last one)
        pick = [0, batch - 1]
        o = oracle.solve(case["field"][pick], case["mask"][pick], lambda_=0.05, sigma=0.25, tau=0.25, max_iters=iters,
                         tol=tol, b0_dir=b0)
        assert np.all(np.abs(it[pick] - o["iters_done"]) <= 1)
        same = it[pick] == o["iters_done"]          # a stop one iteration apart (R16) is another iterate
        assert same.any()
        assert slice_rel(g[pick][same], o["chi"][same]).max() < TOL_FULL


def test_static_workspace_rejects_what_does_not_fit(torch, pd):
    f = torch.zeros((2, 64, 64), device="cuda")
    out = torch.empty_like(f)

    def code(nx, ny, batch):
        return pd.lib().pd_solve_static(nx, ny, batch, pd.B0_Y, 0.05, 0.25, 0.25, 1.0, f.data_ptr(), None, out.data_ptr(),
                                        1, 0.0, None, None, None, None)
    assert code(512, 512, 1) == pd.ESTATIC                     # no 512-point lines in the static workspace
    assert code(256, 258, 2) == pd.ESTATIC                     # general lengths: pd_plan / pd_solve
    assert code(256, 256, 3) == pd.ESTATIC                     # 2 pairs of 256x256 = 131072 cells > 65536
    assert code(128, 128, 9) == pd.ESTATIC                     # 5 pairs of 128x128
    assert code(64, 64, pd.STATIC_MAX_BATCH + 1) == pd.ESTATIC
    assert code(64, 64, 0) == pd.EINVAL
    assert "65536" in pd.strerror(pd.ESTATIC) and "pd_solve" in pd.strerror(pd.ESTATIC)
    assert code(64, 64, 2) == pd.OK                            # the pointers above are real for exactly this shape
    torch.cuda.synchronize()
    assert float(out.abs().max()) == 0.0                       # a zero field gives chi = 0
    # the maximum sizes run: 32 slices of 64x64, 8 of 128x128, 2 of 256x256
    for n, batch in [(64, 32), (128, 8), (256, 2)]:
        case = synth.random_case(n, n, batch, seed=n, with_mask=False)
        g = torch.from_numpy(case["field"]).cuda()
        o = torch.full_like(g, float("nan"))
        pd.solve_static(g, None, o, 3, lambda_=0.05)
        plan = pd.Plan(n, n, batch, pd.B0_Y, 0.05, 0.25, 0.25, 1.0)
        plan.set_option(pd.OPT_VARIANT, pd.VARIANT_STREAMING)
        plan.set_option(pd.OPT_GRAPH_LOOP, 0)
        r = torch.full_like(g, float("nan"))
        plan.solve(g, None, r, 3, 0.0)
        torch.cuda.synchronize()
        plan.destroy()
        assert torch.equal(o, r)
