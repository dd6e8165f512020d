#!/usr/bin/env python
"""Small solves through every kernel family of libpd_b200.so, for `compute-sanitizer`:

    compute-sanitizer --tool memcheck  python tests/sanitizer_smoke.py
    compute-sanitizer --tool synccheck python tests/sanitizer_smoke.py
    compute-sanitizer --tool racecheck python tests/sanitizer_smoke.py

No oracle, no assertions on values beyond "finite": the parity tests do that; this only drives the kernels (resident with
the state on chip, resident literal, streaming two-launch and literal, l1 regulariser, general lengths, hybrid schedule,
tolerance stop, graphed loop and plain launches, the static-workspace entry point, pre-processing and coil combination,
the 3-D variant) at sizes a sanitizer finishes in minutes.  Prints one line per case.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import torch  # noqa: E402

from paper_2006_09808_b200 import binding as pd, synth  # noqa: E402


def run(name, nx, ny, batch, iters, *, variant="auto", weight=False, options=(), tol=0.0, mask=True, angle=None):
    case = synth.random_case(nx, ny, batch, seed=nx + ny + batch, with_mask=mask, with_weight=weight)
    plan = pd.Plan(nx, ny, batch, pd.B0_Y, 0.2, 0.25, 0.25, 1.0)
    if variant == "streaming":
        plan.set_option(pd.OPT_VARIANT, pd.VARIANT_STREAMING)
    for k, v in options:
        plan.set_option(k, v)
    if angle is not None:
        plan.set_b0_angle(angle)
    f = torch.from_numpy(case["field"]).cuda()
    m = torch.from_numpy(case["mask"]).cuda() if mask else None
    w = torch.from_numpy(case["weight"]).cuda() if weight else None
    plan.set_weight(w)
    out = torch.full_like(f, float("nan"))
    plan.solve(f, m, out, iters, tol)
    torch.cuda.synchronize()
    it, gap, res = plan.stats()
    ok = bool(torch.isfinite(out).all().item())
    print("%-44s %4dx%-4d batch %2d  iters %s  finite %s" % (name, ny, nx, batch, list(it[:3]), ok), flush=True)
    plan.destroy()
    if not ok:
        raise SystemExit("non-finite output in " + name)


def main():
    assert torch.cuda.is_available()
    pd.lib()
    full = "--full" in sys.argv
    # resident, state on chip (W = I): one CTA pair, a 4-CTA cluster, an 8-CTA cluster with DSMEM halos
    run("resident tm 64", 64, 64, 3, 3)
    run("resident tm 128", 128, 128, 3, 3)
    run("resident tm 256 (hybrid off)", 256, 256, 3, 2, options=[(pd.OPT_HYBRID_TAIL, 0)])
    run("resident tm 128, l1", 128, 128, 2, 3, options=[(pd.OPT_REGULARISER, pd.REG_L1)])
    run("resident tm 64, aniso, tolerance stop", 64, 64, 4, 30, options=[(pd.OPT_TV_MODE, pd.TV_ANISO)], tol=5e-2)
    # resident literal (W set)
    run("resident literal 64, W", 64, 64, 3, 3, weight=True)
    run("resident literal 128, W", 128, 128, 2, 2, weight=True)
    # hybrid schedule: resident clusters + streaming tail on the second stream
    run("hybrid 256, tail 1", 256, 256, 5, 2, options=[(pd.OPT_HYBRID_TAIL, 1)])
    # streaming, W = I: two launches per iteration, graphed loop and plain launches, every line length
    run("streaming fd 64x128", 128, 64, 3, 3, variant="streaming")
    run("streaming fd 256x64, no mask", 64, 256, 3, 3, variant="streaming", mask=False)
    run("streaming fd 512x512", 512, 512, 2, 2, variant="streaming")
    run("streaming fd 128, plain launches, tol", 128, 128, 3, 30, variant="streaming", options=[(pd.OPT_GRAPH_LOOP, 0)], tol=5e-2)
    run("streaming fd 64, l1, oblique B0", 64, 64, 3, 3, variant="streaming", options=[(pd.OPT_REGULARISER, pd.REG_L1)], angle=0.6)
    # streaming literal (W set): four launches per iteration
    run("streaming literal 128x64, W", 64, 128, 3, 3, variant="streaming", weight=True)
    run("streaming literal 512x64, W", 64, 512, 2, 2, variant="streaming", weight=True)
    # general lengths (the paper's 132 and 258 among them)
    run("general 20x12", 12, 20, 3, 3, weight=True)
    run("general 128x132", 132, 128, 3, 2)
    run("general 36x66, l1, tol", 66, 36, 3, 20, options=[(pd.OPT_REGULARISER, pd.REG_L1)], tol=5e-2)
    if full:
        run("general 256x258", 258, 256, 2, 2)
        run("resident tm 256, two waves", 256, 256, 40, 2, options=[(pd.OPT_HYBRID_TAIL, 0)])
    # host-buffer entry point (chunked pipeline on plan-owned streams)
    case = synth.random_case(64, 64, 200, seed=5, with_mask=True)
    plan = pd.Plan(64, 64, 200, pd.B0_Y, 0.2, 0.25, 0.25, 1.0)
    chi = np.empty_like(case["field"])
    plan.solve_host(case["field"], case["mask"], chi, 3, 0.0)
    print("%-44s finite %s" % ("pd_solve_host 64x64 x200 (chunks)", bool(np.isfinite(chi).all())), flush=True)
    plan.destroy()
    # the allocation-free entry point (static workspace), the steps either side, the 3-D variant (both line-transform
    # families, the fused x kernel, the literal path with W)
    case = synth.random_case(128, 64, 5, seed=7, with_mask=True)
    f, m = torch.from_numpy(case["field"]).cuda(), torch.from_numpy(case["mask"]).cuda()
    out = torch.empty_like(f)
    pd.solve_static(f, m, out, 3, lambda_=0.2)
    torch.cuda.synchronize()
    print("%-44s finite %s" % ("pd_solve_static 64x128 x5", bool(torch.isfinite(out).all())), flush=True)
    e = synth.echo_pair(0, nslices=3)
    a, b = torch.from_numpy(e["s0"]).cuda(), torch.from_numpy(e["s1"]).cuda()
    fm, w, mk = (torch.empty(e["s0"].shape, device="cuda") for _ in range(3))
    wmax = torch.zeros(1, device="cuda")
    pd.preprocess(a, b, e["fscale"], 0.3, field=fm, weight=w, mask=mk, wmax=wmax)
    comb = torch.empty((1,) + tuple(fm.shape[1:]), device="cuda")
    pd.combine_coils(fm, w, 3, comb)
    torch.cuda.synchronize()
    print("%-44s finite %s" % ("pd_preprocess / pd_combine_coils", bool(torch.isfinite(fm).all() and torch.isfinite(comb).all())), flush=True)
    for name, (nx, ny, nz), weighted in [("3-D 16x8x8 (radix-2 lines)", (16, 8, 8), False), ("3-D 64x32x16 (register lines, fused x)", (64, 32, 16), False),
                                         ("3-D 64x32x16, W (literal)", (64, 32, 16), True)]:
        case = synth.volume_case(nx, ny, nz, nvol=3, seed=nx)
        f3, m3 = torch.from_numpy(case["field"]).cuda(), torch.from_numpy(case["mask"]).cuda()
        plan3 = pd.Plan3D(nx, ny, nz, 3, 2, 0.02, 0.25, 0.25, 1.0)
        if weighted:
            plan3.set_weight(0.2 + 0.8 * torch.rand(f3.shape, device="cuda"))
        out3 = torch.empty_like(f3)
        plan3.solve(f3, m3, out3, 3)
        torch.cuda.synchronize()
        plan3.destroy()
        print("%-44s finite %s" % (name, bool(torch.isfinite(out3).all())), flush=True)
    print("sanitizer_smoke: done")


if __name__ == "__main__":
    main()
