"""Seeded input generator (paper_2006_09808_b200/synth.py) and the oracle regression fixture."""
import json
import os

import numpy as np

from paper_2006_09808_b200 import synth

HERE = os.path.dirname(os.path.abspath(__file__))


def test_streams_are_reproducible_and_distinct():
    k1 = synth.stream_key(2, 5, 0, 3)
    assert k1 == synth.stream_key(2, 5, 0, 3)
    keys = {int(synth.stream_key(c, s, co, p)) for c in range(3) for s in range(3) for co in range(2) for p in (1, 2, 3)}
    assert len(keys) == 54
    u = synth.uniform01(k1, 1000)
    assert np.array_equal(u, synth.uniform01(k1, 1000))
    assert np.array_equal(u[100:200], synth.uniform01(k1, 100, offset=100))   # counter based
    assert 0 <= u.min() and u.max() < 1 and abs(u.mean() - 0.5) < 0.05
    z = synth.normal01(k1, 200001)
    assert abs(z.mean()) < 0.01 and abs(z.std() - 1) < 0.01 and abs((z ** 3).mean()) < 0.03


def test_config_shapes_and_recipe():
    d = synth.generate(0, want_truth=True)
    assert d["field"].shape == (1, 64, 64) and d["field"].dtype == np.float32
    assert np.all(d["mask"] == 1)
    chi = d["chi_true"][0]
    assert 195 < chi.max() < 205 and (chi > 100).sum() in range(25, 33)      # disc r=3: 29 px
    assert np.abs(chi[chi < 100]).max() <= 0.1
    d1 = synth.generate(1, nslices=3, want_truth=True)
    assert d1["field"].shape == (3, 128, 128)
    assert abs(d1["mask"][0].sum() - np.pi * 60 ** 2) < 0.01 * np.pi * 60 ** 2
    assert all(140 < d1["chi_true"][i].max() < 520 for i in range(3))
    d2 = synth.generate(2, nslices=2, want_truth=True)
    seeds = (d2["chi_true"][0] == 180.0).sum()
    assert 100 < seeds <= 20 * 16                                            # 20 ellipses, pi*4.5*0.8 = 11.3 px each
    assert np.all(d2["mask"][0][d2["chi_true"][0] == 180.0] == 1)            # seeds lie inside the mask
    # subsets are prefixes of the full stack
    assert np.array_equal(synth.generate(2, nslices=1)["field"][0], d2["field"][0])
    assert np.array_equal(synth.generate(2, nslices=1, first_slice=1)["field"][0], d2["field"][1])


def test_multicoil_layout_and_noise_levels():
    d = synth.generate(3, nslices=2)
    f = d["field"].astype(np.float64)
    assert f.shape == (16, 256, 256)                                         # batch = slice*ncoils + coil
    # coils of one slice share the noiseless field: pairwise differences are pure noise, sigma in [0.005,0.02]*max|phi|
    amp = np.abs(f[:8].mean(axis=0)).max()
    for c in range(1, 8):
        sd = (f[c] - f[0]).std()
        assert 0.005 * amp * 0.9 < sd < 0.02 * amp * 1.6
    assert np.abs(f[8] - f[0]).max() > 10 * np.abs(f[1] - f[0]).std()        # next slice is a different phantom
    ns = synth.generate(5, nslices=2)
    assert ns["field"].shape == (2, 256, 256)


def test_simulated_field_agrees_with_oracle_operator(oracle):
    """The generator's measurement model (numpy.fft) and the oracle's K (own radix-2 FFT) are written separately;
    they must describe the same physics."""
    d = synth.generate(1, nslices=1, want_truth=True)
    chi = d["chi_true"][0]
    a = synth.simulate_field(chi, "y")
    b = oracle.apply_K(chi, oracle.B0_Y)
    assert np.linalg.norm(a - b) < 1e-12 * np.linalg.norm(b)
    noise = d["field"][0].astype(np.float64) - b
    assert abs(noise.std() / (0.01 * np.abs(b).max()) - 1) < 0.05


def test_golden_c0_oracle_regression(oracle):
    with open(os.path.join(HERE, "golden", "c0_oracle.json")) as f:
        g = json.load(f)
    d = synth.generate(0)
    cfg = d["cfg"]
    assert abs(np.linalg.norm(d["field"].astype(np.float64)) - g["field_l2"]) < 1e-9 * g["field_l2"]
    out = oracle.solve(d["field"], d["mask"], lambda_=cfg.lam, sigma=cfg.sigma, tau=cfg.tau, max_iters=cfg.iters)
    for n, gap, res in zip(g["iters"], g["relgap"], g["relres"]):
        assert abs(out["relgap"][0, n - 1] - gap) < 1e-9 * gap
        assert abs(out["relres"][0, n - 1] - res) < 1e-9 * res
    chi = out["chi"][0]
    assert abs(np.linalg.norm(chi) - g["chi_l2"]) < 1e-9 * g["chi_l2"]
    for k, v in g["chi_samples"].items():
        y, x = map(int, k.split(","))
        assert abs(chi[y, x] - v) < 1e-8 * max(1.0, abs(v))


def test_P13_gap_trajectory_matches_independent_probe(oracle):
    """SURVEY.md section 8(c) P13 lists a relgap / relres trajectory obtained with a separate NumPy probe on config-0-like
    input ("nearly input-independent"); the C++ oracle must reproduce its shape within 20 %."""
    d = synth.generate(0)
    out = oracle.solve(d["field"], d["mask"], lambda_=0.01, sigma=0.25, tau=0.25, max_iters=200)
    probe_gap = {1: .64, 2: .38, 3: .215, 5: 5.6e-2, 10: 7.1e-3, 20: 1.2e-2, 30: 2.4e-3, 50: 3.2e-4, 70: 1.0e-4,
                 100: 2.8e-5, 200: 2.2e-6}
    probe_res = {1: 1, 2: .638, 3: .457, 5: .277, 10: .115, 20: 3.3e-2, 50: 7.4e-3, 100: 2.7e-3, 200: 1.0e-3}
    for n, v in probe_gap.items():
        assert abs(out["relgap"][0, n - 1] / v - 1) < 0.2
    for n, v in probe_res.items():
        assert abs(out["relres"][0, n - 1] / v - 1) < 0.2
