"""Pins of oracle/pd_prepost_oracle.py (NEXT-4: pre-processing and coil combination; readings R20-R22 of DESIGN.md)
against things other than itself: closed forms, hand-computed values, pure-Python brute force.  No GPU."""
import cmath
import math
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, os.path.join(ROOT, "oracle"))
import pd_prepost_oracle as po  # noqa: E402

from paper_2006_09808_b200 import synth  # noqa: E402


def test_p17_field_map_closed_form():
    """s0 = A e^{ia}, s1 = B e^{i(a+d)}  =>  field = d * fscale for d in (-pi, pi), whatever A, B, a (R20)."""
    rng = np.random.default_rng(17)
    d = np.linspace(-3.1, 3.1, 63).reshape(7, 9)
    a = rng.uniform(-np.pi, np.pi, d.shape)
    A, B = rng.uniform(0.1, 5.0, d.shape), rng.uniform(0.1, 5.0, d.shape)
    s0, s1 = A * np.exp(1j * a), B * np.exp(1j * (a + d))
    assert np.allclose(po.field_map(s0, s1, 0.37), 0.37 * d, atol=1e-12)
    # hand values: s0 = 1, s1 = i -> +pi/2 ; s1 = -i -> -pi/2 ; s1 = 1 + i -> pi/4 ; s0 = i, s1 = 1 -> -pi/2
    assert po.field_map(np.array([[1, 1, 1, 1j]]), np.array([[1j, -1j, 1 + 1j, 1]]), 1.0)[0].tolist() == \
        pytest.approx([math.pi / 2, -math.pi / 2, math.pi / 4, -math.pi / 2])
    # principal value: a difference of pi + 0.3 comes back as -pi + 0.3 (no unwrapping); exactly pi stays +pi
    assert po.field_map(np.array([[1.0]]), np.array([[cmath.exp(1j * (math.pi + 0.3))]]), 2.0)[0, 0] == pytest.approx(2 * (0.3 - math.pi))
    assert po.field_map(np.array([[2.0]]), np.array([[-3.0 + 0j]]), 1.0)[0, 0] == pytest.approx(math.pi)
    # antisymmetry under exchange of the two echoes, and a zero pixel gives 0
    assert np.allclose(po.field_map(s1, s0, 0.37), -po.field_map(s0, s1, 0.37))
    assert po.field_map(np.zeros((1, 1), complex), np.ones((1, 1), complex), 1.0)[0, 0] == 0.0
    assert po.field_map(np.zeros((1, 2), complex), np.array([[-1 - 1j, -2.0]]), 1.0).tolist() == [[0.0, 0.0]]   # not pi from a -0


def test_p17b_field_map_recovers_the_simulated_field():
    """On the synthetic echo pair without noise the field map IS the field the pair was built from (input recipe)."""
    e = synth.echo_pair(0, nslices=2, noise=0.0)
    got = po.field_map(e["s0"], e["s1"], e["fscale"])
    assert np.abs(got - e["field"]).max() < 2e-6 * e["fscale"] * 4   # complex64 storage of the inputs


def test_p18_weight_and_mask_hand_values():
    """|3+4i| = 5, |20i| = 20 -> m = sqrt(100) = 10 ; |2| = 2, |8| = 8 -> m = 4 ; zero pixel -> 0 (R21)."""
    s0 = np.array([[[3 + 4j, 2, 0, 1]]])
    s1 = np.array([[[20j, -8, 5, 1j]]])
    assert po.magnitude(s0, s1)[0, 0].tolist() == pytest.approx([10.0, 4.0, 0.0, 1.0])
    W = po.weight(s0, s1)
    assert W[0, 0].tolist() == pytest.approx([1.0, 0.4, 0.0, 0.1])          # scaled by the stack maximum
    assert po.weight(s0, s1, wscale=0.5)[0, 0].tolist() == pytest.approx([5.0, 2.0, 0.0, 0.5])
    assert po.mask_from_weight(W, 0.25).tolist() == [[[1.0, 1.0, 0.0, 0.0]]]
    assert po.mask_from_weight(W, 0.4 + 1e-12).tolist() == [[[1.0, 0.0, 0.0, 0.0]]]    # strict inequality
    assert po.weight(np.zeros((1, 2, 2), complex), np.zeros((1, 2, 2), complex)).max() == 0.0


def test_p18b_fp32_decisions_agree_with_the_definition_away_from_the_threshold():
    e = synth.echo_pair(0, nslices=3)
    W64 = po.weight(e["s0"], e["s1"])
    Wf = po.weight_f32(e["s0"], e["s1"])
    assert Wf.dtype == np.float32 and np.abs(Wf - W64).max() < 1e-6
    assert float(Wf.max()) == 1.0 or abs(float(Wf.max()) - 1.0) < 2e-7
    for thr in (0.3, 0.5, 0.7):
        mf, m64 = po.mask_f32(e["s0"], e["s1"], thr), po.mask_from_weight(W64, thr)
        far = np.abs(W64 - thr) > 1e-6
        assert far.mean() > 0.999 and np.array_equal(mf[far], m64[far])
        assert 0.02 < mf.mean() < 0.98                                        # both classes present
    # pure-Python restatement of the fp32 sequence on a few pixels (struct-free: numpy scalars, one rounding per step)
    f = np.float32
    for (b, y, x) in [(0, 0, 0), (1, 17, 40), (2, 63, 63), (0, 31, 5)]:
        z0, z1 = e["s0"][b, y, x], e["s1"][b, y, x]
        a0 = f(f(f(z0.real) * f(z0.real)) + f(f(z0.imag) * f(z0.imag)))
        a1 = f(f(f(z1.real) * f(z1.real)) + f(f(z1.imag) * f(z1.imag)))
        assert po.magnitude_f32(e["s0"], e["s1"])[b, y, x] == f(math.sqrt(f(math.sqrt(f(a0 * a1)))))


def test_p19_combine_coils_hand_values_and_brute_force():
    """chi = (1, 3): W = (1, 1) -> 2 ; W = (1, 2) -> (1 + 4*3)/5 = 2.6 ; W = (0, 0) -> 0 ; W = (0, 7) -> 3 (R22)."""
    chi = np.array([1.0, 3.0]).reshape(2, 1, 1)
    for w, want in [((1, 1), 2.0), ((1, 2), 2.6), ((0, 0), 0.0), ((0, 7), 3.0), ((-2, 1), 1.4)]:
        assert po.combine_coils(chi, np.array(w, float).reshape(2, 1, 1), 2)[0, 0, 0] == pytest.approx(want)
    rng = np.random.default_rng(19)
    ns, nc, ny, nx = 3, 4, 5, 6
    chi = rng.normal(size=(ns * nc, ny, nx))
    W = rng.uniform(0, 1, size=(ns * nc, ny, nx))
    W[rng.uniform(size=W.shape) < 0.2] = 0.0
    W[0:nc, 2, 3] = 0.0                                                        # a pixel no coil sees
    got = po.combine_coils(chi, W, nc)
    assert got.shape == (ns, ny, nx)
    for s in range(ns):                                                        # brute force, pure Python
        for y in range(ny):
            for x in range(nx):
                num = sum(W[s * nc + c, y, x] ** 2 * chi[s * nc + c, y, x] for c in range(nc))
                den = sum(W[s * nc + c, y, x] ** 2 for c in range(nc))
                assert got[s, y, x] == pytest.approx(num / den if den > 0 else 0.0, abs=1e-14)
    assert got[0, 2, 3] == 0.0
    # invariants: a common factor on the weights changes nothing ; identical coil maps come back unchanged where seen ;
    # the result lies between the smallest and largest coil value ; ncoils = 1 is the identity where W != 0
    assert np.allclose(po.combine_coils(chi, 3.7 * W, nc), got)
    same = np.repeat(rng.normal(size=(ns, 1, ny, nx)), nc, axis=1).reshape(ns * nc, ny, nx)
    seen = (W.reshape(ns, nc, ny, nx) ** 2).sum(1) > 0
    assert np.allclose(po.combine_coils(same, W, nc)[seen], same.reshape(ns, nc, ny, nx)[:, 0][seen])
    c4 = chi.reshape(ns, nc, ny, nx)
    assert np.all(got[seen] <= c4.max(1)[seen] + 1e-12) and np.all(got[seen] >= c4.min(1)[seen] - 1e-12)
    assert np.allclose(po.combine_coils(chi, W, 1)[W != 0], chi[W != 0])
    with pytest.raises(ValueError):
        po.combine_coils(chi[:5], W[:5], nc)
