"""CPU oracle of the steps either side of the iteration: pre-processing of the two echo-shifted
volumes into field map, weighting matrix and mask (flow step (1)) and the combination of the per-coil
susceptibility maps.

TEST INFRASTRUCTURE ONLY: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  Plain numpy, float64, one whole-array statement per step; pinned by tests/test_oracle_prepost_pins.py
against closed forms, hand-computed values and pure-Python brute force.

The paper names these steps and gives no formulas; the readings are DESIGN.md R20-R22 (that the code computes them is
pinned; that they are the authors' own pre-processing is PARITY UNPINNED -- there is nothing in the paper to pin against):
  R20  field = arg(s1 * conj(s0)) * fscale, principal value in (-pi, pi], 0 where the product is 0, no unwrapping ("two data were acquired (with or
       w/o echo shift) for measuring the field map"; fscale = 1 / (2 pi T_shift gamma B0) is the caller's).
  R21  magnitude m = sqrt(|s0| |s1|); W = m * wscale with wscale = 1 / max(m over the whole stack) unless given (so that
       |W| <= 1, which the step bound of PAPER.md:44 assumes); Mask = 1 where W > threshold, else 0.
  R22  chi(x) = sum_c W_c(x)^2 chi_c(x) / sum_c W_c(x)^2 over the coils of a slice, 0 where the denominator is 0 (the
       magnitude-squared weighted mean; every coil map is reconstructed independently).
Where floating point decides an integer (the mask; the stack maximum that scales W) the decision is specified in the
kernel's precision, fp32, as a fixed sequence of correctly rounded IEEE operations -- *_f32 below -- and the double
precision definition pins it away from the threshold.
"""
import numpy as np


def field_map(s0, s1, fscale):
    """R20.  s0, s1: complex [..][ny][nx]; returns float64."""
    d = np.asarray(s1, np.complex128) * np.conj(np.asarray(s0, np.complex128))
    return np.where(d == 0, 0.0, np.arctan2(d.imag, d.real)) * float(fscale)   # a zero product has no phase: 0


def magnitude(s0, s1):
    """R21: sqrt(|s0| |s1|), float64."""
    return np.sqrt(np.abs(np.asarray(s0, np.complex128)) * np.abs(np.asarray(s1, np.complex128)))


def weight(s0, s1, wscale=None):
    """R21: W = m * wscale, wscale = 1 / max(m) over everything passed in unless given.  float64."""
    m = magnitude(s0, s1)
    if wscale is None:
        mx = float(m.max())
        wscale = 1.0 / mx if mx > 0.0 else 0.0
    return m * float(wscale)


def mask_from_weight(W, threshold):
    """R21 in double precision (the definition): 1 where W > threshold."""
    return (np.asarray(W, np.float64) > float(threshold)).astype(np.float64)


def magnitude_f32(s0, s1):
    """The fp32 sequence behind the integer decisions: a_k = fl(fl(re_k^2) + fl(im_k^2)); m = sqrt(sqrt(fl(a_0 a_1))),
    every operation rounded to nearest in single precision, in this order, no fused multiply-add."""
    s0 = np.asarray(s0, np.complex64)
    s1 = np.asarray(s1, np.complex64)
    f = np.float32
    a0 = (s0.real.astype(f) * s0.real.astype(f)).astype(f) + (s0.imag.astype(f) * s0.imag.astype(f)).astype(f)
    a1 = (s1.real.astype(f) * s1.real.astype(f)).astype(f) + (s1.imag.astype(f) * s1.imag.astype(f)).astype(f)
    return np.sqrt(np.sqrt((a0.astype(f) * a1.astype(f)).astype(f)).astype(f)).astype(f)


def wscale_f32(s0, s1):
    """fl(1 / max(m_f32)) over the whole stack (0 when the stack is identically zero)."""
    mx = np.float32(magnitude_f32(s0, s1).max())
    return np.float32(1.0) / mx if mx > 0 else np.float32(0.0)


def weight_f32(s0, s1, wscale=None):
    w = wscale_f32(s0, s1) if wscale is None else np.float32(wscale)
    return (magnitude_f32(s0, s1) * w).astype(np.float32)


def mask_f32(s0, s1, threshold, wscale=None):
    """The mask as decided in fp32: fl(m_f32 * wscale) > fl(threshold)."""
    return (weight_f32(s0, s1, wscale) > np.float32(threshold)).astype(np.float32)


def combine_coils(chi, W, ncoils):
    """R22.  chi, W: [nslices*ncoils][ny][nx], batch index slice*ncoils + coil (BASELINE.json configs[3]).  Returns
    float64 [nslices][ny][nx]."""
    chi = np.asarray(chi, np.float64)
    W = np.asarray(W, np.float64)
    b, ny, nx = chi.shape
    if b % ncoils:
        raise ValueError("batch must be a multiple of ncoils")
    chi = chi.reshape(b // ncoils, ncoils, ny, nx)
    w2 = W.reshape(b // ncoils, ncoils, ny, nx) ** 2
    num = (w2 * chi).sum(axis=1)
    den = w2.sum(axis=1)
    out = np.zeros_like(num)
    np.divide(num, den, out=out, where=den > 0)
    return out
