"""Seeded synthetic inputs shaped like the workloads of arXiv 2006.09808 (configs C0..C4).

This module serves BOTH the CPU oracle tests and the CUDA path, and therefore holds none of the
solver's arithmetic: no PD step, no prox, no gradient, no solver FFT.  It only *simulates the
measurement*: a susceptibility phantom chi_true, the field it would induce (numpy.fft in float64
with the dipole kernel fixed by BASELINE.json north_star) and additive Gaussian noise.  Neither
the oracle nor the CUDA kernels import anything from here but the arrays it returns.

The paper's three datasets (stent 256x258x25, seeds in meat 128x132x12, needle
128x132x42) are not available; these stand in for them.  Recipe: DESIGN.md "Input recipe"
(SURVEY.md section 8(d)).

Random numbers: a counter-based generator -- SplitMix64's output function applied to
key + (i+1)*golden -- so that every (config, slice, coil, purpose) stream is reproducible and
independent of generation order.  Normal deviates by Box-Muller.
"""
from dataclasses import dataclass, field as _dc_field

import numpy as np

BASE_SEED = 200609808
_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)

# purposes (stream ids)
_BG, _SHAPES, _NOISE, _COILSIG = 1, 2, 3, 4


def _mix64(z):
    z = np.asarray(z, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        return z ^ (z >> np.uint64(31))


def stream_key(config, slice_, coil, purpose, base_seed=BASE_SEED):
    """64-bit key of one random stream: f(base_seed, config, slice, coil, purpose)."""
    k = _mix64(np.uint64(base_seed))
    for v in (config, slice_, coil, purpose):
        with np.errstate(over="ignore"):
            k = _mix64(k ^ (np.uint64(v + 1) * _GOLDEN))
    return np.uint64(k)


def uniform01(key, n, offset=0):
    """n doubles in [0,1): counter i -> mix64(key + (i+1)*golden) >> 11 scaled by 2^-53."""
    i = np.arange(offset + 1, offset + n + 1, dtype=np.uint64)
    with np.errstate(over="ignore"):
        bits = _mix64(np.uint64(key) + i * _GOLDEN)
    return (bits >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def normal01(key, n):
    """n standard normal deviates (Box-Muller on consecutive pairs of the stream)."""
    m = (n + 1) // 2
    u = uniform01(key, 2 * m)
    u1 = 1.0 - u[0::2]  # (0,1]
    u2 = u[1::2]
    r = np.sqrt(-2.0 * np.log(u1))
    z = np.empty(2 * m, np.float64)
    z[0::2] = r * np.cos(2.0 * np.pi * u2)
    z[1::2] = r * np.sin(2.0 * np.pi * u2)
    return z[:n]


class _Stream:
    """Sequential reader of one uniform stream (for rejection sampling of shape centres)."""

    def __init__(self, key):
        self.key, self.pos = key, 0

    def u(self, n=1):
        out = uniform01(self.key, n, self.pos)
        self.pos += n
        return out if n > 1 else float(out[0])


def dipole_kernel(nx, ny, b0_dir="y"):
    """Measurement model only: D = 1/3 - k_b^2/(kx^2+ky^2), D(0,0)=0 (BASELINE.json north_star)."""
    kx = np.fft.fftfreq(nx)[None, :]
    ky = np.fft.fftfreq(ny)[:, None]
    k2 = kx * kx + ky * ky
    kb2 = (ky * ky if b0_dir == "y" else kx * kx) + 0.0 * k2
    D = np.zeros((ny, nx))
    nz = k2 > 0
    D[nz] = 1.0 / 3.0 - kb2[nz] / k2[nz]
    return D


def simulate_field(chi_true, b0_dir="y"):
    """Noise-free field the phantom would induce: IFFT2(D * FFT2(chi_true)), float64."""
    ny, nx = chi_true.shape[-2:]
    D = dipole_kernel(nx, ny, b0_dir)
    return np.real(np.fft.ifft2(D * np.fft.fft2(chi_true, axes=(-2, -1)), axes=(-2, -1)))


def background(nx, ny, key):
    """U[-0.1,0.1] i.i.d. per pixel, then a 5x5 box mean with periodic wrap."""
    bg = (uniform01(key, nx * ny) * 0.2 - 0.1).reshape(ny, nx)
    acc = np.zeros_like(bg)
    for dy in range(-2, 3):
        for dx in range(-2, 3):
            acc += np.roll(np.roll(bg, dy, axis=0), dx, axis=1)
    return acc / 25.0


def _disc(nx, ny, cx, cy, r):
    yy, xx = np.mgrid[0:ny, 0:nx]
    return ((xx - cx) ** 2 + (yy - cy) ** 2) <= r * r


def _ellipse(nx, ny, cx, cy, a, b, ang):
    """Pixels with (u/a)^2+(v/b)^2 <= 1, (u,v) the coordinates rotated by ang about (cx,cy)."""
    yy, xx = np.mgrid[0:ny, 0:nx]
    dx, dy = xx - cx, yy - cy
    u = dx * np.cos(ang) + dy * np.sin(ang)
    v = -dx * np.sin(ang) + dy * np.cos(ang)
    return (u / a) ** 2 + (v / b) ** 2 <= 1.0


@dataclass
class Config:
    cid: int
    name: str
    nx: int
    ny: int
    nslices: int
    ncoils: int
    iters: int
    lam: float
    tol: float = 0.0
    sigma: float = 0.25
    tau: float = 0.25
    theta: float = 1.0
    b0_dir: str = "y"
    extra: dict = _dc_field(default_factory=dict)

    @property
    def batch(self):
        return self.nslices * self.ncoils


CONFIGS = {
    0: Config(0, "C0 1x64x64 needle", 64, 64, 1, 1, 100, 0.01),
    1: Config(1, "C1 16x128x128 cylinders", 128, 128, 16, 1, 200, 0.01),
    2: Config(2, "C2 64x256x256 brachytherapy seeds", 256, 256, 64, 1, 200, 0.005),
    3: Config(3, "C3 128x8coils x256x256 seeds", 256, 256, 128, 8, 200, 0.005),
    4: Config(4, "C4 256x512x512 mixed, tol stop", 512, 512, 256, 1, 500, 0.002, tol=1e-4),
}
# The stack BASELINE.json's north_star quotes its target on: 128 slices of 256x256, 200 iterations
# (C3's phantoms with a single coil map per slice).
CONFIGS[5] = Config(5, "NS 128x256x256 seeds (north-star stack)", 256, 256, 128, 1, 200, 0.005)
# Stand-ins in the PAPER'S OWN matrix sizes (256x258x25, 128x132x12, 128x132x42; the data sets themselves are
# not available): E1 with C2's seed phantoms, E2 and E3 with C1's cylinders; x (fastest axis) takes the odd length.
# `like` names the config whose phantom and mask recipe is reused (its random streams too, scaled to the new size).
CONFIGS[6] = Config(6, "E1 25x256x258 seeds (paper's matrix)", 258, 256, 25, 1, 200, 0.005, extra={"like": 2})
CONFIGS[7] = Config(7, "E2 12x128x132 cylinders (paper's matrix)", 132, 128, 12, 1, 200, 0.01, extra={"like": 1})
CONFIGS[8] = Config(8, "E3 42x128x132 cylinders (paper's matrix)", 132, 128, 42, 1, 200, 0.01, extra={"like": 1})


def _like(cfg):
    """The config whose phantom / mask recipe `cfg` uses (itself unless it is one of the paper-sized stand-ins)."""
    return CONFIGS[cfg.extra["like"]] if "like" in cfg.extra else cfg


def _mask(cfg, nx, ny):
    cfg = _like(cfg)
    if cfg.cid in (0, 4):
        return np.ones((ny, nx), np.float32)
    if cfg.cid == 1:
        return _disc(nx, ny, nx / 2.0, ny / 2.0, 60.0 * nx / 128.0).astype(np.float32)
    yy, xx = np.mgrid[0:ny, 0:nx]  # C2, C3, NS: centred ellipse, semi-axes (0.45 nx, 0.40 ny)
    return ((((xx - nx / 2.0) / (0.45 * nx)) ** 2 + ((yy - ny / 2.0) / (0.40 * ny)) ** 2) <= 1.0).astype(np.float32)


def _phantom(cfg, s, nx, ny):
    """chi_true of slice s (float64 [ny][nx])."""
    cfg = _like(cfg)
    pcid = 3 if cfg.cid == 5 else cfg.cid  # the north-star stack reuses C3's per-slice phantoms
    chi = background(nx, ny, stream_key(pcid, s, 0, _BG))
    st = _Stream(stream_key(pcid, s, 0, _SHAPES))
    if cfg.cid == 0:
        r = 3.0
        cx = (r + 8) + st.u() * (nx - 2 * (r + 8))
        cy = (r + 8) + st.u() * (ny - 2 * (r + 8))
        chi = chi + 200.0 * _disc(nx, ny, cx, cy, r)
    elif cfg.cid == 1:
        k = 1 + int(st.u() * 3)
        for _ in range(k):
            r = float(2 + int(st.u() * 4))
            val = 150.0 + 100.0 * st.u()
            while True:  # centre uniform inside radius 50 of the slice centre (rejection)
                dx, dy = (2 * st.u() - 1) * 50.0, (2 * st.u() - 1) * 50.0
                if dx * dx + dy * dy <= 2500.0:
                    break
            chi = chi + val * _disc(nx, ny, nx / 2.0 + dx, ny / 2.0 + dy, r)
    else:
        if cfg.cid == 4:
            r = 4.0
            cx = 12 + st.u() * (nx - 24)
            cy = 12 + st.u() * (ny - 24)
            chi = chi + 200.0 * _disc(nx, ny, cx, cy, r)
        nseeds = 30 if cfg.cid == 4 else 20
        ax, ay = 0.45 * nx - 8.0, 0.40 * ny - 8.0  # mask shrunk by 8 px
        for _ in range(nseeds):
            while True:
                cx, cy = st.u() * nx, st.u() * ny
                if cfg.cid == 4:
                    if 12 <= cx <= nx - 12 and 12 <= cy <= ny - 12:
                        break
                elif ((cx - nx / 2.0) / ax) ** 2 + ((cy - ny / 2.0) / ay) ** 2 <= 1.0:
                    break
            ang = np.pi * st.u()
            chi = np.where(_ellipse(nx, ny, cx, cy, 4.5, 0.8, ang), 180.0, chi)  # value SET to 180
    return chi


def generate(cid, nslices=None, first_slice=0, want_truth=False):
    """Inputs of config `cid` (0..4, 5 = north-star stack) as float32 arrays.

    nslices / first_slice select a contiguous subset of the stack's slices (all coils of each).
    Returns dict(cfg, field [batch][ny][nx], mask [batch][ny][nx], chi_true (optional, [nslices][ny][nx])).
    Batch index = slice*ncoils + coil (BASELINE.json configs[3]).
    """
    cfg = CONFIGS[cid]
    ns = cfg.nslices if nslices is None else int(nslices)
    nx, ny, nc = cfg.nx, cfg.ny, cfg.ncoils
    field = np.empty((ns * nc, ny, nx), np.float32)
    mask = np.empty((ns * nc, ny, nx), np.float32)
    truth = np.empty((ns, ny, nx), np.float64) if want_truth else None
    m = _mask(cfg, nx, ny)
    for i in range(ns):
        s = first_slice + i
        chi = _phantom(cfg, s, nx, ny)
        phi = simulate_field(chi, cfg.b0_dir)
        amp = float(np.max(np.abs(phi)))
        if want_truth:
            truth[i] = chi
        for c in range(nc):
            if nc == 1:
                sig = 0.01 * amp
            else:  # per coil sigma_c ~ U[0.005, 0.02] * max|phi|
                sig = (0.005 + 0.015 * float(uniform01(stream_key(cfg.cid, s, c, _COILSIG), 1)[0])) * amp
            noise = normal01(stream_key(cfg.cid, s, c, _NOISE), nx * ny).reshape(ny, nx)
            field[i * nc + c] = (phi + sig * noise).astype(np.float32)
            mask[i * nc + c] = m
    return {"cfg": cfg, "field": field, "mask": mask, "chi_true": truth}


def random_case(nx, ny, batch, seed, with_mask=True, with_weight=False):
    """Small unstructured test inputs: smooth-ish random field, random disc mask, optional weights in [0.2,1]."""
    out = {}
    f = np.empty((batch, ny, nx), np.float32)
    m = np.ones((batch, ny, nx), np.float32)
    w = np.ones((batch, ny, nx), np.float32) if with_weight else None
    for b in range(batch):
        f[b] = (10.0 * normal01(stream_key(100 + seed, b, 0, _NOISE), nx * ny)).reshape(ny, nx)
        if with_mask:
            u = uniform01(stream_key(100 + seed, b, 0, _SHAPES), 3)
            m[b] = _disc(nx, ny, nx * (0.4 + 0.2 * u[0]), ny * (0.4 + 0.2 * u[1]), 0.3 * min(nx, ny) * (1 + u[2]))
        if with_weight:
            w[b] = (0.2 + 0.8 * uniform01(stream_key(100 + seed, b, 0, _BG), nx * ny)).reshape(ny, nx)
    out.update(field=f, mask=m, weight=w)
    return out


_ECHO_PHASE, _ECHO_NOISE = 5, 6


def echo_pair(cid, nslices=None, first_slice=0, phase_span=2.5, noise=0.01):
    """The two complex volumes of the acquisition (without / with the echo shift T_shift) whose phase
    difference encodes generate()'s field map -- inputs of the pre-processing step (flow step (1)).

    Per batch entry (slice*ncoils + coil): magnitude A = tissue (1 inside the mask, 0.2 outside) x a smooth coil
    sensitivity (a Gaussian bump centred on a circle around the slice, one position per coil) ; a smooth receive phase
    theta0 ; s0 = A exp(i theta0) + n0, s1 = A exp(i (theta0 + pscale field)) + n1 with complex Gaussian noise of standard
    deviation `noise`, pscale = phase_span / max|field| so that the phase difference stays inside (-pi, pi) (the reason
    T_shift is small).  Returns dict(cfg, s0, s1 (complex64 [batch][ny][nx]), fscale = 1/pscale, field, mask)."""
    d = generate(cid, nslices, first_slice)
    cfg, f, m = d["cfg"], d["field"].astype(np.float64), d["mask"]
    batch, ny, nx = f.shape
    nc = cfg.ncoils
    pscale = phase_span / float(np.max(np.abs(f)))
    yy, xx = np.mgrid[0:ny, 0:nx]
    s0 = np.empty((batch, ny, nx), np.complex64)
    s1 = np.empty((batch, ny, nx), np.complex64)
    for b in range(batch):
        s, c = first_slice + b // nc, b % nc
        ang = 2.0 * np.pi * (c + 0.25) / nc
        cx, cy = nx * (0.5 + 0.45 * np.cos(ang)), ny * (0.5 + 0.45 * np.sin(ang))
        sens = 0.15 + np.exp(-((xx - cx) ** 2 + (yy - cy) ** 2) / (2.0 * (0.45 * min(nx, ny)) ** 2))
        A = sens * np.where(m[b] > 0, 1.0, 0.2)
        theta0 = 2.0 * np.pi * 5.0 * background(nx, ny, stream_key(cfg.cid, s, c, _ECHO_PHASE))
        g = normal01(stream_key(cfg.cid, s, c, _ECHO_NOISE), 4 * nx * ny).reshape(4, ny, nx)
        s0[b] = (A * np.exp(1j * theta0) + noise * (g[0] + 1j * g[1])).astype(np.complex64)
        s1[b] = (A * np.exp(1j * (theta0 + pscale * f[b])) + noise * (g[2] + 1j * g[3])).astype(np.complex64)
    return {"cfg": cfg, "s0": s0, "s1": s1, "fscale": 1.0 / pscale, "field": d["field"], "mask": m}


_VOL = 7


def volume_case(nx, ny, nz, nvol=1, seed=0, b0_axis=2, noise=0.01):
    """Inputs of the true 3-D variant (NEXT-2): per volume a phantom of a few ellipsoids (susceptibility sources) and a
    thin needle along a random direction in a zero background, the field it induces through the 3-D dipole kernel
    (numpy.fft, float64: the measurement is simulated, nothing is solved), Gaussian noise of `noise` x max|field|, and an
    ellipsoidal mask.  Returns dict(field, mask: float32 [nvol][nz][ny][nx], chi_true float64)."""
    zz, yy, xx = np.mgrid[0:nz, 0:ny, 0:nx]
    kz, ky, kx = np.meshgrid(np.fft.fftfreq(nz), np.fft.fftfreq(ny), np.fft.fftfreq(nx), indexing="ij")
    k2 = kx * kx + ky * ky + kz * kz
    kb = (kx, ky, kz)[b0_axis]
    D = 1.0 / 3.0 - kb * kb / np.where(k2 == 0, 1.0, k2)
    D[0, 0, 0] = 0.0
    field = np.empty((nvol, nz, ny, nx), np.float32)
    mask = np.empty((nvol, nz, ny, nx), np.float32)
    truth = np.empty((nvol, nz, ny, nx), np.float64)
    for v in range(nvol):
        u = uniform01(stream_key(900 + seed, v, 0, _VOL), 64)
        chi = np.zeros((nz, ny, nx))
        for e in range(3):
            c = (nx * (0.3 + 0.4 * u[6 * e]), ny * (0.3 + 0.4 * u[6 * e + 1]), nz * (0.3 + 0.4 * u[6 * e + 2]))
            r = [max(1.0, 0.08 * n * (0.5 + u[6 * e + 3 + a])) for a, n in enumerate((nx, ny, nz))]
            chi[((xx - c[0]) / r[0]) ** 2 + ((yy - c[1]) / r[1]) ** 2 + ((zz - c[2]) / r[2]) ** 2 <= 1.0] += 1.0 + u[40 + e]
        d = np.array([u[50] - 0.5, u[51] - 0.5, u[52] - 0.5])
        d /= max(np.linalg.norm(d), 1e-6)
        rel = np.stack([xx - nx / 2.0, yy - ny / 2.0, zz - nz / 2.0])
        along = (rel * d[:, None, None, None]).sum(0)
        perp2 = (rel ** 2).sum(0) - along ** 2
        chi[(perp2 <= 1.5) & (np.abs(along) <= 0.3 * min(nx, ny, nz))] += 5.0
        phi = np.real(np.fft.ifftn(D * np.fft.fftn(chi)))
        g = normal01(stream_key(900 + seed, v, 1, _VOL), nx * ny * nz).reshape(nz, ny, nx)
        field[v] = (phi + noise * np.abs(phi).max() * g).astype(np.float32)
        mask[v] = (((xx - nx / 2.0) / (0.46 * nx)) ** 2 + ((yy - ny / 2.0) / (0.46 * ny)) ** 2 + ((zz - nz / 2.0) / (0.48 * nz)) ** 2 <= 1.0)
        truth[v] = chi
    return {"field": field, "mask": mask, "chi_true": truth}


def echo_volumes(nx, ny, nz, ncoils, seed=0, b0_axis=2, phase_span=2.5, noise=0.01):
    """The two complex acquisitions of ONE object seen by `ncoils` coils, as volumes [ncoils][nz][ny][nx]:
    volume_case's phantom field (one volume, the same for every coil), per coil a Gaussian sensitivity around a point on a
    circle in the x-y plane times the tissue magnitude (1 inside the ellipsoidal mask, 0.2 outside), a smooth receive
    phase, the second echo rotated by pscale x field, complex Gaussian noise.  Returns dict(s0, s1, fscale, field, mask)."""
    case = volume_case(nx, ny, nz, nvol=1, seed=seed, b0_axis=b0_axis, noise=0.0)
    f, m = case["field"][0].astype(np.float64), case["mask"][0]
    pscale = phase_span / float(np.abs(f).max())
    zz, yy, xx = np.mgrid[0:nz, 0:ny, 0:nx]
    s0 = np.empty((ncoils, nz, ny, nx), np.complex64)
    s1 = np.empty((ncoils, nz, ny, nx), np.complex64)
    for c in range(ncoils):
        ang = 2.0 * np.pi * (c + 0.25) / ncoils
        cx, cy = nx * (0.5 + 0.45 * np.cos(ang)), ny * (0.5 + 0.45 * np.sin(ang))
        A = (0.15 + np.exp(-((xx - cx) ** 2 + (yy - cy) ** 2) / (2.0 * (0.45 * min(nx, ny)) ** 2))) * np.where(m > 0, 1.0, 0.2)
        u = uniform01(stream_key(950 + seed, c, 0, _ECHO_PHASE), 6)
        theta0 = 2.0 * np.pi * (u[0] * xx / nx + u[1] * yy / ny + u[2] * zz / nz) + 0.5 * np.sin(2.0 * np.pi * (xx / nx + u[3]))
        g = normal01(stream_key(950 + seed, c, 0, _ECHO_NOISE), 4 * nx * ny * nz).reshape(4, nz, ny, nx)
        s0[c] = (A * np.exp(1j * theta0) + noise * (g[0] + 1j * g[1])).astype(np.complex64)
        s1[c] = (A * np.exp(1j * (theta0 + pscale * f)) + noise * (g[2] + 1j * g[3])).astype(np.complex64)
    return {"s0": s0, "s1": s1, "fscale": 1.0 / pscale, "field": case["field"][0], "mask": m}
