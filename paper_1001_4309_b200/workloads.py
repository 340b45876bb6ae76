"""Seeded synthetic inputs and the five BASELINE.json configs.

This module serves BOTH the CUDA path's tests/bench and the oracle's tests.  It holds none of
the Shifted-Fresnel arithmetic (no chirps, no scaled DFT): only the workload descriptions and
a hologram *generator*, which propagates a synthetic object with a float64 angular-spectrum
transfer function — a different method, used only to make frames that look like the paper's
in-line Gabor holograms (1 024 x 1 024, 8-bit, 4.65 um pitch, 632.8 nm).
The paper's own CCD frames (USAF target, mosquito, fly) are not available; these stand in.

Pure NumPy; imports neither the oracle nor the CUDA binding.  Recipe: DESIGN.md §4.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

LAMBDA = 632.8e-9      # He-Ne
PITCH = 4.65e-6        # CCD pixel pitch

IN_U8 = 0              # matches SFD_U8 in include/sfd.h
IN_F32 = 1             # matches SFD_F32


# --------------------------------------------------------------------------------------
# hologram generator G(N, z_obj, seed)
# --------------------------------------------------------------------------------------
def _object_transmittance(N2, N, pitch, rng):
    """Unit-transmittance plane (N2 x N2 samples) with 20 opaque disks and 3 groups of 3
    opaque bars placed inside the central N x N window.  Draw order (fixed, so that a seed
    names one object): for each disk (cx, cy, r); then for each bar group
    (w, orientation, cx, cy)."""
    t = np.ones((N2, N2), dtype=np.float64)
    lo = (N2 - N) // 2
    span = N * pitch

    def to_px(c):                      # window coordinate in metres -> sample index
        return lo + c / pitch

    yy, xx = np.mgrid[0:N2, 0:N2]
    for _ in range(20):
        cx = rng.uniform(0.0, span)
        cy = rng.uniform(0.0, span)
        r = rng.uniform(5e-6, 40e-6)
        px, py, pr = to_px(cx), to_px(cy), r / pitch
        x0, x1 = int(max(px - pr - 1, 0)), int(min(px + pr + 2, N2))
        y0, y1 = int(max(py - pr - 1, 0)), int(min(py + pr + 2, N2))
        sub = (xx[y0:y1, x0:x1] - px) ** 2 + (yy[y0:y1, x0:x1] - py) ** 2 <= pr * pr
        t[y0:y1, x0:x1][sub] = 0.0
    for _ in range(3):
        w = rng.uniform(10e-6, 60e-6)
        horizontal = bool(rng.integers(0, 2))
        cx = rng.uniform(0.0, span)
        cy = rng.uniform(0.0, span)
        length = 5.0 * w
        for b in range(3):             # three bars, period 2w, centred on (cx, cy)
            off = (b - 1) * 2.0 * w
            if horizontal:             # long side along x, bars stacked in y
                bx0, bx1 = cx - length / 2, cx + length / 2
                by0, by1 = cy + off - w / 2, cy + off + w / 2
            else:
                bx0, bx1 = cx + off - w / 2, cx + off + w / 2
                by0, by1 = cy - length / 2, cy + length / 2
            ix0 = int(np.clip(np.ceil(to_px(bx0)), 0, N2))
            ix1 = int(np.clip(np.floor(to_px(bx1)) + 1, 0, N2))
            iy0 = int(np.clip(np.ceil(to_px(by0)), 0, N2))
            iy1 = int(np.clip(np.floor(to_px(by1)) + 1, 0, N2))
            t[iy0:iy1, ix0:ix1] = 0.0
    return t


def gabor_hologram(N, z_obj, seed, lam=LAMBDA, pitch=PITCH):
    """G(N, z_obj, seed): uint8 in-line Gabor hologram, N x N.

    Object of ``_object_transmittance`` on a 2N x 2N grid; scattered field
    ``u = IFFT2[FFT2[t - 1] exp(i 2 pi z sqrt(1/lambda^2 - fx^2 - fy^2))]`` in float64 with
    evanescent components and (band-limited angular spectrum) ``|f| > 1/(lambda
    sqrt((2 df z)^2 + 1))`` per axis zeroed; ``I = |1 + u|^2`` cropped to the central N x N;
    ``uint8 = rint(255 I / max I)``."""
    rng = np.random.default_rng(seed)
    N2 = 2 * N
    t = _object_transmittance(N2, N, pitch, rng)
    f = np.fft.fftfreq(N2, d=pitch)
    fx2 = (f * f)[None, :]
    fy2 = (f * f)[:, None]
    arg = 1.0 / (lam * lam) - fx2 - fy2
    df = 1.0 / (N2 * pitch)
    flim = 1.0 / (lam * np.sqrt((2.0 * df * z_obj) ** 2 + 1.0))
    keep = (arg > 0.0) & (np.abs(f)[None, :] <= flim) & (np.abs(f)[:, None] <= flim)
    kz = np.sqrt(np.where(arg > 0.0, arg, 0.0))
    ph = z_obj * kz
    ph -= np.floor(ph)
    H = np.where(keep, np.exp(2j * np.pi * ph), 0.0)
    u = np.fft.ifft2(np.fft.fft2(t - 1.0) * H)
    lo = (N2 - N) // 2
    I = np.abs(1.0 + u[lo:lo + N, lo:lo + N]) ** 2
    return np.rint(255.0 * I / I.max()).astype(np.uint8)


# --------------------------------------------------------------------------------------
# workloads = BASELINE.json configs
# --------------------------------------------------------------------------------------
@dataclass
class Workload:
    name: str
    N: int
    lam: float
    p1: np.ndarray          # hologram pitch per view [m]
    p2: np.ndarray          # reconstruction pitch per view [m]
    z: np.ndarray           # depth per view [m]
    Ox: np.ndarray          # x shift per view [m]
    Oy: np.ndarray          # y shift per view [m]
    in_dtype: int           # IN_U8 | IN_F32
    z_obj: float = 0.0      # object distance of the generated hologram (0: not generated)
    seed: int = 0
    n_frames: int = 1
    extra: dict = field(default_factory=dict)

    @property
    def n_views(self):
        return len(self.z)

    def hologram(self, frame=0):
        """Hologram of frame ``frame`` (host array, [N][N], uint8 or float32)."""
        if self.in_dtype == IN_F32:
            return np.random.default_rng(self.seed + frame).random((self.N, self.N),
                                                                   dtype=np.float32)
        return gabor_hologram(self.N, self.z_obj, self.seed + frame, self.lam, PITCH)


def _arr(*v):
    return np.asarray(v, dtype=np.float64)


_VIEWS4 = dict(
    z=_arr(0.08, 0.06, 0.08, 0.08),
    p2=_arr(4.65e-6, 4.65e-6, 1.5e-6, 1.0e-6),
    Ox=_arr(0.0, 0.0, 0.5e-3, -0.6e-3),
    Oy=_arr(0.0, 0.0, 0.2e-3, -0.4e-3),
)


def config(i, n_frames=None):
    """The i-th entry of BASELINE.json ``configs`` (0 Tiny ... 4 Scale stress)."""
    if i == 0:
        return Workload("tiny", 64, LAMBDA, _arr(PITCH), _arr(PITCH), _arr(0.05), _arr(0.0),
                        _arr(0.0), IN_F32, seed=0)
    if i == 1:
        return Workload("single_view_1024", 1024, LAMBDA, _arr(PITCH), _arr(2.0e-6), _arr(0.08),
                        _arr(0.4e-3), _arr(-0.3e-3), IN_U8, z_obj=0.08, seed=1)
    if i == 2:
        return Workload("paper_4view_1024", 1024, LAMBDA, np.full(4, PITCH), _VIEWS4["p2"],
                        _VIEWS4["z"], _VIEWS4["Ox"], _VIEWS4["Oy"], IN_U8, z_obj=0.08, seed=1)
    if i == 3:
        return Workload("realtime_stream_1024", 1024, LAMBDA, np.full(4, PITCH), _VIEWS4["p2"],
                        _VIEWS4["z"], _VIEWS4["Ox"], _VIEWS4["Oy"], IN_U8, z_obj=0.08,
                        seed=1000, n_frames=256 if n_frames is None else n_frames)
    if i == 4:
        V = 16
        rng = np.random.default_rng(40)
        O = rng.uniform(-1e-3, 1e-3, size=(V, 2))
        p2 = _arr(0.5e-6, 1.0e-6, 2.0e-6, 4.65e-6)[np.arange(V) % 4]
        z = 0.02 + np.arange(V) * (0.10 / 15.0)
        return Workload("scale_stress_2048", 2048, LAMBDA, np.full(V, PITCH), p2, z,
                        O[:, 0].copy(), O[:, 1].copy(), IN_U8, z_obj=0.10, seed=4)
    raise ValueError("config index must be 0..4")


def small_multiview(N=256, V=3, seed=7):
    """Parity-test case between Tiny and the 1 024^2 configs: uint8 Gabor hologram, V views
    with mixed signs of z, pitches and shifts; spans several tiles of every kernel."""
    rng = np.random.default_rng(seed)
    z = rng.uniform(0.03, 0.10, V) * np.where(np.arange(V) % 3 == 2, -1.0, 1.0)
    p2 = rng.uniform(0.8e-6, 4.65e-6, V)
    O = rng.uniform(-0.3e-3, 0.3e-3, size=(V, 2))
    return Workload(f"small_{N}x{V}", N, LAMBDA, np.full(V, PITCH), p2, z, O[:, 0].copy(),
                    O[:, 1].copy(), IN_U8, z_obj=0.05, seed=seed)


def depth_stack(N=1024, V=16, z0=0.04, z1=0.12, p2=PITCH, seed=1, z_obj=0.08):
    """Row f2: one Gabor hologram (object at ``z_obj``), V views that differ only in z (linear sweep
    z0..z1), no shift — the focus sweep a user of the microscope runs to find the object plane."""
    z = np.linspace(z0, z1, V)
    zero = np.zeros(V)
    return Workload(f"depth_stack_{N}x{V}", N, LAMBDA, np.full(V, PITCH), np.full(V, p2), z, zero,
                    zero.copy(), IN_U8, z_obj=z_obj, seed=seed)


# --------------------------------------------------------------------------------------
# host-side sharding for --gpus N (views and frames are independent: no collective)
# --------------------------------------------------------------------------------------
def shard_range(n_units, rank, world):
    """Contiguous block partition of ``n_units`` independent units (frames or views) over
    ``world`` ranks; the first ``n_units % world`` ranks take one extra.  Returns
    ``(start, stop)``."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad rank/world")
    base, rem = divmod(n_units, world)
    start = rank * base + min(rank, rem)
    return start, start + base + (1 if rank < rem else 0)
