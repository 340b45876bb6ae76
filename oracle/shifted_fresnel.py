"""Float64 CPU oracle for Shifted-Fresnel diffraction (arxiv/paper_1001_4309).

TEST INFRASTRUCTURE ONLY.  Nothing in the product path (``paper_1001_4309_b200``) may
import, call or link this module; only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` use it.  It shares no code,
table generator or helper with the CUDA path and never imports it.

What it computes (§2.1): from an ``N_y x N_x`` hologram ``u0`` sampled at
pitch ``(p_x0, p_y0)``, the complex field ``u1`` on an ``N_y x N_x`` window of arbitrary
pitch ``(p_x1, p_y1)`` shifted off axis by ``(O_x1, O_y1)`` at distance ``z``, and its
intensity ``I = |u1|^2`` (Eq. 5).

Three forms, slowest and plainest first:

* ``direct_sum``          form D — the discretised Fresnel double sum that Eq.(1) L50 expands
                          (O(N^4); tiny N only).  This is the *definition*.
* ``separable_matrices``  form M — the same sum with the separable kernel written as two dense
                          matrices (O(N^3)); the definition at full size.
* ``bluestein_fft``       form B — the paper's own algorithm, Eq.(1)-(4) and steps (ii)-(x)
                          (L85-95), written step by step, unpruned, with a library FFT.

Readings of the paper used here (DESIGN.md §3 lists all of them with line numbers):

* Arrays are ``[n][m]`` row-major; ``m`` <-> x <-> column, ``n`` <-> y <-> row (reading 4).
* Indices run over ``[0, N)``; physical coordinates are centred:
  ``x0[m0] = (m0 - N_x/2) p_x0 + O_x0``, ``x1[m1] = (m1 - N_x/2) p_x1 + O_x1`` with every
  ``O`` in metres (readings 1, 2).  With these, Eq.(2)-(3)'s ``(-N_x/2 + O)`` factors are
  recovered with ``O`` counted in pixels.
* ``N_x, N_y`` are the un-padded sizes (reading 3); the doubling to ``2N`` (L86, L115) is an
  implementation device of form B only.
* FFT^-1 is the true inverse (1/M^2 included) (reading 8).
* All of C1 (Eq. 2) is kept and the sum carries the area element ``p_x0 p_y0`` (reading 9):
  ``c0 = p_x0 p_y0 exp(ikz) / (i lambda z)``, ``k = 2 pi / lambda`` (reading 10).
* ``z < 0`` is allowed (reading 11); ``z = 0`` is an error.

Every phase is formed in cycles (phase / 2 pi) in float64 and reduced modulo 1 before the
complex exponential, so that ``exp`` never sees an argument larger than pi.

All three forms are pinned by ``tests/test_oracle_pins.py`` (closed forms, the textbook
single-FFT Fresnel transform, brute force, symmetries).  Nothing here is "parity unpinned".
"""
from __future__ import annotations

import os

import numpy as np
import scipy.fft as _fft

#: threads handed to scipy.fft in form B (the timed CPU baseline reports this number)
FFT_WORKERS = os.cpu_count() or 1


# --------------------------------------------------------------------------------------
# small helpers
# --------------------------------------------------------------------------------------
def _cis_cycles(c):
    """exp(2 pi i c) for a phase ``c`` given in cycles; ``c`` is reduced mod 1 first."""
    c = np.asarray(c, dtype=np.float64)
    c = c - np.rint(c)
    return np.exp(2j * np.pi * c)


def _pair(v):
    """Scalar -> (v, v); pair -> (x, y)."""
    if np.ndim(v) == 0:
        return float(v), float(v)
    x, y = v
    return float(x), float(y)


def _check(u0, lam, z):
    u0 = np.asarray(u0)
    if u0.ndim != 2:
        raise ValueError("u0 must be a 2-D array [n][m]")
    if not (lam > 0.0):
        raise ValueError("lambda must be positive")
    if z == 0.0 or not np.isfinite(z):
        raise ValueError("z must be finite and non-zero")
    return u0.astype(np.complex128)


def coordinates(N, pitch, offset):
    """Physical sample positions of a centred window (PAPER.md L67 with reading 1):
    ``x[m] = (m - N/2) pitch + offset`` for ``m`` in ``[0, N)``."""
    return (np.arange(N, dtype=np.float64) - N / 2.0) * pitch + offset


def c0_factor(lam, z, p0x, p0y):
    """Constant part of C1, Eq.(2), times the area element (reading 9):
    ``p_x0 p_y0 exp(i k z) / (i lambda z)``; ``exp(ikz) = exp(2 pi i frac(z/lambda))``."""
    return p0x * p0y * _cis_cycles(z / lam) / (1j * lam * z)


def intensity(u1):
    """Eq.(5): ``I = |u1|^2``."""
    u1 = np.asarray(u1)
    return u1.real * u1.real + u1.imag * u1.imag


def focus_moments(I):
    """Row f2 (depth stacks, PAPER.md L33 / Fig. 1): per view the first two moments of the intensity
    of Eq.(5) over the N x N window, ``(sum I, sum I^2)``, in float64.  ``I`` is ``[V, N, N]``.
    The paper defines no focus measure; ``normalised_variance`` is the usual one built on them."""
    I = np.asarray(I, dtype=np.float64)
    return np.stack([I.sum(axis=(-2, -1)), (I * I).sum(axis=(-2, -1))], axis=-1)


def normalised_variance(moments, n_pixels):
    """``var(I) / mean(I)^2 = P sum I^2 / (sum I)^2 - 1`` from ``focus_moments`` (P pixels)."""
    m = np.asarray(moments, dtype=np.float64)
    return n_pixels * m[..., 1] / (m[..., 0] * m[..., 0]) - 1.0


def quantise_u8(I):
    """Real-time mode output (step xi L95, reading 15): per image,
    ``I8 = round_half_even(255 I / max I)`` as uint8; an all-zero image maps to zeros."""
    I = np.asarray(I, dtype=np.float64)
    mx = I.max() if I.size else 0.0
    if not (mx > 0.0):
        return np.zeros(I.shape, dtype=np.uint8)
    return np.rint(255.0 * I / mx).astype(np.uint8)


def input_scale(u0):
    """Hologram samples as the method sees them (reading 12): uint8 -> value/255 in [0,1];
    floating input is used as is."""
    u0 = np.asarray(u0)
    if u0.dtype == np.uint8:
        return u0.astype(np.float64) / 255.0
    return u0.astype(np.float64)


def crop_window(frame, Ny, Nx, row0=None, col0=None):
    """the 1 360 x 1 024 CCD frame is "resized" to 1 024 x 1 024 before the transform.
    Reading 13: a crop - the only resize that keeps the 4.65 um sample pitch the paper
    goes on to use (L107: field of view 4.8 mm = 1 024 x 4.65 um).  Returns the ``Ny x Nx`` window
    whose first sample is ``frame[row0][col0]``; ``None`` centres the window (168 columns are cut on
    either side of a 1 360-wide frame).  A centred window keeps the optical axis at index N/2, so no
    offset O_0 is needed; a window shifted by (dr, dc) samples off centre is the hologram window of
    Eq.(2)-(3) with ``O_0 = (dc p_x0, dr p_y0)``."""
    frame = np.asarray(frame)
    rows, cols = frame.shape
    row0 = (rows - Ny) // 2 if row0 is None else int(row0)
    col0 = (cols - Nx) // 2 if col0 is None else int(col0)
    if row0 < 0 or col0 < 0 or row0 + Ny > rows or col0 + Nx > cols:
        raise ValueError("window exceeds the frame")
    return frame[row0:row0 + Ny, col0:col0 + Nx]


# --------------------------------------------------------------------------------------
# form D: the definition, O(N^4)
# --------------------------------------------------------------------------------------
def direct_sum(u0, lam, z, p0, p1, O1=(0.0, 0.0), O0=(0.0, 0.0)):
    """Form D.  The double sum of Eq.(1) L50 before any algebra:

        u1[n1,m1] = c0 * sum_{n0,m0} u0[n0,m0]
                         * exp( i pi [ (x1[m1]-x0[m0])^2 + (y1[n1]-y0[n0])^2 ] / (lambda z) )

    ``p0``/``p1`` are the hologram / reconstruction pitches (scalar or ``(x, y)``), ``O1`` /
    ``O0`` the window shifts ``(x, y)`` in metres.  Use for N <= 64."""
    u0 = _check(u0, lam, z)
    Ny, Nx = u0.shape
    p0x, p0y = _pair(p0)
    p1x, p1y = _pair(p1)
    x0 = coordinates(Nx, p0x, O0[0])
    y0 = coordinates(Ny, p0y, O0[1])
    x1 = coordinates(Nx, p1x, O1[0])
    y1 = coordinates(Ny, p1y, O1[1])
    u1 = np.empty((Ny, Nx), dtype=np.complex128)
    inv = 1.0 / (2.0 * lam * z)          # pi r^2 / (lambda z) in cycles = r^2 / (2 lambda z)
    for n1 in range(Ny):
        dy2 = (y1[n1] - y0) ** 2                     # [n0]
        for m1 in range(Nx):
            dx2 = (x1[m1] - x0) ** 2                 # [m0]
            ph = (dy2[:, None] + dx2[None, :]) * inv
            u1[n1, m1] = np.sum(u0 * _cis_cycles(ph))
    return c0_factor(lam, z, p0x, p0y) * u1


# --------------------------------------------------------------------------------------
# form M: the definition with its separable kernel, O(N^3)
# --------------------------------------------------------------------------------------
def fresnel_matrix(N, lam, z, pitch0, pitch1, off0, off1):
    """``K[m1, m0] = exp(i pi (x1[m1] - x0[m0])^2 / (lambda z))``."""
    x0 = coordinates(N, pitch0, off0)
    x1 = coordinates(N, pitch1, off1)
    d = x1[:, None] - x0[None, :]
    return _cis_cycles(d * d / (2.0 * lam * z))


def separable_matrices(u0, lam, z, p0, p1, O1=(0.0, 0.0), O0=(0.0, 0.0)):
    """Form M.  exp(i pi[(dx)^2 + (dy)^2]/lambda z) factorises, so the sum of form D is
    ``u1 = c0 * K_y @ u0 @ K_x^T``."""
    u0 = _check(u0, lam, z)
    Ny, Nx = u0.shape
    p0x, p0y = _pair(p0)
    p1x, p1y = _pair(p1)
    Kx = fresnel_matrix(Nx, lam, z, p0x, p1x, O0[0], O1[0])
    Ky = fresnel_matrix(Ny, lam, z, p0y, p1y, O0[1], O1[1])
    return c0_factor(lam, z, p0x, p0y) * (Ky @ u0 @ Kx.T)


# --------------------------------------------------------------------------------------
# form B: the paper's algorithm, Eq.(1)-(4), steps (ii)-(x)
# --------------------------------------------------------------------------------------
def scale_factor(lam, z, pitch0, pitch1):
    """``S = p_0 p_1 / (lambda z)`` (L67)."""
    return pitch0 * pitch1 / (lam * z)


def pre_chirp(N, lam, z, pitch0, pitch1, off0, off1):
    """1-D factor of Eq.(3) L61-62 along one axis, index ``m0`` in ``[0, N)``:

        exp(i pi x0^2/(lambda z)) * exp(-i 2 pi m0 p_0 a1/(lambda z)) * exp(-i pi S m0^2)

    with ``a1 = x1[0] = -N/2 p_1 + O_1``.  ``p_0 a1/(lambda z) = S (-N/2 + O_1/p_1)`` is the
    paper's ``S_x(-N_x/2 + O_x1)`` with the shift in pixels."""
    m = np.arange(N, dtype=np.float64)
    x0 = coordinates(N, pitch0, off0)
    a1 = -N / 2.0 * pitch1 + off1
    S = scale_factor(lam, z, pitch0, pitch1)
    lz = lam * z
    return (_cis_cycles(x0 * x0 / (2.0 * lz))
            * _cis_cycles(-(m * pitch0 * a1) / lz)
            * _cis_cycles(-0.5 * S * m * m))


def post_chirp(N, lam, z, pitch0, pitch1, off0, off1):
    """1-D factor of C1, Eq.(2), along one axis, index ``m1`` in ``[0, N)``:

        exp(i pi x1^2/(lambda z)) * exp(-i (2 pi/(lambda z)) a0 x1) * exp(-i pi S m1^2)

    with ``a0 = x0[0] = (-N/2) p_0 + O_0`` — the paper's ``(-N_x/2 + O_x0) p_x0``."""
    m = np.arange(N, dtype=np.float64)
    x1 = coordinates(N, pitch1, off1)
    a0 = -N / 2.0 * pitch0 + off0
    S = scale_factor(lam, z, pitch0, pitch1)
    lz = lam * z
    return (_cis_cycles(x1 * x1 / (2.0 * lz))
            * _cis_cycles(-(a0 * x1) / lz)
            * _cis_cycles(-0.5 * S * m * m))


def chirp_kernel(N, M, S, free_sample=None):
    """Eq.(4) L64-65 along one axis on the padded, wrapped grid of length ``M >= 2N-1``:
    ``h1[j] = exp(i pi S d^2)``, lag ``d = j`` for ``j <= M/2`` and ``d = j - M`` above
    (steps v, L89; reading 5/6).  Lags ``|d| >= N`` never reach a kept output; for
    ``M = 2N`` that is the single sample ``j = N``, which ``free_sample`` may overwrite."""
    j = np.arange(M, dtype=np.float64)
    d = np.where(j <= M // 2, j, j - M)
    h1 = _cis_cycles(0.5 * S * d * d)
    if free_sample is not None:
        if M != 2 * N:
            raise ValueError("free_sample is defined for M = 2N only")
        h1[N] = free_sample
    return h1


def bluestein_fft(u0, lam, z, p0, p1, O1=(0.0, 0.0), O0=(0.0, 0.0), M=None, free_sample=None):
    """Form B.  PAPER.md Eq.(1) third line, L54, and the step list L85-95:

    (ii)  zero-pad to ``M x M`` (M = 2N, "doubled size", L86)
    (iii) multiply by the exponentials of Eq.(3)
    (iv)  forward 2-D FFT
    (v)   generate h, Eq.(4)          (vi) its 2-D FFT
    (vii) multiply the spectra        (viii) inverse 2-D FFT
    (ix)  keep ``[0,N)^2``            then C1 (Eq. 2); (x) ``|u1|^2`` is ``intensity()``.

    ``h`` is the product of an x- and a y-chirp, so its 2-D FFT is the outer product of two
    1-D FFTs; that identity is exact and is the only algebra used beyond the paper's steps."""
    u0 = _check(u0, lam, z)
    Ny, Nx = u0.shape
    p0x, p0y = _pair(p0)
    p1x, p1y = _pair(p1)
    Mx = 2 * Nx if M is None else int(M)
    My = 2 * Ny if M is None else int(M)
    if Mx < 2 * Nx - 1 or My < 2 * Ny - 1:
        raise ValueError("padded size must be at least 2N-1 (linear convolution, L86/L115)")
    w = FFT_WORKERS
    # (iii) Eq.(3)
    pre_x = pre_chirp(Nx, lam, z, p0x, p1x, O0[0], O1[0])
    pre_y = pre_chirp(Ny, lam, z, p0y, p1y, O0[1], O1[1])
    a = np.zeros((My, Mx), dtype=np.complex128)            # (ii)
    a[:Ny, :Nx] = u0 * pre_y[:, None] * pre_x[None, :]
    # (iv)
    A = _fft.fft2(a, workers=w)
    # (v), (vi) Eq.(4)
    Hx = _fft.fft(chirp_kernel(Nx, Mx, scale_factor(lam, z, p0x, p1x), free_sample))
    Hy = _fft.fft(chirp_kernel(Ny, My, scale_factor(lam, z, p0y, p1y), free_sample))
    # (vii), (viii)
    G = _fft.ifft2(A * (Hy[:, None] * Hx[None, :]), workers=w)
    # (ix) + Eq.(2)
    g = G[:Ny, :Nx]
    post_x = post_chirp(Nx, lam, z, p0x, p1x, O0[0], O1[0])
    post_y = post_chirp(Ny, lam, z, p0y, p1y, O0[1], O1[1])
    return c0_factor(lam, z, p0x, p0y) * (post_y[:, None] * post_x[None, :]) * g


# --------------------------------------------------------------------------------------
# multi-view front end with the north_star's argument list
# --------------------------------------------------------------------------------------
def reconstruct_views(hologram, lam, p1, p2, z, Ox, Oy, form="B"):
    """All views of one frame, arguments as in ``sfd_plan_create`` (north_star): per-view
    arrays ``p1`` (hologram pitch), ``p2`` (reconstruction pitch), ``z``, ``Ox``, ``Oy``.
    Returns ``(field[V,N,N] complex128, intensity[V,N,N] float64)``."""
    fn = {"B": bluestein_fft, "M": separable_matrices, "D": direct_sum}[form]
    u0 = input_scale(hologram)
    V = len(z)
    N = u0.shape[0]
    field = np.empty((V, N, u0.shape[1]), dtype=np.complex128)
    for v in range(V):
        field[v] = fn(u0, lam, float(z[v]), float(p1[v]), float(p2[v]),
                      O1=(float(Ox[v]), float(Oy[v])))
    return field, intensity(field)
