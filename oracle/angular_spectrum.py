"""Float64 CPU oracle for angular-spectrum propagation.

TEST INFRASTRUCTURE ONLY.  Nothing in the product path (``paper_1001_4309_b200``) may import, call
or link this module; only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s CPU legs use
it.  It shares no code with the CUDA path nor with the hologram generator of ``workloads.py``.

What it computes.  Digital holographic microscopy observes "both the amplitude and phase of a
specimen"; the second propagator of the field, next to the paper's Shifted-Fresnel
transform, is the angular-spectrum method that SURVEY.md §8(d) uses to define the synthetic
holograms:

    u(z) = IFFT2[ FFT2[u0] * H ],   H(fx, fy) = exp(i 2 pi z sqrt(1/lambda^2 - fx^2 - fy^2))

on the periodic ``Ny x Nx`` grid of pitch ``(px, py)`` (no padding: the method is a circular
convolution), with ``fx = kx / (Nx px)`` for ``kx`` in FFT order (``kx >= Nx/2`` are negative
frequencies), evanescent components (``fx^2 + fy^2 >= 1/lambda^2``) set to zero and, optionally,
the band limit of SURVEY.md §8(d): per axis ``|f| <= 1/(lambda sqrt((2 df z)^2 + 1))``,
``df = 1/(N p)``.  Unlike the Fresnel kernel the transfer function does not factorise into an x- and
a y-part.  Outputs: the complex field, its intensity ``|u|^2``, amplitude ``|u|`` and phase
``arg u`` in ``(-pi, pi]``.

Readings: exact (non-paraxial) transfer function; ``z`` of either sign and
``z = 0`` (identity on the propagating band) are valid; the phase is formed in cycles, ``z sqrt(.)``,
and reduced modulo 1 before the exponential.

Pinned by ``tests/test_oracle_asm_pins.py``: plane waves are eigenfunctions with the analytic
eigenvalue, the direct O(N^4) double sum on tiny grids, +z then -z, the paraxial Gaussian beam,
agreement with the Fresnel oracle where both hold, unitarity.  Nothing here is "parity unpinned".
"""
from __future__ import annotations

import numpy as np
import scipy.fft as _fft

from .shifted_fresnel import FFT_WORKERS


def _pair(v):
    if np.ndim(v) == 0:
        return float(v), float(v)
    x, y = v
    return float(x), float(y)


def frequencies(N, pitch):
    """Spatial frequencies of the N FFT bins, cycles per metre: ``k/(N p)`` for ``k < N/2``,
    ``(k - N)/(N p)`` from ``N/2`` on."""
    k = np.arange(N, dtype=np.float64)
    k = np.where(k < N / 2.0, k, k - N)
    return k / (N * pitch)


def band_limit_frequency(N, pitch, lam, z):
    """``1 / (lambda sqrt((2 df z)^2 + 1))`` with ``df = 1/(N p)`` - beyond it the
    sampled transfer function is aliased."""
    df = 1.0 / (N * pitch)
    return 1.0 / (lam * np.sqrt((2.0 * df * z) ** 2 + 1.0))


def transfer_function(Ny, Nx, lam, z, pitch, band_limit=False):
    """``H[ky, kx] = exp(i 2 pi z sqrt(1/lambda^2 - fx^2 - fy^2))`` where the root is real and
    positive, 0 elsewhere (evanescent cut); with ``band_limit`` also 0 beyond the per-axis limit."""
    if not (lam > 0.0) or not np.isfinite(z):
        raise ValueError("lambda must be positive and z finite")
    px, py = _pair(pitch)
    fx = frequencies(Nx, px)[None, :]
    fy = frequencies(Ny, py)[:, None]
    w2 = 1.0 / (lam * lam) - fx * fx - fy * fy
    keep = w2 > 0.0
    if band_limit:
        keep = keep & (np.abs(fx) <= band_limit_frequency(Nx, px, lam, z))
        keep = keep & (np.abs(fy) <= band_limit_frequency(Ny, py, lam, z))
    cycles = z * np.sqrt(np.where(w2 > 0.0, w2, 0.0))
    cycles = cycles - np.rint(cycles)
    return np.where(keep, np.exp(2j * np.pi * cycles), 0.0)


def propagate(u0, lam, z, pitch, band_limit=False):
    """``IFFT2[FFT2[u0] * H]``, true inverse (1/(Nx Ny) included)."""
    u0 = np.asarray(u0)
    if u0.ndim != 2:
        raise ValueError("u0 must be a 2-D array [n][m]")
    Ny, Nx = u0.shape
    H = transfer_function(Ny, Nx, lam, z, pitch, band_limit)
    A = _fft.fft2(u0.astype(np.complex128), workers=FFT_WORKERS)
    return _fft.ifft2(A * H, workers=FFT_WORKERS)


def propagate_planes(u0, lam, zs, pitch, band_limit=False):
    """All planes of one input, arguments as in ``sfd_asm_plan_create``.  Returns
    ``(field[P,Ny,Nx] complex128, intensity, phase)``."""
    f = np.stack([propagate(u0, lam, float(z), pitch, band_limit) for z in zs])
    return f, intensity(f), phase(f)


def intensity(u):
    u = np.asarray(u)
    return u.real * u.real + u.imag * u.imag


def amplitude(u):
    return np.abs(np.asarray(u))


def phase(u):
    """``arg u`` in ``(-pi, pi]`` (``atan2(im, re)``); 0 where ``u = 0``."""
    u = np.asarray(u)
    return np.arctan2(u.imag, u.real)
