"""Pins of the angular-spectrum oracle (oracle/angular_spectrum.py) against what
the mathematics fixes: eigenfunctions with typed-out eigenvalues, the direct double sum on tiny grids,
inverse propagation, the paraxial Gaussian beam, the Fresnel oracle where both hold, unitarity."""
import cmath
import math

import numpy as np
import pytest

from oracle import angular_spectrum as A
from oracle import shifted_fresnel as O

LAM, PITCH = 632.8e-9, 4.65e-6


def _plane_wave(Ny, Nx, ky, kx):
    n, m = np.mgrid[0:Ny, 0:Nx]
    return np.exp(2j * np.pi * (kx * m / Nx + ky * n / Ny))


@pytest.mark.parametrize("Ny,Nx,ky,kx,px,py,z", [
    (16, 16, 0, 0, PITCH, PITCH, 0.05),         # on axis: eigenvalue exp(i k z)
    (16, 16, 3, 5, PITCH, PITCH, 0.05),
    (16, 32, 13, 30, PITCH, PITCH, -0.02),      # bins above N/2 are negative frequencies; z < 0
    (32, 16, 2, 7, 3.0e-6, 5.0e-6, 0.011),      # rectangular grid, anisotropic pitch
])
def test_plane_waves_are_eigenfunctions_with_the_analytic_eigenvalue(Ny, Nx, ky, kx, px, py, z):
    """A sampled plane wave exp(2 pi i (fx x + fy y)) propagates to itself times
    exp(i 2 pi z sqrt(1/lambda^2 - fx^2 - fy^2)); the eigenvalue is typed out here with math/cmath."""
    u0 = _plane_wave(Ny, Nx, ky, kx)
    fx = (kx if kx < Nx / 2 else kx - Nx) / (Nx * px)
    fy = (ky if ky < Ny / 2 else ky - Ny) / (Ny * py)
    cyc = z * math.sqrt(1.0 / LAM ** 2 - fx ** 2 - fy ** 2)
    eig = cmath.exp(2j * math.pi * (cyc - round(cyc)))
    u = A.propagate(u0, LAM, z, (px, py))
    assert np.max(np.abs(u - eig * u0)) < 2e-9      # |d phase| = 2 pi * 1e5 cycles * 2^-53


def test_evanescent_components_are_cut():
    """Pitch 0.2 um: bins beyond 1/lambda are evanescent and must vanish; the ones inside propagate."""
    N, p = 32, 0.2e-6                               # f_max = 2.5e6 > 1/lambda = 1.58e6
    k_ev = 12                                       # f = 12/(32 * 0.2e-6) = 1.875e6 > 1/lambda
    k_ok = 8                                        # 1.25e6 < 1/lambda
    assert k_ev / (N * p) > 1 / LAM > k_ok / (N * p)
    u = A.propagate(_plane_wave(N, N, 0, k_ev) + _plane_wave(N, N, k_ok, 0), LAM, 3e-6, p)
    cyc = 3e-6 * math.sqrt(1 / LAM ** 2 - (k_ok / (N * p)) ** 2)
    want = cmath.exp(2j * math.pi * cyc) * _plane_wave(N, N, k_ok, 0)
    assert np.max(np.abs(u - want)) < 1e-12
    H = A.transfer_function(N, N, LAM, 3e-6, p)
    fx = A.frequencies(N, p)
    inside = (fx[None, :] ** 2 + fx[:, None] ** 2) < 1 / LAM ** 2
    assert np.all(np.abs(H[inside]) == pytest.approx(1.0)) and np.all(H[~inside] == 0)


def test_direct_double_sum_on_a_tiny_grid():
    """Brute force: u[n,m] = 1/(Nx Ny) sum_k H[k] exp(+2 pi i k.r) sum_j u0[j] exp(-2 pi i k.j), plain loops,
    rectangular grid, anisotropic pitch, H typed out."""
    Ny, Nx, px, py, z = 6, 8, 3.1e-6, 4.65e-6, 0.004
    rng = np.random.default_rng(0)
    u0 = rng.standard_normal((Ny, Nx)) + 1j * rng.standard_normal((Ny, Nx))
    want = np.zeros((Ny, Nx), complex)
    for ky in range(Ny):
        for kx in range(Nx):
            fx = (kx if kx < Nx / 2 else kx - Nx) / (Nx * px)
            fy = (ky if ky < Ny / 2 else ky - Ny) / (Ny * py)
            H = cmath.exp(2j * math.pi * z * math.sqrt(1 / LAM ** 2 - fx * fx - fy * fy))
            Ak = sum(u0[n, m] * cmath.exp(-2j * math.pi * (kx * m / Nx + ky * n / Ny))
                     for n in range(Ny) for m in range(Nx))
            for n in range(Ny):
                for m in range(Nx):
                    want[n, m] += H * Ak * cmath.exp(2j * math.pi * (kx * m / Nx + ky * n / Ny)) / (Nx * Ny)
    got = A.propagate(u0, LAM, z, (px, py))
    assert np.max(np.abs(got - want)) < 1e-9


def test_forward_then_backward_is_the_identity_and_the_map_is_unitary():
    rng = np.random.default_rng(1)
    u0 = rng.standard_normal((64, 48)) + 1j * rng.standard_normal((64, 48))
    u = A.propagate(u0, LAM, 0.03, PITCH)           # at 4.65 um every bin propagates
    back = A.propagate(u, LAM, -0.03, PITCH)
    assert np.max(np.abs(back - u0)) < 1e-9
    assert abs(np.sum(A.intensity(u)) / np.sum(A.intensity(u0)) - 1) < 1e-12
    assert np.max(np.abs(A.propagate(u0, LAM, 0.0, PITCH) - u0)) < 1e-13
    # linearity and composition of distances
    v0 = rng.standard_normal((64, 48))
    assert np.max(np.abs(A.propagate(2 * u0 - 3j * v0, LAM, 0.03, PITCH)
                         - (2 * u - 3j * A.propagate(v0, LAM, 0.03, PITCH)))) < 1e-11
    assert np.max(np.abs(A.propagate(A.propagate(u0, LAM, 0.01, PITCH), LAM, 0.02, PITCH) - u)) < 1e-9


@pytest.mark.parametrize("z", [0.02, -0.05])
def test_paraxial_gaussian_beam(z):
    """u0 = exp(-r^2/w0^2), w0 = 100 um on 256^2 x 4.65 um: the exact transfer function reproduces the
    paraxial closed form exp(ikz)/(1 + i z/zR) exp(-r^2/(w0^2 (1 + i z/zR))) up to the paraxial error
    k z theta^4 / 8 with theta = lambda/(pi w0) = 2e-3, i.e. about 1e-6; the beam stays inside the window
    (w(z) <= 141 um of 595 um), so the periodic wrap is below 1e-7."""
    N, w0 = 256, 100e-6
    x = (np.arange(N) - N / 2) * PITCH
    r2 = x[None, :] ** 2 + x[:, None] ** 2
    u = A.propagate(np.exp(-r2 / w0 ** 2), LAM, z, PITCH)
    q = 1 + 1j * z / (np.pi * w0 ** 2 / LAM)
    zl = z / LAM
    want = np.exp(2j * np.pi * (zl - np.rint(zl))) / q * np.exp(-r2 / (w0 ** 2 * q))
    assert np.linalg.norm(u - want) / np.linalg.norm(want) < 5e-6


def test_agrees_with_the_fresnel_oracle_where_both_hold():
    """At S = 1/N (z = N p^2 / lambda) the Shifted-Fresnel transform keeps the pitch; for a compact
    smooth object (two Gaussian blobs, bandwidth 5e3 cycles/m) the Fresnel approximation error
    2 pi z lambda^3 f^4 / 8 is below 1e-5 rad and both oracles give the same field."""
    N, w0 = 256, 60e-6
    z = N * PITCH ** 2 / LAM
    x = (np.arange(N) - N / 2) * PITCH
    X, Y = x[None, :], x[:, None]
    u0 = np.exp(-((X - 80e-6) ** 2 + (Y + 40e-6) ** 2) / w0 ** 2) + 0.5j * np.exp(-((X + 120e-6) ** 2 + Y ** 2) / w0 ** 2)
    fres = O.separable_matrices(u0, LAM, z, PITCH, PITCH)
    asm = A.propagate(u0, LAM, z, PITCH)
    assert np.linalg.norm(asm - fres) / np.linalg.norm(fres) < 2e-5


def test_band_limit_and_phase_conventions():
    N, z = 64, 0.5
    H = A.transfer_function(N, N, LAM, z, PITCH, band_limit=True)
    fl = 1.0 / (LAM * math.sqrt((2.0 * z / (N * PITCH)) ** 2 + 1.0))      # typed out, SURVEY 8(d)
    f = A.frequencies(N, PITCH)
    keep = (np.abs(f)[None, :] <= fl) & (np.abs(f)[:, None] <= fl)
    assert 0 < keep.sum() < N * N
    assert np.all(H[~keep] == 0) and np.allclose(np.abs(H[keep]), 1.0)
    assert A.frequencies(8, 0.5).tolist() == [0.0, 0.25, 0.5, 0.75, -1.0, -0.75, -0.5, -0.25]
    u = np.array([[1 + 0j, 1j, -1, -1j, 0, 1 - 1j]])
    assert np.allclose(A.phase(u), [[0, math.pi / 2, math.pi, -math.pi / 2, 0, -math.pi / 4]])
    assert np.allclose(A.amplitude(u), [[1, 1, 1, 1, 0, math.sqrt(2)]])
    assert np.allclose(A.intensity(u), [[1, 1, 1, 1, 0, 2]])
    f3, I3, p3 = A.propagate_planes(np.ones((8, 8)), LAM, [0.01, -0.02], PITCH)
    assert f3.shape == (2, 8, 8) and np.allclose(I3, 1.0)
    with pytest.raises(ValueError):
        A.propagate(np.ones(4), LAM, 0.1, PITCH)
