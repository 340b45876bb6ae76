"""Pins of the float64 oracle against what the paper and the mathematics fix (CPU only).

The paper prints no worked numeric example (only sizes, L42/L86/L107/L115), so the pins are
closed forms, a textbook library-routine special case, brute force and invariants — chosen
so that a dropped term, a wrong sign or index, a swapped x/y operand or a wrong constant in
any of the oracle's three forms fails at least one of them.  Numbering follows SURVEY.md §8(c).
"""
import pathlib

import numpy as np
import pytest

from oracle import shifted_fresnel as O

LAM = 632.8e-9
P = 4.65e-6
GOLD = pathlib.Path(__file__).parent / "golden"


def rel_l2(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def rnd_complex(rng, shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


# parameter sets: (z, p0, p1, O1, O0) — anisotropic pitches, both signs of z, aliased S*N > 1/2
CASES = [
    (0.05, P, P, (0.0, 0.0), (0.0, 0.0)),
    (0.08, P, 2.0e-6, (0.4e-3, -0.3e-3), (0.0, 0.0)),
    (-0.06, P, 1.3e-6, (-0.2e-3, 0.1e-3), (0.0, 0.0)),
    (0.03, (P, 3.1e-6), (1.7e-6, 2.9e-6), (0.15e-3, 0.05e-3), (-0.07e-3, 0.11e-3)),
    (0.0007, P, P, (30e-6, -20e-6), (0.0, 0.0)),      # S*N = 0.78 at N = 16: aliased chirp
    (-0.0004, P, (2.0e-6, 4.0e-6), (0.0, 10e-6), (5e-6, 0.0)),
]


# ---- P1: brute force ------------------------------------------------------------------
@pytest.mark.parametrize("case", CASES)
def test_p1_forms_agree_n16(case):
    z, p0, p1, O1, O0 = case
    rng = np.random.default_rng(11)
    u0 = rnd_complex(rng, (16, 16))
    d = O.direct_sum(u0, LAM, z, p0, p1, O1, O0)
    m = O.separable_matrices(u0, LAM, z, p0, p1, O1, O0)
    b = O.bluestein_fft(u0, LAM, z, p0, p1, O1, O0)
    assert rel_l2(m, d) < 1e-13
    assert rel_l2(b, d) < 1e-12


def test_p1_forms_agree_rectangular():
    """N_y != N_x: catches any mix-up of the row and column sizes or pitches."""
    rng = np.random.default_rng(12)
    u0 = rnd_complex(rng, (12, 20))
    args = (LAM, 0.02, (P, 3.0e-6), (2.0e-6, 1.1e-6), (0.1e-3, -0.05e-3), (0.02e-3, 0.03e-3))
    d = O.direct_sum(u0, *args)
    assert rel_l2(O.separable_matrices(u0, *args), d) < 1e-13
    assert rel_l2(O.bluestein_fft(u0, *args), d) < 1e-12


def test_p1_config0_direct_sum_n64():
    """BASELINE.json config 0 at full size: the O(N^4) sum against the FFT form."""
    u0 = np.random.default_rng(0).random((64, 64), dtype=np.float32).astype(np.float64)
    d = O.direct_sum(u0, LAM, 0.05, P, P)
    b = O.bluestein_fft(u0, LAM, 0.05, P, P)
    m = O.separable_matrices(u0, LAM, 0.05, P, P)
    assert rel_l2(b, d) < 1e-12
    assert rel_l2(m, d) < 1e-13


# ---- P2: the definition at full size ----------------------------------------------------
def test_p2_fft_form_equals_definition_n1024():
    rng = np.random.default_rng(2)
    u0 = rng.random((1024, 1024))
    for z, p1, O1 in [(0.08, 2.0e-6, (0.4e-3, -0.3e-3)), (0.06, P, (0.0, 0.0))]:
        b = O.bluestein_fft(u0, LAM, z, P, p1, O1)
        m = O.separable_matrices(u0, LAM, z, P, p1, O1)
        assert rel_l2(b, m) < 1e-12


# ---- P3: textbook special case, a library routine ------------------------------------------
@pytest.mark.parametrize("N", [16, 64, 256])
def test_p3_reduces_to_single_fft_fresnel(N):
    """S = 1/N, zero shift (ordinary Fresnel diffraction, output pitch tied to
    lambda z / (N p0)): u1 = c0 exp(i pi r1^2/lz) * centred-DFT2[u0 exp(i pi r0^2/lz)], with the
    centred DFT = fftshift(fft2(ifftshift(.))) from numpy."""
    rng = np.random.default_rng(3)
    u0 = rnd_complex(rng, (N, N))
    p1 = 3.0e-6
    z = N * P * p1 / LAM                    # S = P p1 / (lam z) = 1/N
    x0 = (np.arange(N) - N / 2) * P
    x1 = (np.arange(N) - N / 2) * p1
    q0 = np.exp(1j * np.pi * (x0[None, :] ** 2 + x0[:, None] ** 2) / (LAM * z))
    q1 = np.exp(1j * np.pi * (x1[None, :] ** 2 + x1[:, None] ** 2) / (LAM * z))
    c0 = P * P * np.exp(2j * np.pi * (z / LAM % 1.0)) / (1j * LAM * z)
    ref = c0 * q1 * np.fft.fftshift(np.fft.fft2(np.fft.ifftshift(u0 * q0)))
    assert rel_l2(O.bluestein_fft(u0, LAM, z, P, p1), ref) < 1e-11
    assert rel_l2(O.separable_matrices(u0, LAM, z, P, p1), ref) < 1e-11
    if N <= 16:
        assert rel_l2(O.direct_sum(u0, LAM, z, P, p1), ref) < 1e-11


# ---- P4: closed form, delta input ------------------------------------------------------------
@pytest.mark.parametrize("form", ["D", "M", "B"])
@pytest.mark.parametrize("case", CASES[:4])
def test_p4_delta_gives_pure_chirp(form, case):
    z, p0, p1, O1, O0 = case
    N = 16 if form == "D" else 48
    fn = {"D": O.direct_sum, "M": O.separable_matrices, "B": O.bluestein_fft}[form]
    p0x, p0y = O._pair(p0)
    p1x, p1y = O._pair(p1)
    n0s, m0s = 5, 11                                      # off-diagonal: x/y swaps show
    u0 = np.zeros((N, N))
    u0[n0s, m0s] = 1.0
    x0s = (m0s - N / 2) * p0x + O0[0]
    y0s = (n0s - N / 2) * p0y + O0[1]
    x1 = (np.arange(N) - N / 2) * p1x + O1[0]
    y1 = (np.arange(N) - N / 2) * p1y + O1[1]
    c0 = p0x * p0y * np.exp(2j * np.pi * ((z / LAM) % 1.0)) / (1j * LAM * z)
    ref = c0 * np.exp(1j * np.pi * ((x1[None, :] - x0s) ** 2 + (y1[:, None] - y0s) ** 2)
                      / (LAM * z))
    got = fn(u0, LAM, z, p0, p1, O1, O0)
    assert rel_l2(got, ref) < 1e-11
    assert np.allclose(np.abs(got), p0x * p0y / (LAM * abs(z)), rtol=1e-12)


# ---- P5: closed form, Gaussian beam (pins the absolute normalisation, reading 9) --------------
@pytest.mark.parametrize("z,p1,O1", [(0.05, P, (0.0, 0.0)), (0.08, 2.0e-6, (40e-6, -25e-6)),
                                     (-0.03, 3.0e-6, (-30e-6, 10e-6)), (0.12, 6.0e-6, (0.0, 50e-6))])
def test_p5_gaussian_beam(z, p1, O1):
    N, w0 = 256, 100e-6
    x0 = (np.arange(N) - N / 2) * P
    u0 = np.exp(-(x0[None, :] ** 2 + x0[:, None] ** 2) / w0 ** 2)
    zR = np.pi * w0 ** 2 / LAM
    q = 1.0 + 1j * z / zR
    x1 = (np.arange(N) - N / 2) * p1 + O1[0]
    y1 = (np.arange(N) - N / 2) * p1 + O1[1]
    ref = (np.exp(2j * np.pi * ((z / LAM) % 1.0)) / q
           * np.exp(-(x1[None, :] ** 2 + y1[:, None] ** 2) / (w0 ** 2 * q)))
    for fn in (O.bluestein_fft, O.separable_matrices):
        got = fn(u0, LAM, z, P, p1, O1)
        assert np.max(np.abs(got - ref)) < 1e-11 * np.max(np.abs(ref))


# ---- P6: integer-pixel shifts are translations ---------------------------------------------------
@pytest.mark.parametrize("form", ["M", "B"])
def test_p6_integer_shift_is_translation(form):
    fn = {"M": O.separable_matrices, "B": O.bluestein_fft}[form]
    rng = np.random.default_rng(6)
    N, z, p1 = 64, 0.04, 2.2e-6
    u0 = rnd_complex(rng, (N, N))
    base = fn(u0, LAM, z, P, p1)
    kx, ky = 7, -4
    sh = fn(u0, LAM, z, P, p1, O1=(kx * p1, ky * p1))
    # sh[n1, m1] = base[n1 + ky, m1 + kx] on the overlap, all C1 phases included
    a = sh[4:N, 0:N - 7]
    b = base[0:N - 4, 7:N]
    assert rel_l2(a, b) < 1e-11


# ---- P7: +z then -z recovers the input (exact only at |S| N = 1) -------------------------------
@pytest.mark.parametrize("form", ["M", "B"])
def test_p7_round_trip(form):
    fn = {"M": O.separable_matrices, "B": O.bluestein_fft}[form]
    rng = np.random.default_rng(7)
    N, p1 = 64, 2.5e-6
    z = N * P * p1 / LAM
    O1 = (0.13e-3, -0.08e-3)
    u0 = rnd_complex(rng, (N, N))
    u1 = fn(u0, LAM, z, P, p1, O1=O1)
    back = fn(u1, LAM, -z, p1, P, O1=(0.0, 0.0), O0=O1)
    assert rel_l2(back, u0) < 1e-11


# ---- P8: symmetries and invariants -----------------------------------------------------------------
def test_p8_linearity():
    rng = np.random.default_rng(8)
    a, b = rnd_complex(rng, (32, 32)), rnd_complex(rng, (32, 32))
    args = (LAM, 0.05, P, 1.9e-6, (0.1e-3, 0.0))
    s = O.bluestein_fft(2.5 * a - 1.5j * b, *args)
    assert rel_l2(s, 2.5 * O.bluestein_fft(a, *args) - 1.5j * O.bluestein_fft(b, *args)) < 1e-12


def test_p8_conjugate_symmetry_real_hologram():
    rng = np.random.default_rng(9)
    u0 = rng.random((64, 64))
    args = (P, 2.0e-6, (0.2e-3, -0.1e-3))
    up = O.bluestein_fft(u0, LAM, +0.07, *args)
    um = O.bluestein_fft(u0, LAM, -0.07, *args)
    assert rel_l2(um, np.conj(up)) < 1e-12
    assert np.allclose(O.intensity(up), O.intensity(um), rtol=1e-10, atol=0)


def test_p8_energy_conservation_at_unitary_point():
    rng = np.random.default_rng(10)
    N, p1 = 128, 3.3e-6
    z = N * P * p1 / LAM
    u0 = rnd_complex(rng, (N, N))
    u1 = O.bluestein_fft(u0, LAM, z, P, p1)
    assert np.isclose(np.sum(O.intensity(u1)) * p1 * p1, np.sum(np.abs(u0) ** 2) * P * P,
                      rtol=1e-11)


def test_p8_independent_of_padding_and_free_sample():
    rng = np.random.default_rng(13)
    N = 32
    u0 = rnd_complex(rng, (N, N))
    args = (LAM, 0.03, P, 2.0e-6, (0.05e-3, 0.02e-3))
    ref = O.bluestein_fft(u0, *args)
    assert rel_l2(O.bluestein_fft(u0, *args, M=2 * N - 1), ref) < 1e-12
    assert rel_l2(O.bluestein_fft(u0, *args, M=96), ref) < 1e-12
    assert rel_l2(O.bluestein_fft(u0, *args, free_sample=123.0 - 7j), ref) < 1e-12
    with pytest.raises(ValueError):
        O.bluestein_fft(u0, *args, M=2 * N - 2)


def test_chirp_tables_are_eq2_eq3_with_pixel_offsets():
    """pre/post tables against Eq.(2)-(3) typed with the paper's own pixel-unit offsets."""
    N, z, p1 = 32, 0.05, 2.0e-6
    Ox1_m = 0.1e-3
    S = P * p1 / (LAM * z)
    m = np.arange(N)
    Ox1_px = Ox1_m / p1
    x0 = (m - N / 2) * P
    eq3 = (np.exp(1j * np.pi * x0 ** 2 / (LAM * z))
           * np.exp(-2j * np.pi * m * S * (-N / 2 + Ox1_px))
           * np.exp(-1j * np.pi * S * m ** 2))
    assert np.allclose(O.pre_chirp(N, LAM, z, P, p1, 0.0, Ox1_m), eq3, atol=1e-9)
    x1 = (m - N / 2) * p1 + Ox1_m
    eq2 = (np.exp(1j * np.pi * x1 ** 2 / (LAM * z))
           * np.exp(-2j * np.pi / (LAM * z) * (-N / 2) * P * x1)
           * np.exp(-1j * np.pi * S * m ** 2))
    assert np.allclose(O.post_chirp(N, LAM, z, P, p1, 0.0, Ox1_m), eq2, atol=1e-9)
    j = np.arange(2 * N)
    d = np.where(j <= N, j, j - 2 * N)
    assert np.allclose(O.chirp_kernel(N, 2 * N, S), np.exp(1j * np.pi * S * d ** 2), atol=1e-10)


# ---- the paper's printed constants ---------------------------------------------------------------------
def _paper_constants():
    vals = {}
    for line in (GOLD / "paper_constants.txt").read_text().splitlines():
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split("=")
            vals[k.strip()] = float(v)
    return vals


def test_paper_constants_field_of_view_and_sizes():
    c = _paper_constants()
    N = int(c["N"])
    x = O.coordinates(N, c["pitch_m"], 0.0)
    fov = x[-1] - x[0] + c["pitch_m"]
    assert abs(fov - c["field_of_view_m"]) < 0.05e-3          # "about 4.8 mm", L107
    assert int(c["padded"]) == 2 * N                           # L86, L115
    # ordinary-Fresnel distance at which the output pitch equals the CCD pitch (S = 1/N)
    z_unit = N * c["pitch_m"] ** 2 / c["lambda_m"]
    assert np.isclose(O.scale_factor(c["lambda_m"], z_unit, c["pitch_m"], c["pitch_m"]), 1 / N)


def test_golden_regression_n8():
    """Stored oracle output (written by tests/golden/make_golden.py from oracle/ only)."""
    g = np.loadtxt(GOLD / "oracle_n8.txt")
    u0 = np.arange(64, dtype=np.float64).reshape(8, 8) / 63.0
    u1 = O.direct_sum(u0, LAM, 0.002, P, 2.0e-6, O1=(3e-6, -2e-6))
    assert np.allclose(u1.real.ravel(), g[:, 0], rtol=0, atol=1e-15 + 1e-11 * np.abs(g).max())
    assert np.allclose(u1.imag.ravel(), g[:, 1], rtol=0, atol=1e-15 + 1e-11 * np.abs(g).max())


# ---- output helpers ---------------------------------------------------------------------------------------
def test_intensity_and_u8_quantisation():
    u = np.array([[3 + 4j, 0], [1j, -2]])
    assert np.array_equal(O.intensity(u), [[25.0, 0.0], [1.0, 4.0]])
    I = np.array([0.0, 0.5, 1.5, 2.5, 254.5, 255.0]) / 255.0 * 7.0     # ties -> even
    assert np.array_equal(O.quantise_u8(I), [0, 0, 2, 2, 254, 255])
    assert np.array_equal(O.quantise_u8(np.zeros((2, 2))), np.zeros((2, 2), np.uint8))
    assert np.array_equal(O.input_scale(np.array([[0, 255, 51]], np.uint8)), [[0.0, 1.0, 0.2]])


def test_argument_errors():
    u0 = np.ones((4, 4))
    with pytest.raises(ValueError):
        O.bluestein_fft(u0, LAM, 0.0, P, P)
    with pytest.raises(ValueError):
        O.direct_sum(u0, -1.0, 0.1, P, P)
    with pytest.raises(ValueError):
        O.separable_matrices(np.ones(4), LAM, 0.1, P, P)


def test_reconstruct_views_front_end():
    rng = np.random.default_rng(5)
    h = rng.integers(0, 256, (16, 16), dtype=np.uint8)
    z = np.array([0.01, -0.02]); p2 = np.array([2e-6, P]); ox = np.array([1e-5, 0.0])
    oy = np.array([0.0, -2e-5]); p1 = np.full(2, P)
    fb, ib = O.reconstruct_views(h, LAM, p1, p2, z, ox, oy, form="B")
    fd, _ = O.reconstruct_views(h, LAM, p1, p2, z, ox, oy, form="D")
    assert fb.shape == (2, 16, 16) and ib.shape == (2, 16, 16)
    assert rel_l2(fb, fd) < 1e-12
    assert np.allclose(ib, np.abs(fd) ** 2, rtol=1e-10)


# ---- row f2: focus moments of a depth stack ---------------------------------------------------
def test_focus_moments_closed_forms():
    """``focus_moments`` against values fixed without it: (a) a delta reconstructs to constant
    modulus p0^2/(lambda |z|) (P4), so sum I = N^2 c^2, sum I^2 = N^2 c^4 and the normalised
    variance is 0 at every depth; (b) at S = 1/N the map is unitary (P8): sum I p1^2 = sum |u0|^2 p0^2;
    (c) two-valued image: moments by counting."""
    N = 32
    u0 = np.zeros((N, N))
    u0[7, 20] = 1.0
    zs = [0.03, 0.05, -0.08]
    I = np.stack([O.intensity(O.bluestein_fft(u0, LAM, z, P, 2.0e-6, (0.1e-3, 0.0))) for z in zs])
    m = O.focus_moments(I)
    c2 = np.array([(P * P / (LAM * abs(z))) ** 2 for z in zs])
    assert np.allclose(m[:, 0], N * N * c2, rtol=1e-11)
    assert np.allclose(m[:, 1], N * N * c2 * c2, rtol=1e-11)
    assert np.all(np.abs(O.normalised_variance(m, N * N)) < 1e-10)
    rng = np.random.default_rng(21)
    p1 = 3.3e-6
    z = N * P * p1 / LAM
    u = rng.random((N, N))
    m = O.focus_moments(O.intensity(O.bluestein_fft(u, LAM, z, P, p1))[None])
    assert np.isclose(m[0, 0] * p1 * p1, np.sum(u * u) * P * P, rtol=1e-11)
    img = np.full((1, 4, 4), 2.0)
    img[0, :2] = 3.0                       # 8 pixels of 3, 8 pixels of 2
    m = O.focus_moments(img)
    assert m[0, 0] == 40.0 and m[0, 1] == 8 * 9 + 8 * 4
    assert np.isclose(O.normalised_variance(m, 16)[0], 16 * 104 / 1600 - 1)


def test_crop_window_reading_13():
    """PAPER.md L42 / reading 13: the 1 360 x 1 024 frame is cropped to its central 1 024 columns; a
    window moved off centre by (dr, dc) samples equals the centred transform of the same samples with
    the hologram-window offset O_0 = (dc p, dr p) (the physical positions of the samples are what count)."""
    rng = np.random.default_rng(3)
    frame = rng.integers(0, 256, (1024, 1360), dtype=np.uint8)
    w = O.crop_window(frame, 1024, 1024)
    assert w.shape == (1024, 1024) and np.array_equal(w, frame[:, 168:1192])
    assert np.array_equal(O.crop_window(frame, 64, 32, 5, 7), frame[5:69, 7:39])
    with pytest.raises(ValueError):
        O.crop_window(frame, 1024, 1024, 1, 0)
    # physics: a 24 x 40 frame, window 16 x 16 moved by (dr, dc) = (3, -5) off centre
    small = rng.random((24, 40))
    lam, z, p = 632.8e-9, 0.004, 4.65e-6
    dr, dc = 3, -5
    win = O.crop_window(small, 16, 16, (24 - 16) // 2 + dr, (40 - 16) // 2 + dc)
    got = O.separable_matrices(win, lam, z, p, 2e-6, O1=(1e-5, -2e-5), O0=(dc * p, dr * p))
    # the same samples placed at their physical positions inside a zero frame, centred transform,
    # evaluated on the same output window
    big = np.zeros((24, 40))
    big[4 + dr:20 + dr, 12 + dc:28 + dc] = win
    Kx = O.fresnel_matrix(40, lam, z, p, 2e-6, 0.0, 1e-5 + (40 - 16) / 2 * 2e-6)[:16]
    Ky = O.fresnel_matrix(24, lam, z, p, 2e-6, 0.0, -2e-5 + (24 - 16) / 2 * 2e-6)[:16]
    want = O.c0_factor(lam, z, p, p) * (Ky @ big @ Kx.T)
    assert np.linalg.norm(got - want) / np.linalg.norm(want) < 1e-12
