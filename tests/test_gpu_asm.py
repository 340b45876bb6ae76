"""GPU parity of angular-spectrum propagation: sfd_asm_* through the C ABI against
the float64 oracle (oracle/angular_spectrum.py), element by element, at the north_star tolerance
(rel-L2 <= 2e-5, max |du| <= 1e-4 max|u| per plane; phase to 2e-4 rad where |u| is not small)."""
import math

import numpy as np
import pytest
import torch

from oracle import angular_spectrum as A
from paper_1001_4309_b200 import build as sfd_build
from paper_1001_4309_b200 import workloads as W

sfd_build.build()
from paper_1001_4309_b200 import binding as B  # noqa: E402

pytestmark = pytest.mark.gpu
REL_L2, REL_MAX = 2e-5, 1e-4


def _dev():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device (no CPU fallback exists)"
    return torch.device("cuda:0")


def _check(f, I, ph, want, what):
    for p in range(want.shape[0]):
        d = f[p].astype(np.complex128) - want[p]
        l2 = np.linalg.norm(d) / np.linalg.norm(want[p])
        mx = np.abs(d).max() / np.abs(want[p]).max()
        assert l2 <= REL_L2 and mx <= REL_MAX, f"{what} plane {p}: rel-L2 {l2:.2e}, max {mx:.2e}"
        Iw = A.intensity(want[p])
        assert np.abs(I[p] - Iw).max() <= REL_MAX * Iw.max()
        big = np.abs(want[p]) > 0.05 * np.abs(want[p]).max()
        dphi = np.angle(np.exp(1j * (ph[p] - A.phase(want[p]))))        # wrapped difference
        assert np.abs(dphi[big]).max() < 2e-4, f"{what} plane {p}: phase off by {np.abs(dphi[big]).max():.2e}"
        assert ph[p].min() >= -math.pi - 1e-6 and ph[p].max() <= math.pi + 1e-6


@pytest.mark.parametrize("Nx,Ny,dtype,pitch,zs,bl", [
    (128, 128, B.SFD_C64, W.PITCH, [0.01, -0.02], False),
    (256, 128, B.SFD_F32, (3.0e-6, 5.0e-6), [0.004, 0.05, 0.0], False),      # rectangular, anisotropic, z = 0
    (512, 1024, B.SFD_C64, W.PITCH, [0.08], True),                           # band limit active
    (1024, 1024, B.SFD_C64, W.PITCH, [0.08, -0.06], False),                  # the warp-FFT kernels
    (1024, 1024, B.SFD_F32, (4.0e-6, 5.5e-6), [0.03, 0.0, -0.11, 0.2, 0.051], True),  # 5 planes: tile and table reuse
    (2048, 2048, B.SFD_F32, W.PITCH, [0.08], True),                          # the hologram generator's grid: pair-of-warps kernels
    (2048, 2048, B.SFD_C64, (4.0e-6, 5.5e-6), [0.05, -0.12, 0.0], False),    # 3 planes: spectrum kept, tile and table reuse
    (4096, 2048, B.SFD_C64, 0.4e-6, [20e-6], False),                         # evanescent bins (pitch < lambda/2 .. )
])
def test_asm_against_oracle(Nx, Ny, dtype, pitch, zs, bl):
    rng = np.random.default_rng(Nx + Ny)
    if dtype == B.SFD_F32:
        u0 = rng.random((Ny, Nx), dtype=np.float32)
        u0[Ny - 1, Nx - 1] = 9.0
    else:
        u0 = (rng.standard_normal((Ny, Nx)) + 1j * rng.standard_normal((Ny, Nx))).astype(np.complex64)
        u0[Ny - 1, Nx - 1] = 9.0 - 4.0j
        u0[0, Nx - 2] = -7.0j
    with B.AsmPlan(Nx, Ny, W.LAMBDA, pitch, zs, dtype, bl) as plan:
        n0 = B.sfd_launch_count()
        f, I, ph = plan.execute(torch.from_numpy(u0).to(_dev()))
        torch.cuda.synchronize()
        assert B.sfd_launch_count() - n0 == 3
        assert plan.device_bytes > 0
    want, _, _ = A.propagate_planes(u0, W.LAMBDA, zs, pitch, bl)
    _check(f.cpu().numpy(), I.cpu().numpy(), ph.cpu().numpy(), want, f"{Nx}x{Ny}")


def test_plane_wave_eigenvalue_on_gpu_output():
    """The oracle's pin applied to the CUDA path: a plane wave comes back multiplied by the analytic H."""
    N, kx, ky, z = 256, 200, 17, 0.031
    n, m = np.mgrid[0:N, 0:N]
    u0 = np.exp(2j * np.pi * (kx * m / N + ky * n / N)).astype(np.complex64)
    with B.AsmPlan(N, N, W.LAMBDA, W.PITCH, [z]) as plan:
        f, _, _ = plan.execute(torch.from_numpy(u0).to(_dev()), intensity=False, phase=False)
        torch.cuda.synchronize()
    fx, fy = (kx - N) / (N * W.PITCH), ky / (N * W.PITCH)
    cyc = z * math.sqrt(1 / W.LAMBDA ** 2 - fx * fx - fy * fy)
    eig = np.exp(2j * np.pi * (cyc - round(cyc)))
    assert np.abs(f[0].cpu().numpy() - eig * u0.astype(np.complex128)).max() < 2e-5


def test_gabor_hologram_generator_on_the_gpu():
    """What row f4 is for: the synthetic-hologram recipe of SURVEY.md 8(d) (object transmittance t on a 2N
    grid, u = ASM(t - 1), I = |1 + u|^2) with the propagation done by the library, against the oracle."""
    N, z = 512, 0.05
    rng = np.random.default_rng(12)
    t = np.ones((2 * N, 2 * N), np.float32)
    for _ in range(12):
        cy, cx, r = rng.integers(N // 2, 3 * N // 2, 2).tolist() + [int(rng.integers(2, 9))]
        yy, xx = np.ogrid[-r:r + 1, -r:r + 1]
        t[cy - r:cy + r + 1, cx - r:cx + r + 1][yy * yy + xx * xx <= r * r] = 0.0
    with B.AsmPlan(2 * N, 2 * N, W.LAMBDA, W.PITCH, [z], B.SFD_F32, band_limit=True) as plan:
        f, _, _ = plan.execute(torch.from_numpy(t - 1.0).to(_dev()), intensity=False, phase=False)
        I = (1.0 + f[0]).abs().square()[N // 2:N // 2 + N, N // 2:N // 2 + N]
        torch.cuda.synchronize()
    u = A.propagate((t - 1.0).astype(np.float64), W.LAMBDA, z, W.PITCH, band_limit=True)
    Iw = np.abs(1.0 + u[N // 2:N // 2 + N, N // 2:N // 2 + N]) ** 2
    assert np.abs(I.cpu().numpy() - Iw).max() < 1e-4 * Iw.max()
    g8, w8 = np.rint(255 * I.cpu().numpy() / I.max().item()), np.rint(255 * Iw / Iw.max())
    assert np.abs(g8 - w8).max() <= 1 and (g8 != w8).mean() < 1e-3


@pytest.mark.parametrize("N", [128, 1024])      # generic line kernels, warp-FFT kernels
def test_asm_outputs_optional_and_reusable(N):
    u0 = torch.randn(N, N, dtype=torch.complex64, device=_dev())
    with B.AsmPlan(N, N, W.LAMBDA, W.PITCH, [0.02]) as plan:
        f, I, ph = plan.execute(u0)
        f2, none_i, none_p = plan.execute(u0, intensity=False, phase=False)
        none_f, I2, ph2 = plan.execute(u0, field=False)
        torch.cuda.synchronize()
        assert none_i is None and none_p is None and none_f is None
        assert torch.equal(f, f2) and torch.equal(I, I2) and torch.equal(ph, ph2)
        with pytest.raises(B.SfdError) as e:
            plan.execute(u0, field=False, intensity=False, phase=False)
        assert e.value.code == B.SFD_EINVAL


def test_asm_1024_back_to_back_calls_do_not_interfere():
    """The three warp-FFT kernels are chained by programmatic dependent launch and reuse the plan's A and W
    buffers: calls queued without synchronisation on different inputs must each give their own result."""
    N, zs = 1024, [0.05, 0.09, -0.02]
    rng = np.random.default_rng(5)
    ins = [(rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))).astype(np.complex64) for _ in range(3)]
    dev_in = [torch.from_numpy(u).to(_dev()) for u in ins]
    with B.AsmPlan(N, N, W.LAMBDA, W.PITCH, zs) as plan:
        outs = [plan.execute(d, phase=False) for d in dev_in for _ in range(2)]   # a, a, b, b, c, c
        torch.cuda.synchronize()
    for i, u in enumerate(ins):
        want, _, _ = A.propagate_planes(u, W.LAMBDA, zs, W.PITCH)
        for f, I, _ in outs[2 * i:2 * i + 2]:
            d = f.cpu().numpy().astype(np.complex128) - want
            assert np.linalg.norm(d) / np.linalg.norm(want) <= REL_L2
            assert np.abs(I.cpu().numpy() - A.intensity(want)).max() <= REL_MAX * A.intensity(want).max()
        assert torch.equal(outs[2 * i][0], outs[2 * i + 1][0])


def test_asm_2048_rejects_an_input_that_is_not_16_byte_aligned():
    """The 2048 x 2048 kernels fetch input rows as bulk copies (16-byte granules): an input 8 bytes off is an
    argument error, not a fault; the same view shifted back works."""
    N = 2048
    buf = torch.randn(N * N + 2, dtype=torch.complex64, device=_dev())
    assert buf.data_ptr() % 16 == 0
    with B.AsmPlan(N, N, W.LAMBDA, W.PITCH, [0.05]) as plan:
        with pytest.raises(B.SfdError) as e:
            plan.execute(buf[1:1 + N * N].view(N, N), intensity=False, phase=False)
        assert e.value.code == B.SFD_EINVAL
        f, _, _ = plan.execute(buf[2:2 + N * N].view(N, N), intensity=False, phase=False)
        torch.cuda.synchronize()
        assert torch.isfinite(f.abs().max())


@pytest.mark.parametrize("seed", range(8))
def test_random_asm_plans_against_oracle(seed):
    """Seeded sweep: grid sides drawn from 128 .. 2048 independently (square 1024 and 2048 forced in for two seeds:
    the warp-FFT paths), 1 - 3 planes of either sign, real or complex input, anisotropic pitch, band limit on or off."""
    rng = np.random.default_rng(2000 + seed)
    Nx, Ny = (int(2 ** rng.integers(7, 12)) for _ in range(2))
    if seed == 0:
        Nx = Ny = 1024
    if seed == 1:
        Nx = Ny = 2048
    zs = list(rng.uniform(0.005, 0.2, int(rng.integers(1, 4))) * rng.choice([-1.0, 1.0]))
    dtype = B.SFD_F32 if rng.random() < 0.5 else B.SFD_C64
    pitch = (float(rng.uniform(2e-6, 6e-6)), float(rng.uniform(2e-6, 6e-6)))
    bl = bool(rng.random() < 0.5)
    if dtype == B.SFD_F32:
        u0 = rng.random((Ny, Nx), dtype=np.float32)
    else:
        u0 = (rng.standard_normal((Ny, Nx)) + 1j * rng.standard_normal((Ny, Nx))).astype(np.complex64)
    with B.AsmPlan(Nx, Ny, W.LAMBDA, pitch, zs, dtype, bl) as plan:
        f, I, ph = plan.execute(torch.from_numpy(u0).to(_dev()))
        torch.cuda.synchronize()
    want, _, _ = A.propagate_planes(u0, W.LAMBDA, zs, pitch, bl)
    _check(f.cpu().numpy(), I.cpu().numpy(), ph.cpu().numpy(), want, f"seed {seed}: {Nx}x{Ny}, {len(zs)} planes")
