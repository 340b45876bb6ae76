"""GPU parity: the CUDA path (through the C ABI) against the float64 oracle, element by element.

Tolerances are the north_star's (BASELINE.json): per view, relative L2 error <= 2e-5 and
max|du| <= 1e-4 max|u|; the same bounds are applied to the intensity."""
import numpy as np
import pytest
import torch

from oracle import shifted_fresnel as O
from paper_1001_4309_b200 import build as sfd_build
from paper_1001_4309_b200 import workloads as W

sfd_build.build()
from paper_1001_4309_b200 import binding as B  # noqa: E402

pytestmark = pytest.mark.gpu

REL_L2 = 2e-5
REL_MAX = 1e-4


def _dev():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device (no CPU fallback exists)"
    return torch.device("cuda:0")


def _assert_close(got, want, what):
    got = np.asarray(got)
    want = np.asarray(want)
    assert got.shape == want.shape
    for v in range(want.shape[0]):
        d = got[v].astype(want.dtype) - want[v]
        l2 = np.linalg.norm(d) / np.linalg.norm(want[v])
        mx = np.max(np.abs(d)) / np.max(np.abs(want[v]))
        assert l2 <= REL_L2, f"{what} view {v}: rel-L2 {l2:.3e} > {REL_L2}"
        assert mx <= REL_MAX, f"{what} view {v}: max err {mx:.3e} > {REL_MAX}"


def _run(wl, holo=None, kernels=None, **kw):
    holo = wl.hologram() if holo is None else holo
    with B.Plan(wl) as plan:
        if kernels is not None:
            plan.select_kernels(kernels)
        f, I = plan.execute(torch.from_numpy(holo).to(_dev()), **kw)
        torch.cuda.synchronize()
        return holo, (None if f is None else f.cpu().numpy()), (None if I is None else I.cpu().numpy())


def test_config0_tiny_against_the_definition():
    """Config 0: 64x64 float32, 1 view; oracle form D (direct O(N^4) double sum) and form B."""
    wl = W.config(0)
    holo, f, I = _run(wl)
    fD, ID = O.reconstruct_views(holo, wl.lam, wl.p1, wl.p2, wl.z, wl.Ox, wl.Oy, form="D")
    fB, _ = O.reconstruct_views(holo, wl.lam, wl.p1, wl.p2, wl.z, wl.Ox, wl.Oy, form="B")
    _assert_close(f, fD, "field vs form D")
    _assert_close(f, fB, "field vs form B")
    _assert_close(I, ID, "intensity vs form D")


def test_small_multiview_all_forms():
    """256^2 uint8, 3 views with mixed sign of z: several CTAs per pass, several views."""
    wl = W.small_multiview()
    holo, f, I = _run(wl)
    fB, IB = O.reconstruct_views(holo, wl.lam, wl.p1, wl.p2, wl.z, wl.Ox, wl.Oy, form="B")
    fM, _ = O.reconstruct_views(holo, wl.lam, wl.p1, wl.p2, wl.z, wl.Ox, wl.Oy, form="M")
    _assert_close(f, fB, "field vs form B")
    _assert_close(f, fM, "field vs form M")
    _assert_close(I, IB, "intensity")


@pytest.mark.parametrize("cfg", [1, 2])
def test_configs_1024_full(cfg):
    """Configs 1 and 2 at full size, every output element, in the launch configuration bench.py
    times (same plan parameters, uint8 hologram from the same generator)."""
    wl = W.config(cfg)
    holo, f, I = _run(wl)
    fB, IB = O.reconstruct_views(holo, wl.lam, wl.p1, wl.p2, wl.z, wl.Ox, wl.Oy, form="B")
    _assert_close(f, fB, f"config {cfg} field")
    _assert_close(I, IB, f"config {cfg} intensity")


@pytest.mark.parametrize("in_dtype", [W.IN_U8, W.IN_F32])
def test_1024_generic_and_warp_kernels_agree_with_oracle(in_dtype):
    """N = 1024 has two kernel sets (one warp per line; generic Stockham, 5.3).
    Both must meet the tolerance against the oracle, for both input types, with a delta in the
    last row/column so that an indexing slip at the tile edges shows."""
    wl = W.config(2)
    if in_dtype == W.IN_F32:
        holo = np.random.default_rng(5).random((1024, 1024), dtype=np.float32)
        holo[1023, 1023] = 40.0
        holo[0, 1021] = 25.0
        wl = W.Workload("rand1024", 1024, wl.lam, wl.p1, wl.p2, wl.z, wl.Ox, wl.Oy, W.IN_F32)
    else:
        holo = wl.hologram().copy()
        holo[1023, 1023] = 255
        holo[0, 1021] = 0
    fB, IB = O.reconstruct_views(holo, wl.lam, wl.p1, wl.p2, wl.z, wl.Ox, wl.Oy, form="B")
    for which in (B.SFD_KERNELS_AUTO, B.SFD_KERNELS_GENERIC):
        _, f, I = _run(wl, holo, kernels=which)
        _assert_close(f, fB, f"kernels={which} field")
        _assert_close(I, IB, f"kernels={which} intensity")


def test_config4_scale_stress_full():
    """Config 4: 2048^2, 16 views (4096-point FFTs), contains aliased views (reading 16)."""
    wl = W.config(4)
    holo, f, I = _run(wl)
    fB, IB = O.reconstruct_views(holo, wl.lam, wl.p1, wl.p2, wl.z, wl.Ox, wl.Oy, form="B")
    _assert_close(f, fB, "config 4 field")
    _assert_close(I, IB, "config 4 intensity")


@pytest.mark.parametrize("N", [64, 128, 256, 512, 1024, 2048])
def test_every_size_float_input(N):
    """Every supported N (each has its own radix schedule), float32 input, two views (z<0 too)."""
    rng = np.random.default_rng(N)
    holo = rng.random((N, N), dtype=np.float32)
    wl = W.Workload(f"rand{N}", N, W.LAMBDA, np.full(2, W.PITCH), np.array([3.1e-6, 4.65e-6]),
                    np.array([0.07, -0.04]), np.array([0.2e-3, 0.0]), np.array([-0.1e-3, 0.0]),
                    W.IN_F32)
    _, f, I = _run(wl, holo)
    fB, IB = O.reconstruct_views(holo, wl.lam, wl.p1, wl.p2, wl.z, wl.Ox, wl.Oy, form="B")
    _assert_close(f, fB, f"N={N} field")
    _assert_close(I, IB, f"N={N} intensity")


def test_delta_closed_form_on_gpu_output():
    """Pin P4 applied to the GPU result itself: a single bright sample reconstructs to the pure
    chirp c0 exp(i pi [(x1-x0*)^2 + (y1-y0*)^2]/(lambda z)) (Eq. 1 with one term)."""
    N, lam, p1, p2, z, Ox, Oy = 256, W.LAMBDA, W.PITCH, 2.3e-6, 0.04, 0.15e-3, -0.25e-3
    holo = np.zeros((N, N), np.float32)
    n0, m0 = 37, 201
    holo[n0, m0] = 1.0
    wl = W.Workload("delta", N, lam, np.array([p1]), np.array([p2]), np.array([z]), np.array([Ox]),
                    np.array([Oy]), W.IN_F32)
    _, f, I = _run(wl, holo)
    x0 = (m0 - N / 2) * p1
    y0 = (n0 - N / 2) * p1
    x1 = (np.arange(N) - N / 2) * p2 + Ox
    y1 = (np.arange(N) - N / 2) * p2 + Oy
    ph = ((x1[None, :] - x0) ** 2 + (y1[:, None] - y0) ** 2) / (2 * lam * z)
    zl = z / lam
    want = p1 * p1 * np.exp(2j * np.pi * (zl - np.rint(zl))) / (1j * lam * z) * np.exp(
        2j * np.pi * (ph - np.rint(ph)))
    _assert_close(f, want[None], "delta field")
    assert np.allclose(I[0], (p1 * p1 / (lam * abs(z))) ** 2, rtol=2e-4)


def test_outputs_optional_and_consistent():
    wl = W.small_multiview(N=128, V=2, seed=11)
    holo, f, I = _run(wl)
    _, f2, none_i = _run(wl, holo, intensity=False)
    _, none_f, I2 = _run(wl, holo, field=False)
    assert none_i is None and none_f is None
    assert np.array_equal(f, f2) and np.array_equal(I, I2)
    with B.Plan(wl) as plan:
        with pytest.raises(B.SfdError) as e:
            plan.execute(torch.from_numpy(holo).to(_dev()), field=False, intensity=False)
        assert e.value.code == B.SFD_EINVAL


def test_plan_reuse_two_plans_and_side_stream():
    """One plan executed many times gives the same bits; two live plans do not disturb each other;
    execution on a non-default stream is ordered by that stream."""
    dev = _dev()
    wa, wb = W.small_multiview(N=256, V=2, seed=3), W.small_multiview(N=128, V=3, seed=5)
    ha, hb = torch.from_numpy(wa.hologram()).to(dev), torch.from_numpy(wb.hologram()).to(dev)
    with B.Plan(wa) as pa, B.Plan(wb) as pb:
        fa0, _ = pa.execute(ha)
        fb0, _ = pb.execute(hb)
        s = torch.cuda.Stream()
        s.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(s):
            for _ in range(5):
                fa, _ = pa.execute(ha)
                fb, _ = pb.execute(hb)
        s.synchronize()
        assert torch.equal(fa, fa0) and torch.equal(fb, fb0)
    fB, _ = O.reconstruct_views(wa.hologram(), wa.lam, wa.p1, wa.p2, wa.z, wa.Ox, wa.Oy)
    _assert_close(fa.cpu().numpy(), fB, "reused plan")


def test_update_view_rebuilds_tables():
    wl = W.small_multiview(N=128, V=2, seed=9)
    holo = wl.hologram()
    dev = _dev()
    with B.Plan(wl) as plan:
        plan.update_view(1, W.PITCH, 1.7e-6, -0.033, 0.05e-3, 0.02e-3)
        f, _ = plan.execute(torch.from_numpy(holo).to(dev))
        f = f.cpu().numpy()
    p2 = wl.p2.copy(); z = wl.z.copy(); Ox = wl.Ox.copy(); Oy = wl.Oy.copy()
    p2[1], z[1], Ox[1], Oy[1] = 1.7e-6, -0.033, 0.05e-3, 0.02e-3
    fB, _ = O.reconstruct_views(holo, wl.lam, wl.p1, p2, z, Ox, Oy)
    _assert_close(f, fB, "updated view")


def _u8_check(got, I_oracle, what):
    """8-bit output (reading 15): equal to the oracle's quantisation except where 255 I/max sits
    within float32 rounding of a .5 boundary; there +-1 LSB is allowed."""
    for v in range(I_oracle.shape[0]):
        want = O.quantise_u8(I_oracle[v]).astype(np.int16)
        d = np.abs(got[v].astype(np.int16) - want)
        assert d.max() <= 1, f"{what} view {v}: off by {d.max()} LSB"
        x = 255.0 * I_oracle[v] / I_oracle[v].max()
        near = np.abs(x - np.floor(x) - 0.5) < 1e-3 * np.maximum(x, 1.0)
        assert not np.any((d == 1) & ~near), f"{what} view {v}: 1-LSB error away from a boundary"
        assert (d == 1).mean() < 5e-3


def test_execute_u8_against_oracle_quantisation():
    wl = W.small_multiview(N=256, V=3, seed=21)
    holo = wl.hologram()
    with B.Plan(wl) as plan:
        out = plan.execute_u8(torch.from_numpy(holo).to(_dev())).cpu().numpy()
    _, IB = O.reconstruct_views(holo, wl.lam, wl.p1, wl.p2, wl.z, wl.Ox, wl.Oy)
    _u8_check(out, IB, "execute_u8")
    # an all-zero hologram gives all-zero images (degenerate max)
    with B.Plan(wl) as plan:
        z = plan.execute_u8(torch.zeros((wl.N, wl.N), dtype=torch.uint8, device=_dev()))
        assert int(z.max()) == 0


def test_stream_run_matches_execute_u8_and_oracle():
    """Config 3 shape (1024^2, 4 views) on 6 frames: the double-buffered pinned pipeline returns,
    frame by frame, the same bytes as sfd_execute_u8, and those match the oracle."""
    wl = W.config(3, n_frames=6)
    frames = np.stack([wl.hologram(f) for f in range(wl.n_frames)])
    pinned = torch.from_numpy(frames).pin_memory()
    dev = _dev()
    with B.Plan(wl) as plan:
        out, sec = plan.stream_run(pinned)
        assert sec > 0
        for f in range(wl.n_frames):
            ref = plan.execute_u8(pinned[f].to(dev))
            assert torch.equal(ref.cpu(), out[f]), f"frame {f}: stream differs from execute_u8"
        out2, _ = plan.stream_run(pinned)      # the pipeline is reusable
        assert torch.equal(out, out2)
    for f in (0, wl.n_frames - 1):
        _, IB = O.reconstruct_views(frames[f], wl.lam, wl.p1, wl.p2, wl.z, wl.Ox, wl.Oy)
        _u8_check(out[f].numpy(), IB, f"stream frame {f}")


def test_stream_run_edge_cases():
    wl = W.small_multiview(N=128, V=1, seed=2)
    with B.Plan(wl) as plan:
        one = torch.from_numpy(wl.hologram()[None]).pin_memory()
        out, sec = plan.stream_run(one)                      # a single frame (no overlap partner)
        ref = plan.execute_u8(one[0].to(_dev())).cpu()
        assert torch.equal(out[0], ref)
        assert B.sfd_stream_run(plan.handle, one, 0, out) == 0.0   # zero frames: no work, OK


def test_launch_counter_and_kernel_timing():
    wl = W.small_multiview(N=128, V=2, seed=4)
    h = torch.from_numpy(wl.hologram()).to(_dev())
    with B.Plan(wl) as plan:
        n0 = B.sfd_launch_count()
        plan.execute(h)
        assert B.sfd_launch_count() - n0 == 2          # pass y, pass x
        plan.execute_u8(h)
        assert B.sfd_launch_count() - n0 == 5          # + pass y, pass x, quantise
        plan.set_timing(True)
        plan.execute(h)
        ms = plan.last_kernel_ms()
        assert ms[0] > 0 and ms[1] > 0 and ms[2] == 0
        assert plan.device_bytes > 0 and B.sfd_plan_get_m(plan.handle) == 256


# ---- general geometry: S_x != S_y, hologram-window offsets -----------------
_GENERAL = dict(
    p1x=[4.65e-6, 5.5e-6, 4.65e-6], p1y=[4.65e-6, 4.0e-6, 6.2e-6],
    p2x=[2.0e-6, 1.5e-6, 4.65e-6], p2y=[3.0e-6, 1.5e-6, 1.2e-6],
    z=[0.08, 0.06, -0.07],
    O0x=[0.0, 0.15e-3, -0.2e-3], O0y=[0.1e-3, 0.0, 0.3e-3],
    O1x=[0.4e-3, -0.5e-3, 0.0], O1y=[-0.3e-3, 0.2e-3, 0.6e-3])


def _general_oracle(holo, g, form="B"):
    fn = {"B": O.bluestein_fft, "M": O.separable_matrices}[form]
    u0 = O.input_scale(holo)
    return np.stack([fn(u0, W.LAMBDA, g["z"][v], (g["p1x"][v], g["p1y"][v]), (g["p2x"][v], g["p2y"][v]),
                        O1=(g["O1x"][v], g["O1y"][v]), O0=(g["O0x"][v], g["O0y"][v]))
                     for v in range(len(g["z"]))])


@pytest.mark.parametrize("N,in_dtype", [(128, B.SFD_F32), (256, B.SFD_U8), (1024, B.SFD_U8)])
def test_general_geometry_against_oracle(N, in_dtype):
    """Anisotropic pitches (S_x != S_y), shifted hologram and reconstruction windows, z < 0; the
    generic kernels (N = 128, 256) and the N = 1024 warp-pair kernels, against forms B and M."""
    rng = np.random.default_rng(31 + N)
    holo = (rng.random((N, N), dtype=np.float32) if in_dtype == B.SFD_F32
            else rng.integers(0, 256, (N, N), dtype=np.uint8))
    with B.Plan(N=N, lam=W.LAMBDA, in_dtype=in_dtype, **_GENERAL) as plan:
        f, I = plan.execute(torch.from_numpy(holo).to(_dev()))
        torch.cuda.synchronize()
        f, I = f.cpu().numpy(), I.cpu().numpy()
    want = _general_oracle(holo, _GENERAL, "B")
    _assert_close(f, want, "general geometry field vs form B")
    _assert_close(I, O.intensity(want), "general geometry intensity")
    if N <= 256:
        _assert_close(f, _general_oracle(holo, _GENERAL, "M"), "general geometry field vs form M")


def test_general_update_view_and_square_equivalence():
    """sfd_plan_update_view_general rebuilds both axes; with p1x = p1y, p2x = p2y, O0 = 0 the general
    plan is bit-identical to the square one."""
    N = 256
    wl = W.small_multiview(N=N, V=3, seed=7)
    holo = wl.hologram()
    h = torch.from_numpy(holo).to(_dev())
    zero = np.zeros(3)
    with B.Plan(wl) as sq, B.Plan(N=N, lam=wl.lam, in_dtype=wl.in_dtype, p1x=wl.p1, p1y=wl.p1, p2x=wl.p2,
                                  p2y=wl.p2, z=wl.z, O0x=zero, O0y=zero, O1x=wl.Ox, O1y=wl.Oy) as ge:
        f1, _ = sq.execute(h)
        f2, _ = ge.execute(h)
        torch.cuda.synchronize()
        assert torch.equal(f1, f2)
        g = _GENERAL
        for v in range(3):
            ge.update_view_general(v, g["p1x"][v], g["p1y"][v], g["p2x"][v], g["p2y"][v], g["z"][v],
                                   g["O0x"][v], g["O0y"][v], g["O1x"][v], g["O1y"][v])
        f3, _ = ge.execute(h)
        torch.cuda.synchronize()
    _assert_close(f3.cpu().numpy(), _general_oracle(holo, _GENERAL), "after update_view_general")


def test_round_trip_on_gpu_at_unit_SN():
    """Pin P7 applied to the CUDA path: at |S| N = 1 propagating +z from (p1, O0 = 0) to (p2, O1) and
    -z back from that grid recovers the input (needs the hologram-window offset of the general API)."""
    N, p1, p2 = 256, 4.65e-6, 3.1e-6
    z = N * p1 * p2 / W.LAMBDA
    O1x, O1y = 0.12e-3, -0.07e-3
    u0 = np.random.default_rng(5).random((N, N), dtype=np.float32)
    one = lambda v: [v]
    with B.Plan(N=N, lam=W.LAMBDA, in_dtype=B.SFD_F32, p1x=one(p1), p1y=one(p1), p2x=one(p2), p2y=one(p2),
                z=one(z), O0x=one(0.0), O0y=one(0.0), O1x=one(O1x), O1y=one(O1y)) as fwd:
        f, _ = fwd.execute(torch.from_numpy(u0).to(_dev()))
        torch.cuda.synchronize()
    u1 = f[0].cpu().numpy()
    # the way back is linear: real and imaginary parts are propagated separately (float32 inputs)
    with B.Plan(N=N, lam=W.LAMBDA, in_dtype=B.SFD_F32, p1x=one(p2), p1y=one(p2), p2x=one(p1), p2y=one(p1),
                z=one(-z), O0x=one(O1x), O0y=one(O1y), O1x=one(0.0), O1y=one(0.0)) as back:
        fr, _ = back.execute(torch.from_numpy(np.ascontiguousarray(u1.real)).to(_dev()))
        fi, _ = back.execute(torch.from_numpy(np.ascontiguousarray(u1.imag)).to(_dev()))
        torch.cuda.synchronize()
    rec = fr[0].cpu().numpy().astype(np.complex128) + 1j * fi[0].cpu().numpy().astype(np.complex128)
    err = np.linalg.norm(rec - u0) / np.linalg.norm(u0)
    assert err < 5e-6, f"round trip rel-L2 {err:.3e}"


# ---- depth stacks / focus moments ------------------------------------------
@pytest.mark.parametrize("N,V", [(256, 5), (1024, 6)])
def test_focus_moments_of_a_depth_stack(N, V):
    """sfd_execute_focus: per-view (sum I, sum I^2) fused into pass x, against the oracle's moments of
    form B; the intensity written next to them must be the ordinary one; NULL intensity allowed.
    Tolerance: fp32 intensities (rel 1e-6 each, random sign) summed over N^2 pixels, partial sums of
    16-32 pixels in fp32 -> 1e-5 relative is generous."""
    wl = W.depth_stack(N=N, V=V, z0=0.05, z1=0.11)
    holo = wl.hologram()
    h = torch.from_numpy(holo).to(_dev())
    with B.Plan(wl) as plan:
        mom, I = plan.execute_focus(h, intensity=True)
        mom2, none = plan.execute_focus(h)
        _, I_ref = plan.execute(h, field=False)
        torch.cuda.synchronize()
    assert none is None
    assert torch.equal(I, I_ref)
    _, I_or = O.reconstruct_views(holo, wl.lam, wl.p1, wl.p2, wl.z, wl.Ox, wl.Oy, form="B")
    want = O.focus_moments(I_or)
    for got in (mom.cpu().numpy(), mom2.cpu().numpy()):
        assert got.shape == (V, 2)
        assert np.max(np.abs(got / want - 1.0)) < 1e-5
    nv_gpu = O.normalised_variance(mom.cpu().numpy(), N * N)
    nv_or = O.normalised_variance(want, N * N)
    assert np.max(np.abs(nv_gpu - nv_or)) < 1e-4 * np.max(np.abs(nv_or)) + 1e-7
    assert int(np.argmax(nv_gpu)) == int(np.argmax(nv_or)) or np.isclose(np.max(nv_or), np.sort(nv_or)[-2], rtol=1e-4)


def test_focus_moments_delta_closed_form_on_gpu():
    """P4 on the CUDA path: a delta gives constant modulus, so sum I = N^2 c^2, sum I^2 = N^2 c^4."""
    N = 128
    u0 = np.zeros((N, N), dtype=np.float32)
    u0[40, 77] = 1.0
    zs = np.array([0.03, 0.06, -0.09])
    with B.Plan(N=N, lam=W.LAMBDA, p1=np.full(3, W.PITCH), p2=np.full(3, 2.0e-6), z=zs, Ox=np.zeros(3),
                Oy=np.zeros(3), in_dtype=B.SFD_F32) as plan:
        mom, _ = plan.execute_focus(torch.from_numpy(u0).to(_dev()))
        torch.cuda.synchronize()
    c2 = (W.PITCH ** 2 / (W.LAMBDA * np.abs(zs))) ** 2
    m = mom.cpu().numpy()
    assert np.allclose(m[:, 0], N * N * c2, rtol=2e-6)
    assert np.allclose(m[:, 1], N * N * c2 * c2, rtol=4e-6)


# ---- edges of the N = 1024 kernels -------------------------------------------------------------------
def test_1024_many_views_more_than_sms():
    """V = 150 views at N = 1024: more views than SMs, so the grid grows to V CTAs (a CTA's range then
    lies in at most two views) and CTAs run in waves; B, field and intensity are 1.2 + 1.2 + 0.6 GB.
    The oracle checks a sample of views; all views that share parameters must agree bit for bit."""
    V = 150
    rng = np.random.default_rng(77)
    base = W.config(2)
    pick = rng.integers(0, 4, V)                      # every view is one of config 2's four
    kw = dict(N=1024, lam=base.lam, p1=base.p1[pick], p2=base.p2[pick], z=base.z[pick], Ox=base.Ox[pick],
              Oy=base.Oy[pick], in_dtype=base.in_dtype)
    holo = base.hologram()
    with B.Plan(**kw) as plan:
        assert plan.uses_warp_kernels
        f, I = plan.execute(torch.from_numpy(holo).to(_dev()))
        torch.cuda.synchronize()
    want, _ = O.reconstruct_views(holo, base.lam, base.p1, base.p2, base.z, base.Ox, base.Oy, form="B")
    first = {int(k): int(np.flatnonzero(pick == k)[0]) for k in np.unique(pick)}
    for k, v0 in first.items():
        _assert_close(f[v0:v0 + 1].cpu().numpy(), want[k:k + 1], f"view {v0} (= config 2 view {k})")
    for v in (0, 1, 73, 148, 149):
        assert torch.equal(f[v], f[first[int(pick[v])]]), f"view {v} differs from its twin"
        assert torch.equal(I[v], I[first[int(pick[v])]])


def test_1024_unaligned_hologram_falls_back_to_generic_kernels():
    """The N = 1024 kernels read 8 bytes of a hologram row at once; a hologram that does not start on an
    8-byte boundary silently takes the generic kernels (same numbers to rounding)."""
    wl = W.config(1)
    holo = wl.hologram()
    buf = torch.empty(holo.size + 16, dtype=torch.uint8, device=_dev())
    off = 1 if buf.data_ptr() % 8 == 0 else (9 - buf.data_ptr() % 8)
    view = buf[off:off + holo.size].view(1024, 1024)
    assert view.data_ptr() % 8 != 0
    view.copy_(torch.from_numpy(holo))
    with B.Plan(wl) as plan:
        n0 = B.sfd_launch_count()
        f, _ = plan.execute(view)
        torch.cuda.synchronize()
        assert B.sfd_launch_count() - n0 == 2
    fB, _ = O.reconstruct_views(holo, wl.lam, wl.p1, wl.p2, wl.z, wl.Ox, wl.Oy, form="B")
    _assert_close(f.cpu().numpy(), fB, "unaligned hologram")


# ---- the N = 2048 warp kernels (four branches per line, sfd_warp2048.cuh) -----------------------------
@pytest.mark.parametrize("in_dtype", [B.SFD_U8, B.SFD_F32])
def test_2048_warp_and_generic_kernels_general_geometry(in_dtype):
    """N = 2048 has two kernel sets as well.  Both against the oracle on anisotropic, shifted views
    (z < 0 included), with marked samples in the last row/column and at the 1024 fold; then the 8-bit
    mode and the focus moments through the warp kernels."""
    N = 2048
    rng = np.random.default_rng(91)
    if in_dtype == B.SFD_F32:
        holo = rng.random((N, N), dtype=np.float32)
        holo[N - 1, N - 1] = 40.0
        holo[1024, 1023] = 25.0
    else:
        holo = rng.integers(0, 256, (N, N), dtype=np.uint8)
        holo[N - 1, N - 1] = 255
        holo[1024, 1023] = 0
    want = _general_oracle(holo, _GENERAL, "B")
    h = torch.from_numpy(holo).to(_dev())
    with B.Plan(N=N, lam=W.LAMBDA, in_dtype=in_dtype, **_GENERAL) as plan:
        assert plan.uses_warp_kernels
        f, I = plan.execute(h)
        mom, _ = plan.execute_focus(h)
        u8 = plan.execute_u8(h) if in_dtype == B.SFD_U8 else None
        plan.select_kernels(B.SFD_KERNELS_GENERIC)
        assert not plan.uses_warp_kernels
        fg, _ = plan.execute(h)
        torch.cuda.synchronize()
    _assert_close(f.cpu().numpy(), want, "N=2048 warp kernels field")
    _assert_close(I.cpu().numpy(), O.intensity(want), "N=2048 warp kernels intensity")
    _assert_close(fg.cpu().numpy(), want, "N=2048 generic kernels field")
    assert np.max(np.abs(mom.cpu().numpy() / O.focus_moments(O.intensity(want)) - 1.0)) < 1e-5
    if u8 is not None:
        for v in range(3):
            d = np.abs(u8[v].cpu().numpy().astype(int) - O.quantise_u8(O.intensity(want[v])).astype(int))
            assert d.max() <= 1 and (d > 0).mean() < 1e-3


@pytest.mark.parametrize("N,V,in_dtype,iters", [(1024, 4, B.SFD_U8, 120), (1024, 3, B.SFD_F32, 60),
                                                (2048, 2, B.SFD_U8, 40)])
def test_warp_kernels_bit_identical_under_concurrent_load(N, V, in_dtype, iters):
    """The warp kernels synchronise with named barriers, mbarriers, async bulk copies and programmatic
    dependent launch; compute-sanitizer is not available on the GPU pool, so hazards are hunted the other
    way: the field has no atomics in it and must come out bit-identical on every run while a second plan and
    a memory hog on another stream perturb the timing."""
    rng = np.random.default_rng(N + V)
    kw = dict(N=N, lam=W.LAMBDA, p1=np.full(V, W.PITCH), p2=rng.uniform(1e-6, 4.65e-6, V),
              z=rng.uniform(0.03, 0.1, V), Ox=rng.uniform(-3e-4, 3e-4, V), Oy=rng.uniform(-3e-4, 3e-4, V),
              in_dtype=in_dtype)
    host = (rng.integers(0, 256, (N, N), dtype=np.uint8) if in_dtype == B.SFD_U8
            else rng.random((N, N), dtype=np.float32))
    holo = torch.from_numpy(host).to(_dev())
    side = torch.cuda.Stream()
    hog = torch.empty(32 << 20, dtype=torch.float32, device=_dev())
    with B.Plan(**kw) as plan, B.Plan(**kw) as other:
        f0, I0 = plan.execute(holo)
        torch.cuda.synchronize()
        f0, I0 = f0.clone(), I0.clone()
        for it in range(iters):
            with torch.cuda.stream(side):
                if it % 3 == 0:
                    hog.add_(1.0)
                if it % 2 == 0:
                    other.execute(holo)
            f, I = plan.execute(holo)
            torch.cuda.synchronize()
            assert torch.equal(f, f0) and torch.equal(I, I0), f"run {it} differs from the first"


@pytest.mark.parametrize("in_dtype,V", [(B.SFD_U8, 4), (B.SFD_F32, 150)])
def test_512_warp_and_generic_kernels_agree_with_oracle(in_dtype, V):
    """N = 512 has two kernel sets: one warp per line (sfd_warp512.cuh: the padded line is exactly the
    1024-point warp FFT) and the generic Stockham kernels.  Both against the oracle, with marked samples
    in the last row/column; V = 150 > SMs makes CTA ranges straddle views; then the 8-bit mode and the
    focus moments through the warp kernels."""
    N = 512
    rng = np.random.default_rng(512 + V)
    base = W.config(2)
    pick = rng.integers(0, 4, V)
    if in_dtype == B.SFD_F32:
        holo = rng.random((N, N), dtype=np.float32)
        holo[N - 1, N - 1] = 40.0
        holo[0, N - 3] = 25.0
    else:
        holo = rng.integers(0, 256, (N, N), dtype=np.uint8)
        holo[N - 1, N - 1] = 255
        holo[0, N - 3] = 0
    kw = dict(N=N, lam=base.lam, p1=base.p1[pick], p2=base.p2[pick], z=base.z[pick] / 2, Ox=base.Ox[pick] / 2,
              Oy=base.Oy[pick] / 2, in_dtype=in_dtype)
    h = torch.from_numpy(holo).to(_dev())
    with B.Plan(**kw) as plan:
        assert plan.uses_warp_kernels
        f, I = plan.execute(h)
        mom, _ = plan.execute_focus(h)
        u8 = plan.execute_u8(h) if V <= 8 else None
        plan.select_kernels(B.SFD_KERNELS_GENERIC)
        assert not plan.uses_warp_kernels
        fg, _ = plan.execute(h)
        torch.cuda.synchronize()
    want, Iw = O.reconstruct_views(holo, base.lam, base.p1, base.p2, base.z / 2, base.Ox / 2, base.Oy / 2)
    first = {int(k): int(np.flatnonzero(pick == k)[0]) for k in np.unique(pick)}
    for k, v0 in first.items():
        _assert_close(f[v0:v0 + 1].cpu().numpy(), want[k:k + 1], f"N=512 warp kernels, view {v0}")
        _assert_close(I[v0:v0 + 1].cpu().numpy(), Iw[k:k + 1], f"N=512 warp kernels intensity, view {v0}")
        _assert_close(fg[v0:v0 + 1].cpu().numpy(), want[k:k + 1], f"N=512 generic kernels, view {v0}")
    for v in range(V):
        assert torch.equal(f[v], f[first[int(pick[v])]]), f"view {v} differs from its twin"
    m = mom.cpu().numpy()
    assert np.max(np.abs(m / O.focus_moments(Iw)[pick] - 1.0)) < 1e-5
    if u8 is not None:
        _u8_check(u8.cpu().numpy(), Iw[pick], "N=512 u8")


@pytest.mark.parametrize("N", [128, 1024])
def test_execute_is_capturable_in_a_cuda_graph(N):
    """sfd_execute only enqueues kernels on the caller's stream (no allocation, no synchronisation), so a
    frame loop can be captured in a CUDA graph; the programmatic-dependent-launch edges survive the capture.
    Replays must reproduce the directly executed field bit for bit."""
    wl = W.small_multiview(N=N, V=3, seed=11) if N < 1024 else W.config(2)
    holo = torch.from_numpy(wl.hologram()).to(_dev())
    with B.Plan(wl) as plan:
        f, I = plan.execute(holo)
        torch.cuda.synchronize()
        f0, I0 = f.clone(), I.clone()
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):                      # warm-up off the default stream, as torch asks
            plan.execute(holo, field=f, intensity=I)
        torch.cuda.current_stream().wait_stream(side)
        n0 = B.sfd_launch_count()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            for _ in range(4):
                plan.execute(holo, field=f, intensity=I)
        assert B.sfd_launch_count() - n0 == 8
        for _ in range(3):
            f.zero_()
            I.zero_()
            graph.replay()
            torch.cuda.synchronize()
            assert torch.equal(f, f0) and torch.equal(I, I0)


@pytest.mark.parametrize("col0", [16, 8])
def test_2048_uint8_window_alignment(col0):
    """The N = 2048 column kernel reads 16 bytes of a uint8 hologram row at once (the 16 columns of four
    units).  A window of a 2 080-wide frame that starts on a 16-byte boundary runs the warp kernels with
    a row stride that is not N; one that starts on an 8-byte boundary only silently takes the generic
    pass y (a 16-byte load there would fault).  Both against the oracle on the oracle's own crop."""
    N, stride, row0 = 2048, 2080, 1
    rng = np.random.default_rng(col0)
    frame = rng.integers(0, 256, (N + 2, stride), dtype=np.uint8)
    g = {k: v[:2] for k, v in _GENERAL.items()}
    win = np.ascontiguousarray(O.crop_window(frame, N, N, row0, col0))
    fr = torch.from_numpy(frame).to(_dev())
    assert fr.data_ptr() % 16 == 0
    with B.Plan(N=N, lam=W.LAMBDA, in_dtype=B.SFD_U8, **g) as plan:
        plan.set_input_window((N + 2, stride), row0, col0)
        f, _ = plan.execute(fr)
        torch.cuda.synchronize()
    _assert_close(f.cpu().numpy(), _general_oracle(win, g, "B"), f"2048 window at column {col0}")


# ---- round 2: tight regression bound, P5 on the GPU, rectangular grids, frame windows, live updates ------
REG_L2, REG_MAX = 2e-6, 1e-5   # measured 1.5e-7 .. 3.5e-7 / 4e-7 .. 1.1e-6: a 10x loss of precision turns this red


def _assert_tight(got, want, what):
    for v in range(want.shape[0]):
        d = got[v].astype(want.dtype) - want[v]
        l2 = np.linalg.norm(d) / np.linalg.norm(want[v])
        mx = np.max(np.abs(d)) / np.max(np.abs(want[v]))
        assert l2 <= REG_L2 and mx <= REG_MAX, f"{what} view {v}: rel-L2 {l2:.3e}, max {mx:.3e} (regression bound)"


def test_precision_regression_bound_config2():
    """The north_star tolerance (2e-5 / 1e-4) is 70x above what the fp32 path delivers; this bound sits 8x
    above the measured error so that a loss of precision (a table rounded twice, a float32 phase) fails."""
    wl = W.config(2)
    holo, f, I = _run(wl)
    fB, IB = O.reconstruct_views(holo, wl.lam, wl.p1, wl.p2, wl.z, wl.Ox, wl.Oy, form="B")
    _assert_tight(f, fB, "config 2 field")
    _assert_tight(I, IB, "config 2 intensity")


@pytest.mark.parametrize("N,p2,z,Ox,Oy", [(256, 3.1e-6, 0.03, 0.1e-3, -0.05e-3), (1024, 2.0e-6, -0.08, 0.0, 0.2e-3)])
def test_gaussian_beam_closed_form_on_gpu_output(N, p2, z, Ox, Oy):
    """Pin P5 applied to the CUDA path: u0 = exp(-r^2/w0^2) reconstructs to the paraxial Gaussian beam
    exp(ikz)/(1 + i z/zR) exp(-r1^2/(w0^2 (1 + i z/zR))) with no fudge factor (reading 9): absolute scale,
    arbitrary pitch, shift and sign of z.  The beam is well inside the window, so the sampled sum equals
    the integral to ~1e-7; tolerance = the north_star's."""
    lam, p1, w0 = W.LAMBDA, W.PITCH, (100e-6 if N == 256 else 300e-6)
    x0 = (np.arange(N) - N / 2) * p1
    u0 = np.exp(-(x0[None, :] ** 2 + x0[:, None] ** 2) / w0 ** 2).astype(np.float32)
    wl = W.Workload("gauss", N, lam, np.array([p1]), np.array([p2]), np.array([z]), np.array([Ox]),
                    np.array([Oy]), W.IN_F32)
    _, f, _ = _run(wl, u0)
    zR = np.pi * w0 ** 2 / lam
    q = 1 + 1j * z / zR
    x1 = (np.arange(N) - N / 2) * p2 + Ox
    y1 = (np.arange(N) - N / 2) * p2 + Oy
    zl = z / lam
    want = np.exp(2j * np.pi * (zl - np.rint(zl))) / q * np.exp(-(x1[None, :] ** 2 + y1[:, None] ** 2) / (w0 ** 2 * q))
    _assert_close(f, want[None], "Gaussian beam")


def _rect_oracle(holo, g, form="B"):
    fn = {"B": O.bluestein_fft, "M": O.separable_matrices}[form]
    u0 = O.input_scale(holo)
    return np.stack([fn(u0, W.LAMBDA, g["z"][v], (g["p1x"][v], g["p1y"][v]), (g["p2x"][v], g["p2y"][v]),
                        O1=(g["O1x"][v], g["O1y"][v]), O0=(g["O0x"][v], g["O0y"][v]))
                     for v in range(len(g["z"]))])


@pytest.mark.parametrize("Nx,Ny,in_dtype,mask", [
    (128, 64, B.SFD_F32, 0),        # generic kernels on both axes, two radix schedules
    (64, 512, B.SFD_U8, 1),         # pass y = k_cols_512 over 64 columns, pass x generic
    (512, 128, B.SFD_F32, 2),       # pass y generic, pass x = k_rows_512 over 128 rows
    (256, 1024, B.SFD_U8, 1),       # pass y = k_cols_1024 over 256 columns, pass x generic
    (1024, 512, B.SFD_U8, 3),       # pass y = k_cols_512 over 1024 columns, pass x = k_rows_1024 over 512 rows
    (512, 2048, B.SFD_F32, 3),      # k_cols_2048 + k_rows_512
    (2048, 1024, B.SFD_F32, 3),     # k_cols_1024 + k_rows_2048
    (1024, 2048, B.SFD_U8, 3),      # k_cols_2048 + k_rows_1024
])
def test_rectangular_grids_against_oracle(Nx, Ny, in_dtype, mask):
    """Row f3: N_x != N_y (Eq.(2)-(3) carry both, L58-62).  Each axis picks its kernels by its own length;
    anisotropic pitches and shifted windows on top; against the oracle's rectangular path (pinned on 12 x 20
    against the double sum) with marked samples in the last row and column."""
    rng = np.random.default_rng(Nx + 3 * Ny)
    if in_dtype == B.SFD_F32:
        holo = rng.random((Ny, Nx), dtype=np.float32)
        holo[Ny - 1, Nx - 1] = 30.0
        holo[0, Nx - 3] = 20.0
    else:
        holo = rng.integers(0, 256, (Ny, Nx), dtype=np.uint8)
        holo[Ny - 1, Nx - 1] = 255
        holo[0, Nx - 3] = 0
    g = {k: v[:2] for k, v in _GENERAL.items()}
    with B.Plan(Nx=Nx, Ny=Ny, lam=W.LAMBDA, in_dtype=in_dtype, **g) as plan:
        assert plan.warp_kernel_mask == mask
        assert (B.sfd_plan_get_nx(plan.handle), B.sfd_plan_get_ny(plan.handle)) == (Nx, Ny)
        f, I = plan.execute(torch.from_numpy(holo).to(_dev()))
        u8 = plan.execute_u8(torch.from_numpy(holo).to(_dev())) if in_dtype == B.SFD_U8 else None
        mom, _ = plan.execute_focus(torch.from_numpy(holo).to(_dev()))
        torch.cuda.synchronize()
    assert tuple(f.shape) == (2, Ny, Nx)
    want = _rect_oracle(holo, g, "B")
    _assert_close(f.cpu().numpy(), want, f"{Nx}x{Ny} field")
    _assert_close(I.cpu().numpy(), O.intensity(want), f"{Nx}x{Ny} intensity")
    if Nx * Ny <= 256 * 1024:
        _assert_close(f.cpu().numpy(), _rect_oracle(holo, g, "M"), f"{Nx}x{Ny} field vs form M")
    assert np.max(np.abs(mom.cpu().numpy() / O.focus_moments(O.intensity(want)) - 1.0)) < 1e-5
    if u8 is not None:
        _u8_check(u8.cpu().numpy(), O.intensity(want), f"{Nx}x{Ny} u8")


@pytest.mark.parametrize("seed", range(10))
def test_random_plans_against_oracle(seed):
    """Seeded sweep over what a plan can be: grid sides drawn from 64 .. 1024 independently (every pairing of
    the generic, N = 512 and N = 1024 kernels comes up), 1 - 5 views, uint8 or float32 input, pitches,
    distances of either sign and window shifts drawn per view.  Field and intensity against form B."""
    rng = np.random.default_rng(1000 + seed)
    Nx, Ny = (int(2 ** rng.integers(6, 11)) for _ in range(2))
    V = int(rng.integers(1, 6))
    in_dtype = B.SFD_U8 if rng.random() < 0.5 else B.SFD_F32
    g = dict(p1x=rng.uniform(3e-6, 7e-6, V), p1y=rng.uniform(3e-6, 7e-6, V),
             p2x=rng.uniform(0.8e-6, 6e-6, V), p2y=rng.uniform(0.8e-6, 6e-6, V),
             z=rng.uniform(0.03, 0.15, V) * rng.choice([-1.0, 1.0], V),
             O0x=rng.uniform(-3e-4, 3e-4, V), O0y=rng.uniform(-3e-4, 3e-4, V),
             O1x=rng.uniform(-8e-4, 8e-4, V), O1y=rng.uniform(-8e-4, 8e-4, V))
    holo = (rng.integers(0, 256, (Ny, Nx), dtype=np.uint8) if in_dtype == B.SFD_U8
            else rng.random((Ny, Nx), dtype=np.float32))
    with B.Plan(Nx=Nx, Ny=Ny, lam=W.LAMBDA, in_dtype=in_dtype, **g) as plan:
        f, I = plan.execute(torch.from_numpy(holo).to(_dev()))
        torch.cuda.synchronize()
    want = _rect_oracle(holo, g, "B")
    what = f"seed {seed}: {Nx}x{Ny}, {V} views, dtype {in_dtype}"
    _assert_close(f.cpu().numpy(), want, what + " field")
    _assert_close(I.cpu().numpy(), O.intensity(want), what + " intensity")


@pytest.mark.parametrize("col0,row0,warp", [(168, 0, True), (165, 0, False), (8, 3, True)])
def test_ccd_frame_window_read_in_place(col0, row0, warp):
    """Row f3 / PAPER.md L42 (reading 13): the plan reads its 1024 x 1024 window out of a 1 360-wide 8-bit
    frame in place.  col0 = 168 is the centred crop (8-byte aligned: warp kernels); 165 is unaligned and
    takes the generic kernels; (row0, col0) = (3, 8) is a window off centre whose physical shift goes into
    O_0.  Against the oracle on the oracle's own crop."""
    rows, stride, N = 1024 + 4, 1360, 1024
    rng = np.random.default_rng(42)
    frame = rng.integers(0, 256, (rows, stride), dtype=np.uint8)
    base = W.config(2)
    dc, dr = col0 - (stride - N) // 2, row0 - (rows - N) // 2
    V = 2
    kw = dict(N=N, lam=base.lam, in_dtype=B.SFD_U8, p1x=base.p1[:V], p1y=base.p1[:V], p2x=base.p2[2:], p2y=base.p2[2:],
              z=base.z[2:], O0x=np.full(V, dc * W.PITCH), O0y=np.full(V, dr * W.PITCH), O1x=base.Ox[2:], O1y=base.Oy[2:])
    fr = torch.from_numpy(frame).to(_dev())
    with B.Plan(**kw) as plan:
        plan.set_input_window((rows, stride), row0, col0)
        n0 = B.sfd_launch_count()
        f, I = plan.execute(fr)
        u8 = plan.execute_u8(fr)
        torch.cuda.synchronize()
        assert B.sfd_launch_count() - n0 == 5
        plan.set_input_window(None, 0, 0)          # back to dense holograms: same numbers from a copy
        win = np.ascontiguousarray(O.crop_window(frame, N, N, row0, col0))
        f2, _ = plan.execute(torch.from_numpy(win).to(_dev()))
        torch.cuda.synchronize()
        if warp:
            assert torch.equal(f, f2)
    want = np.stack([O.bluestein_fft(O.input_scale(win), base.lam, kw["z"][v], W.PITCH, kw["p2x"][v],
                                     O1=(kw["O1x"][v], kw["O1y"][v]), O0=(kw["O0x"][v], kw["O0y"][v]))
                     for v in range(V)])
    _assert_close(f.cpu().numpy(), want, "window field")
    _assert_close(f2.cpu().numpy(), want, "dense copy field")
    _u8_check(u8.cpu().numpy(), O.intensity(want), "window u8")
    with B.Plan(**kw) as plan:
        with pytest.raises(B.SfdError):
            B.sfd_plan_set_input_window(plan.handle, 1000, 0, 0)     # stride shorter than a window row


@pytest.mark.parametrize("N", [256, 1024])
def test_async_view_updates_are_ordered_by_the_stream(N):
    """Row f1: update -> execute -> update -> execute on one NON-BLOCKING stream without any host
    synchronisation in between; each execute must see exactly the tables of the update before it (the
    kernels read their tables in the prologue, before griddepcontrol.wait).  Then the blocking update
    followed at once by an execute on the non-blocking stream and by sfd_stream_run."""
    wl = W.config(2) if N == 1024 else W.small_multiview(N=N, V=3, seed=5)
    holo = wl.hologram()
    dev = _dev()
    h = torch.from_numpy(holo).to(dev)
    steps = [(1, W.PITCH, 1.7e-6, -0.033, 0.05e-3, 0.02e-3), (0, W.PITCH, 3.3e-6, 0.071, -0.2e-3, 0.1e-3),
             (1, W.PITCH, 2.2e-6, 0.052, 0.0, -0.3e-3)]
    s = torch.cuda.Stream()          # torch side streams are cudaStreamNonBlocking
    outs = []
    with B.Plan(wl) as plan:
        torch.cuda.synchronize()
        with torch.cuda.stream(s):
            for (v, p1, p2, z, Ox, Oy) in steps:
                plan.update_view_async(v, p1, p2, z, Ox, Oy, stream=s)
                f, _ = plan.execute(h, stream=s)
                outs.append(f)
        s.synchronize()
        assert 0.0 < plan.last_update_host_ms < 200.0
        p2_, z_, Ox_, Oy_ = wl.p2.copy(), wl.z.copy(), wl.Ox.copy(), wl.Oy.copy()
        for (v, p1, p2, z, Ox, Oy), f in zip(steps, outs):
            p2_[v], z_[v], Ox_[v], Oy_[v] = p2, z, Ox, Oy
            want, _ = O.reconstruct_views(holo, wl.lam, wl.p1, p2_, z_, Ox_, Oy_)
            _assert_close(f.cpu().numpy(), want, f"after async update of view {v}")
        # blocking update, then immediately a non-blocking stream and the internal streams of stream_run
        plan.update_view(0, W.PITCH, 4.0e-6, 0.09, 0.1e-3, 0.1e-3)
        with torch.cuda.stream(s):
            f, _ = plan.execute(h, stream=s)
        pinned = torch.from_numpy(holo[None]).pin_memory()
        out, _ = plan.stream_run(pinned)
        s.synchronize()
        p2_[0], z_[0], Ox_[0], Oy_[0] = 4.0e-6, 0.09, 0.1e-3, 0.1e-3
        want, Iw = O.reconstruct_views(holo, wl.lam, wl.p1, p2_, z_, Ox_, Oy_)
        _assert_close(f.cpu().numpy(), want, "after blocking update")
        _u8_check(out[0].numpy(), Iw, "stream_run after blocking update")


def test_more_updates_in_flight_than_staging_slots():
    """Eight async updates back to back (the staging ring has four slots): the last one wins."""
    wl = W.small_multiview(N=128, V=2, seed=8)
    holo = wl.hologram()
    h = torch.from_numpy(holo).to(_dev())
    with B.Plan(wl) as plan:
        for i in range(8):
            plan.update_view_async(1, W.PITCH, (1.5 + 0.2 * i) * 1e-6, 0.03 + 0.005 * i, 1e-5 * i, 0.0)
        f, _ = plan.execute(h)
        torch.cuda.synchronize()
    p2, z, Ox, Oy = wl.p2.copy(), wl.z.copy(), wl.Ox.copy(), wl.Oy.copy()
    p2[1], z[1], Ox[1], Oy[1] = 2.9e-6, 0.065, 7e-5, 0.0
    want, _ = O.reconstruct_views(holo, wl.lam, wl.p1, p2, z, Ox, Oy)
    _assert_close(f.cpu().numpy(), want, "after 8 queued updates")


def test_plans_on_two_devices_in_one_process():
    """Per-device initialisation (the dynamic shared-memory opt-in is per device) and the device guard:
    a plan made on cuda:1 executes correctly while cuda:0 is current.  Needs two visible GPUs."""
    if torch.cuda.device_count() < 2:
        pytest.skip("one visible GPU")
    wl = W.config(1)
    holo = wl.hologram()
    want, _ = O.reconstruct_views(holo, wl.lam, wl.p1, wl.p2, wl.z, wl.Ox, wl.Oy)
    plans = []
    for i in (0, 1):
        with torch.cuda.device(i):
            plans.append(B.Plan(wl))
            assert B.sfd_plan_get_device(plans[-1].handle) == i
    torch.cuda.set_device(0)
    for i, plan in enumerate(plans):
        h = torch.from_numpy(holo).to(f"cuda:{i}")
        f = torch.empty((1, 1024, 1024), dtype=torch.complex64, device=f"cuda:{i}")
        B.sfd_execute(plan.handle, h, f, None, torch.cuda.current_stream(i))
        torch.cuda.synchronize(i)
        _assert_close(f.cpu().numpy(), want, f"plan on cuda:{i} with cuda:0 current")
        plan.close()


def test_measure_pipes_reports_sane_numbers():
    tf, cyc_a, cyc_b, ghz = B.sfd_measure_pipes()
    assert 40.0 < tf < 90.0            # 148 SMs x 128 lanes x 2 x ~1.9 GHz = 72 nominal
    assert 300.0 < cyc_a < 700.0 and 380.0 < cyc_b < 900.0
    assert 1.0 < ghz < 2.3


def test_measure_memory_pipes_reports_sane_numbers():
    smem, tm1, tm2, lat = B.sfd_measure_memory_pipes()
    assert 60.0 < smem <= 130.0          # 128 B/clk and SM is the architectural rate
    assert 40.0 < tm1 <= 300.0 and tm1 * 0.9 < tm2 <= 400.0   # measured 148 / 215 B/clk and sub-partition
    assert 10.0 < lat < 200.0
