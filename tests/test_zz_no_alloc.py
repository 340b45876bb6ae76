"""The allocation-free entry point sfd_quantise_u8_static (include/sfd.h): step (xi) / reading 15 for callers
that may not call cudaMalloc.  Its per-view maxima live in a static device array inside the library, shared by
all calls and never cleared between them except by the calls themselves.

This file sorts last on purpose (pytest collects test files alphabetically and the suite runs with ``-x``), and
its test must pass both alone in a fresh process - nothing else has created a plan or touched the GPU - and
after every other test."""
import numpy as np
import pytest
import torch

from oracle import shifted_fresnel as O
from paper_1001_4309_b200 import build as sfd_build
from paper_1001_4309_b200 import workloads as W

sfd_build.build()
from paper_1001_4309_b200 import binding as B  # noqa: E402


@pytest.mark.gpu
def test_static_quantise_matches_execute_u8_twice_in_a_row():
    """Two calls in a row on one stream against the existing path (sfd_execute_u8 of a plan) on the same
    holograms.  The first frame is the bright one: if the second call did not clear the array, the maxima the
    first call left behind would darken every view of the second.  Tolerance: the 8-bit images of the existing
    path are held to <= 1 LSB at isolated pixels against the oracle (tests/test_gpu_parity.py); the two GPU
    paths share the intensity kernels and the quantisation kernel, so they are compared the same way and come
    out equal."""
    assert torch.cuda.is_available(), "GPU tests need a CUDA device (no CPU fallback exists)"
    dev = torch.device("cuda:0")
    wl = W.small_multiview(N=256, V=3, seed=3)
    bright = wl.hologram()
    dim = (bright // 3).astype(np.uint8)                   # a different, darker frame
    V, N = wl.n_views, wl.N
    # the output buffers of the new entry point exist before the calls: nothing is allocated in between
    out = [torch.full((V, N, N), 7, dtype=torch.uint8, device=dev) for _ in range(2)]
    with B.Plan(wl) as plan:
        inten, want = [], []
        for frame in (bright, dim):
            h = torch.from_numpy(frame).to(dev)
            _, I = plan.execute(h, field=False)
            inten.append(I)
            want.append(plan.execute_u8(h))
        torch.cuda.synchronize()
        reserved = torch.cuda.memory_reserved(dev)
        n0 = B.sfd_launch_count()
        for k in range(2):                                 # back to back, no synchronisation in between
            B.sfd_quantise_u8_static(inten[k], V, N * N, out[k])
        torch.cuda.synchronize()
        assert B.sfd_launch_count() - n0 == 4              # two kernels per call
        assert torch.cuda.memory_reserved(dev) == reserved
    for k in range(2):
        got, ref = out[k].cpu().numpy().astype(int), want[k].cpu().numpy().astype(int)
        d = np.abs(got - ref)
        assert d.max() <= 1 and (d > 0).mean() < 1e-3, f"call {k}: {d.max()} LSB, {(d > 0).mean():.2e} of pixels"
        for v in range(V):
            assert got[v].max() == 255                     # every view normalised by its OWN maximum
        # and against the oracle's quantisation of the same float32 intensities (ties aside)
        Ik = inten[k].cpu().numpy().astype(np.float64)
        q = np.stack([O.quantise_u8(Ik[v]) for v in range(V)]).astype(int)    # the oracle normalises one view
        assert np.abs(got - q).max() <= 1 and (got != q).mean() < 1e-3


@pytest.mark.gpu
def test_static_quantise_limits_and_zero_view():
    dev = torch.device("cuda:0")
    I = torch.rand(2, 64, dtype=torch.float32, device=dev)
    I[1].zero_()                                           # an all-zero view gives zeros
    out = torch.full((2, 64), 9, dtype=torch.uint8, device=dev)
    B.sfd_quantise_u8_static(I, 2, 64, out)
    torch.cuda.synchronize()
    assert int(out[0].max()) == 255 and int(out[1].max()) == 0
    too_many = B.sfd_static_max_views() + 1
    big = torch.ones(too_many, 4, dtype=torch.float32, device=dev)
    with pytest.raises(B.SfdError) as e:
        B.sfd_quantise_u8_static(big, too_many, 4, torch.empty(too_many, 4, dtype=torch.uint8, device=dev))
    assert e.value.code == B.SFD_EUNSUPPORTED and "SFD_STATIC_MAX_VIEWS" in str(e.value)
    B.sfd_quantise_u8_static(big, too_many - 1, 4, torch.empty(too_many, 4, dtype=torch.uint8, device=dev))
    torch.cuda.synchronize()


def test_static_quantise_argument_checks_need_no_gpu():
    """Argument errors are reported before any CUDA call."""
    assert B.sfd_static_max_views() == 1024
    lib = B._lib
    assert lib.sfd_quantise_u8_static(None, 1, 64, None, None) == B.SFD_EINVAL
    assert lib.sfd_quantise_u8_static(4096, 0, 64, 4096, None) == B.SFD_EINVAL
    assert lib.sfd_quantise_u8_static(4096, 1, 66, 4096, None) == B.SFD_EINVAL        # not a multiple of 4
    assert lib.sfd_quantise_u8_static(4100, 1, 64, 4096, None) == B.SFD_EINVAL        # input not 16-byte aligned
    assert lib.sfd_quantise_u8_static(4096, 1025, 64, 4096, None) == B.SFD_EUNSUPPORTED
    assert "1025" in B.sfd_static_last_error()
