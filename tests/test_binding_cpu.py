"""CPU-only checks of the C-ABI library: it loads, exports every symbol include/sfd.h declares,
rejects bad arguments before touching CUDA, fails loudly without a GPU, and its float64 host table
builder (Eq. 2-4) agrees with the oracle's independently written tables."""
import ctypes

import numpy as np
import pytest
import torch

from oracle import shifted_fresnel as O
from paper_1001_4309_b200 import build as sfd_build
from paper_1001_4309_b200 import workloads as W

sfd_build.build()
from paper_1001_4309_b200 import binding as B  # noqa: E402


def test_library_exports_every_declared_symbol():
    names = B.declared_symbols()
    assert len(names) >= 17 and "sfd_plan_create" in names and "sfd_stream_run" in names
    lib = ctypes.CDLL(str(B.LIB_PATH))
    for n in names:
        assert hasattr(lib, n), f"libsfd.so does not export {n}"
    # and the binding has a function of the same name for each
    for n in names:
        assert callable(getattr(B, n)), f"binding lacks {n}"


def test_version_and_error_strings():
    assert "sm_100a" in B.sfd_version()
    assert B.sfd_error_string(0) == "success"
    assert "invalid" in B.sfd_error_string(B.SFD_EINVAL)
    assert B.sfd_launch_count() == 0 or torch.cuda.is_available()


@pytest.mark.parametrize("N", [100, 32, 4096, 1000])
def test_sizes_without_kernels_are_unsupported_not_invalid(N):
    """A grid side this build has no kernels for is a valid request that is not implemented."""
    with pytest.raises(B.SfdError) as e:
        B.sfd_plan_create(N, 1, W.LAMBDA, [W.PITCH], [W.PITCH], [0.05], [0.0], [0.0], B.SFD_F32)
    assert e.value.code == B.SFD_EUNSUPPORTED
    one = [W.PITCH]
    with pytest.raises(B.SfdError) as e:
        B.sfd_plan_create_rect(64, N, 1, W.LAMBDA, one, one, one, one, [0.05], [0.0], [0.0], [0.0], [0.0],
                               B.SFD_F32)
    assert e.value.code == B.SFD_EUNSUPPORTED


@pytest.mark.parametrize("bad", [
    dict(N=0), dict(N=-64), dict(n_views=0), dict(lam=0.0), dict(lam=-1e-6),
    dict(p1=[0.0]), dict(p2=[-1e-6]), dict(z=[0.0]), dict(z=[float("nan")]), dict(z=[float("inf")]),
    dict(Ox=[float("nan")]), dict(in_dtype=7),
])
def test_plan_create_rejects_bad_arguments(bad):
    kw = dict(N=64, n_views=1, lam=W.LAMBDA, p1=[W.PITCH], p2=[W.PITCH], z=[0.05], Ox=[0.0],
              Oy=[0.0], in_dtype=B.SFD_F32)
    kw.update(bad)
    with pytest.raises(B.SfdError) as e:
        B.sfd_plan_create(kw["N"], kw["n_views"], kw["lam"], kw["p1"], kw["p2"], kw["z"], kw["Ox"],
                          kw["Oy"], kw["in_dtype"])
    assert e.value.code == B.SFD_EINVAL


def test_null_arguments_are_einval():
    assert B._lib.sfd_execute(None, None, None, None, None) == B.SFD_EINVAL
    assert B._lib.sfd_execute_u8(None, None, None, None) == B.SFD_EINVAL
    assert B._lib.sfd_stream_run(None, None, 1, None, None) == B.SFD_EINVAL
    assert B._lib.sfd_plan_destroy(None) == B.SFD_OK
    assert B._lib.sfd_plan_create(None, 64, 1, 1e-6, None, None, None, None, None, 0) == B.SFD_EINVAL


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_no_gpu_fails_loudly_not_silently():
    """The product has no CPU fallback: without a device a valid plan request is SFD_ECUDA."""
    with pytest.raises(B.SfdError) as e:
        B.sfd_plan_create(64, 1, W.LAMBDA, [W.PITCH], [W.PITCH], [0.05], [0.0], [0.0], B.SFD_F32)
    assert e.value.code == B.SFD_ECUDA
    assert "cuda" in str(e.value).lower()


@pytest.mark.parametrize("N,p2,z,off", [
    (64, 4.65e-6, 0.05, 0.0),
    (256, 2.0e-6, 0.08, 0.4e-3),
    (1024, 1.0e-6, 0.08, -0.6e-3),
    (1024, 4.65e-6, -0.06, 0.0),
    (2048, 4.65e-6, 0.02, 0.9e-3),       # aliased chirp, S*N = 3.5 (reading 16)
])
def test_host_tables_match_oracle_tables(N, p2, z, off):
    """Host logic pin: the plan's float64 tables (own C++ code, long double phases, own FFT) against
    the oracle's Eq.(2)-(4) factors (NumPy, scipy.fft)."""
    lam, p1 = W.LAMBDA, W.PITCH
    pre, post, H = B.sfd_host_tables(N, lam, p1, p2, z, off)
    pre_o = O.pre_chirp(N, lam, z, p1, p2, 0.0, off)
    post_o = O.post_chirp(N, lam, z, p1, p2, 0.0, off)
    h = O.chirp_kernel(N, 2 * N, O.scale_factor(lam, z, p1, p2))
    H_o = np.fft.fft(h) / (2 * N)
    assert np.max(np.abs(pre - pre_o)) < 2e-11
    assert np.max(np.abs(post - post_o)) < 2e-11
    assert np.max(np.abs(H - H_o)) < 1e-12 * max(1.0, np.max(np.abs(H_o)) * 2 * N)


def test_host_tables_reject_bad_arguments():
    with pytest.raises(B.SfdError):
        B.sfd_host_tables(100, W.LAMBDA, W.PITCH, W.PITCH, 0.05, 0.0)
    with pytest.raises(B.SfdError):
        B.sfd_host_tables(64, W.LAMBDA, W.PITCH, W.PITCH, 0.0, 0.0)


@pytest.mark.parametrize("N,p1,p2,z,off0,off", [
    (64, 4.65e-6, 3.0e-6, 0.05, 0.1e-3, -0.2e-3),
    (1024, 6.0e-6, 1.5e-6, 0.08, -0.3e-3, 0.5e-3),
    (1024, 4.65e-6, 4.65e-6, -0.07, 0.25e-3, 0.0),
])
def test_host_tables_general_match_oracle_tables(N, p1, p2, z, off0, off):
    """General geometry (row f3): hologram-window offset O_0 of Eq.(2)-(3), L58-62, and a hologram
    pitch different from the default; the plan's float64 tables against the oracle's factors."""
    lam = W.LAMBDA
    pre, post, H = B.sfd_host_tables_general(N, lam, p1, p2, z, off0, off)
    assert np.max(np.abs(pre - O.pre_chirp(N, lam, z, p1, p2, off0, off))) < 2e-11
    assert np.max(np.abs(post - O.post_chirp(N, lam, z, p1, p2, off0, off))) < 2e-11
    H_o = np.fft.fft(O.chirp_kernel(N, 2 * N, O.scale_factor(lam, z, p1, p2))) / (2 * N)
    assert np.max(np.abs(H - H_o)) < 1e-12 * max(1.0, np.max(np.abs(H_o)) * 2 * N)
    # off0 = 0 is the square entry point
    a, b, c = B.sfd_host_tables_general(N, lam, p1, p2, z, 0.0, off)
    a2, b2, c2 = B.sfd_host_tables(N, lam, p1, p2, z, off)
    assert np.array_equal(a, a2) and np.array_equal(b, b2) and np.array_equal(c, c2)


@pytest.mark.parametrize("bad", [
    dict(N=0), dict(n_views=0), dict(p1y=[0.0]), dict(p2x=[float("nan")]), dict(z=[0.0]),
    dict(O0x=[float("inf")]), dict(O1y=[float("nan")]), dict(in_dtype=-1),
])
def test_general_plan_create_rejects_bad_arguments(bad):
    kw = dict(N=64, n_views=1, lam=W.LAMBDA, p1x=[W.PITCH], p1y=[W.PITCH], p2x=[2e-6], p2y=[3e-6],
              z=[0.05], O0x=[0.0], O0y=[0.0], O1x=[0.0], O1y=[0.0], in_dtype=B.SFD_F32)
    kw.update(bad)
    with pytest.raises(B.SfdError) as e:
        B.sfd_plan_create_general(kw["N"], kw["n_views"], kw["lam"], kw["p1x"], kw["p1y"], kw["p2x"],
                                  kw["p2y"], kw["z"], kw["O0x"], kw["O0y"], kw["O1x"], kw["O1y"],
                                  kw["in_dtype"])
    assert e.value.code == B.SFD_EINVAL


def test_new_entry_points_reject_null():
    assert B._lib.sfd_execute_focus(None, None, None, None, None) == B.SFD_EINVAL
    assert B._lib.sfd_plan_update_view_general(None, 0, 1e-6, 1e-6, 1e-6, 1e-6, 0.1, 0.0, 0.0, 0.0,
                                               0.0) == B.SFD_EINVAL
    assert B._lib.sfd_plan_create_general(None, 64, 1, 1e-6, *([None] * 9), 0) == B.SFD_EINVAL
    with pytest.raises(B.SfdError):
        B.sfd_host_tables_general(100, W.LAMBDA, W.PITCH, W.PITCH, 0.05, 0.0, 0.0)


def test_round2_entry_points_reject_null_and_bad_arguments():
    assert B._lib.sfd_plan_create_rect(None, 64, 128, 1, 1e-6, *([None] * 9), 0) == B.SFD_EINVAL
    assert B._lib.sfd_plan_set_input_window(None, 0, 0, 0) == B.SFD_EINVAL
    assert B._lib.sfd_plan_update_view_async(None, 0, 1e-6, 1e-6, 0.1, 0.0, 0.0, None) == B.SFD_EINVAL
    assert B._lib.sfd_plan_update_view_general_async(None, 0, *([1e-6] * 4), 0.1, 0.0, 0.0, 0.0, 0.0,
                                                     None) == B.SFD_EINVAL
    assert B._lib.sfd_plan_last_update_host_ms(None) == -1.0
    assert B._lib.sfd_plan_get_nx(None) == B.SFD_EINVAL and B._lib.sfd_plan_get_ny(None) == B.SFD_EINVAL
    assert B._lib.sfd_plan_get_device(None) == B.SFD_EINVAL
    assert B._lib.sfd_measure_pipes(None) == B.SFD_EINVAL
    assert B._lib.sfd_measure_memory_pipes(None) == B.SFD_EINVAL
    assert B._lib.sfd_host_dft32(None, None, 0, 0) == B.SFD_EINVAL
    with pytest.raises(B.SfdError):
        B.sfd_host_dft32(np.zeros(32, np.complex64), lane=32)


def test_binding_loads_only_the_in_tree_library(monkeypatch):
    """No environment override: the product imports paper_1001_4309_b200/libsfd.so and nothing else."""
    assert B.LIB_PATH.name == "libsfd.so" and B.LIB_PATH.parent.name == "paper_1001_4309_b200"
    import inspect
    assert "environ" not in inspect.getsource(B)


@pytest.mark.parametrize("lane", [0, 1, 13, 31])
def test_host_butterflies_equal_the_dft(lane):
    """Host logic pin of the register butterflies the warp kernels run (sfd_dft32.cuh: FMA-formulated
    radix-2 stages, sign tracking, inter-stage twiddles folded into stage B): stepped on the CPU they
    must equal the plain 32-point DFT (numpy) resp. the DFT of the twiddled input, to fp32 rounding."""
    rng = np.random.default_rng(100 + lane)
    x = (rng.standard_normal(32) + 1j * rng.standard_normal(32)).astype(np.complex64)
    r = np.arange(32)
    a = B.sfd_host_dft32(x, lane, twiddled=False)
    want = np.fft.fft(x.astype(np.complex128))
    assert np.linalg.norm(a - want) / np.linalg.norm(want) < 3e-7
    b = B.sfd_host_dft32(x, lane, twiddled=True)
    want = np.fft.fft(x.astype(np.complex128) * np.exp(-2j * np.pi * r * lane / 1024))
    assert np.linalg.norm(b - want) / np.linalg.norm(want) < 3e-7
    # a delta at input r gives the r-th row of the DFT matrix: every twiddle index is exercised
    for r0 in (1, 5, 16, 31):
        e = np.zeros(32, np.complex64)
        e[r0] = 1
        got = B.sfd_host_dft32(e, lane, twiddled=True)
        assert np.max(np.abs(got - np.exp(-2j * np.pi * (r0 * lane / 1024 + r0 * r / 32)))) < 3e-7


@pytest.mark.parametrize("bad,code", [
    (dict(Nx=100), B.SFD_EUNSUPPORTED), (dict(Ny=64), B.SFD_EUNSUPPORTED), (dict(Nx=8192), B.SFD_EUNSUPPORTED),
    (dict(Nx=0), B.SFD_EINVAL), (dict(lam=0.0), B.SFD_EINVAL), (dict(px=-1e-6), B.SFD_EINVAL),
    (dict(z=[float("nan")]), B.SFD_EINVAL), (dict(in_dtype=B.SFD_U8), B.SFD_EINVAL),
])
def test_asm_plan_create_rejects_bad_arguments(bad, code):
    kw = dict(Nx=128, Ny=128, lam=W.LAMBDA, px=W.PITCH, py=W.PITCH, z=[0.05], in_dtype=B.SFD_C64)
    kw.update(bad)
    with pytest.raises(B.SfdError) as e:
        B.sfd_asm_plan_create(kw["Nx"], kw["Ny"], 1, kw["lam"], kw["px"], kw["py"], kw["z"], kw["in_dtype"])
    assert e.value.code == code


def test_asm_entry_points_reject_null():
    assert B._lib.sfd_asm_plan_create(None, 128, 128, 1, 1e-6, 1e-6, 1e-6, None, 2, 0) == B.SFD_EINVAL
    assert B._lib.sfd_asm_execute(None, None, None, None, None, None) == B.SFD_EINVAL
    assert B._lib.sfd_asm_plan_destroy(None) == B.SFD_OK
    assert B._lib.sfd_asm_plan_device_bytes(None) == B.SFD_EINVAL
