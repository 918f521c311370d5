"""CPU-side tests of the C-ABI library (no GPU): it loads, exports every symbol include/dm.h
declares, validates arguments, builds integer tables bit-identical to the oracle's, and the
kernels' own FFT pass code (dm_host_fft2) agrees with the oracle FFT."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import oracle
from paper_1808_10375_b200 import build as dm_build
from paper_1808_10375_b200 import synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def dm():
    dm_build.build()
    from paper_1808_10375_b200 import dm as _dm
    _dm.lib()
    return _dm


def test_library_exports_every_declared_symbol(dm):
    hdr = open(os.path.join(ROOT, "include", "dm.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(dm_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(dm.SYMBOLS)
    L = C.CDLL(dm.LIB_PATH)
    for s in declared:
        assert hasattr(L, s), s


def test_status_strings(dm):
    L = dm.lib()
    for code, name in dm.STATUS.items():
        assert L.dm_status_string(code).decode() == name


def test_create_rejects_bad_arguments(dm):
    pos = np.zeros((4, 2), np.int32)
    cases = [
        (dict(N=64, n_views=4, K=1, L=1, obj_h=64, obj_w=64, positions=pos), None),
        (dict(N=96, n_views=4, K=1, L=1, obj_h=128, obj_w=128, positions=pos), 3),     # N unsupported
        (dict(N=64, n_views=4, K=3, L=3, obj_h=64, obj_w=64, positions=pos), 3),       # K*L > 8
        (dict(N=64, n_views=4, K=1, L=1, obj_h=64, obj_w=65, positions=pos), 3),       # odd obj_w
        (dict(N=64, n_views=4, K=1, L=1, obj_h=63, obj_w=64, positions=pos), 2),       # window outside
        (dict(N=64, n_views=4, K=0, L=1, obj_h=64, obj_w=64, positions=pos), 1),
    ]
    for kw, want in cases:
        if want is None:
            dm.DMPlan(**kw).close()
        else:
            with pytest.raises(dm.DMError) as e:
                dm.DMPlan(**kw)
            assert e.value.status == want, kw
    bad = pos.copy()
    bad[2] = (0, 1)
    with pytest.raises(dm.DMError) as e:
        dm.DMPlan(64, 4, 1, 1, 64, 64, bad)
    assert e.value.status == 2 and "view 2" in e.value.text
    h = C.c_void_p()
    assert dm.lib().dm_plan_create(C.byref(h), 64, 4, 1, 1, 64, 64, None) == 1
    assert dm.lib().dm_plan_create(None, 64, 4, 1, 1, 64, 64, pos.ctypes.data_as(C.c_void_p)) == 1


def test_params_and_call_order(dm):
    pos = np.zeros((2, 2), np.int32)
    p = dm.DMPlan(64, 2, 1, 1, 64, 64, pos)
    p.set_param("beta", 0.8)
    for name, v in (("beta", 1.5), ("beta", -0.1), ("alpha_obj", -1), ("alpha_probe", -1), ("eps_f", -1),
                    ("beta", float("nan")), ("path", 7)):
        with pytest.raises(dm.DMError) as e:
            p.set_param(name, v)
        assert e.value.status == 1
    assert p.workspace_bytes() > 2 * 64 * 64 * 8
    w32 = p.workspace_bytes()
    p.set_param("precision", 1)                     # FP64 validation mode: larger workspace (psi + spectra in c128)
    assert p.workspace_bytes() >= w32 + 2 * 2 * 64 * 64 * 16
    p.set_param("precision", 0)
    assert p.workspace_bytes() == w32
    p.set_param("lag", 3)
    p.set_param("lag", 0)
    for name, v in (("precision", 2), ("precision", -1), ("lag", -1), ("lag", 1.5)):
        with pytest.raises(dm.DMError) as e:
            p.set_param(name, v)
        assert e.value.status == 1
    with pytest.raises(dm.DMError) as e:            # no workspace yet
        p._check(p._lib.dm_iterate(p._h, 1, None))
    assert e.value.status == 5
    with pytest.raises(dm.DMError) as e:            # misaligned workspace pointer
        p.set_workspace(0x1001, p.workspace_bytes())
    assert e.value.status == 5
    with pytest.raises(dm.DMError) as e:            # too small
        p.set_workspace(0x10000, 16)
    assert e.value.status == 5
    # a (fake, never dereferenced) aligned pointer: iterate before set_data -> NO_DATA
    p.set_workspace(0x10000, p.workspace_bytes())
    with pytest.raises(dm.DMError) as e:
        p._check(p._lib.dm_iterate(p._h, 1, None))
    assert e.value.status == 4
    for name in ("precision", "lag"):                # both size the workspace: refused once it is set
        with pytest.raises(dm.DMError) as e:
            p.set_param(name, 1)
        assert e.value.status == 1
    p.close()


@pytest.mark.parametrize("cfg_i,ny,nx", [(0, 10, 10), (1, 7, 5), (3, 3, 4), (4, 2, 3)])
def test_tables_bit_exact_vs_oracle(dm, cfg_i, ny, nx):
    cfg = synth.CONFIGS[cfg_i].scaled(ny, nx)
    pos = synth.make_positions(cfg, np.random.default_rng(0))
    p = dm.DMPlan(cfg.N, cfg.n_views, cfg.K, cfg.L, cfg.obj_h, cfg.obj_w, pos)
    assert np.array_equal(p.window_table(), oracle.window_table(pos, cfg.obj_w))
    th, tw, ptr, views = p.coverage()
    optr, oviews = oracle.coverage(cfg.N, pos, cfg.obj_h, cfg.obj_w, th, tw)
    assert np.array_equal(ptr, optr)
    assert np.array_equal(views, oviews)
    p.close()


@pytest.mark.parametrize("cfg_i", [1, 2, 3, 4])
def test_tables_full_configs(dm, cfg_i):
    """Step S0 at BASELINE.json's full sizes: window table and coverage lists bit-identical to the oracle's."""
    cfg = synth.CONFIGS[cfg_i]
    pos = synth.make_positions(cfg, np.random.default_rng(0))
    p = dm.DMPlan(cfg.N, cfg.n_views, cfg.K, cfg.L, cfg.obj_h, cfg.obj_w, pos)
    assert np.array_equal(p.window_table(), oracle.window_table(pos, cfg.obj_w))
    th, tw, ptr, views = p.coverage()
    optr, oviews = oracle.coverage(cfg.N, pos, cfg.obj_h, cfg.obj_w, th, tw)
    assert np.array_equal(ptr, optr) and np.array_equal(views, oviews)
    p.close()


@pytest.mark.parametrize("N", [64, 128, 256, 512])
def test_kernel_fft_pass_code_on_host(dm, N, rng):
    """The radix passes / twiddles / swizzle / digit-reversal the kernels inline, executed on the
    host, against the oracle's textbook FFT (FP32 vs FP64: ~1e-6 relative)."""
    x = (rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))).astype(np.complex64)
    F = dm.host_fft2(x)
    Fo = oracle.fft2(x.astype(np.complex128))
    assert synth.rel_l2(F, Fo) < 2e-6
    xi = dm.host_fft2(Fo.astype(np.complex64), inverse=True)
    assert synth.rel_l2(xi, x) < 2e-6
    # a delta at (3,5): every spectrum entry has modulus 1 and the right phase
    d = np.zeros((N, N), np.complex64)
    d[3, 5] = 1
    Fd = dm.host_fft2(d)
    u = np.arange(N)
    want = np.exp(-2j * np.pi * (3 * u[:, None] + 5 * u[None, :]) / N)
    assert np.abs(Fd - want).max() < 1e-5


def test_register_resident_fft_code_on_host(dm, rng):
    """Path 3 (csrc/dm_regfft.cuh): the register passes, both exchange layouts (32 x 32 in-warp
    transpose in two padded rounds, 16 x 16 cross-warp transpose with a staying bit) and the
    spectrum-layout table, emulated for 512 threads on the host, against the oracle FFT."""
    N = 128
    x = (rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))).astype(np.complex64)
    F = dm.host_fft2(x, path=3)
    Fo = oracle.fft2(x.astype(np.complex128))
    assert synth.rel_l2(F, Fo) < 2e-6
    xi = dm.host_fft2(Fo.astype(np.complex64), inverse=True, path=3)
    assert synth.rel_l2(xi, x) < 2e-6
    d = np.zeros((N, N), np.complex64)
    d[7, 33] = 1
    u = np.arange(N)
    want = np.exp(-2j * np.pi * (7 * u[:, None] + 33 * u[None, :]) / N)
    assert np.abs(dm.host_fft2(d, path=3) - want).max() < 1e-5
    with pytest.raises(dm.DMError):
        dm.host_fft2(np.zeros((64, 64), np.complex64), path=3)


@pytest.mark.parametrize("N", [64, 128, 256, 512])
def test_warp_fft_code_on_host(dm, N, rng):
    """Path 4 (csrc/dm_warpfft.cuh): the warp-level stage-1 / exchange / stage-2 FFT, the
    column-group scratch layout and the spectrum-layout table, emulated for one warp at a time
    on the host (rows -> scratch -> columns), against the oracle FFT."""
    x = (rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))).astype(np.complex64)
    F = dm.host_fft2(x, path=4)
    Fo = oracle.fft2(x.astype(np.complex128))
    assert synth.rel_l2(F, Fo) < 2e-6
    xi = dm.host_fft2(Fo.astype(np.complex64), inverse=True, path=4)
    assert synth.rel_l2(xi, x) < 2e-6
    d = np.zeros((N, N), np.complex64)
    d[7, 33] = 1
    u = np.arange(N)
    want = np.exp(-2j * np.pi * (7 * u[:, None] + 33 * u[None, :]) / N)
    assert np.abs(dm.host_fft2(d, path=4) - want).max() < 1e-5
