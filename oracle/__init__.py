"""ctypes binding of the CPU oracle (oracle/dm_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package; the product path (paper_1808_10375_b200) never does and shares
no code with it.  Argument marshalling only: every number is computed in dm_oracle.c.
"""
from __future__ import annotations

import ctypes as C
import numpy as np

_LIBS: dict = {}
_vp, _i32, _i64, _dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double


def lib(real: str = "f64") -> C.CDLL:
    if real not in _LIBS:
        from . import build as _build
        _build.build()
        L = C.CDLL(_build.lib_path(real))
        rt = _dbl if real == "f64" else C.c_float
        L.oracle_fft2.argtypes = [C.c_int, _vp, _vp, C.c_int]
        L.oracle_fft2.restype = C.c_int
        L.oracle_window_table.argtypes = [C.c_int, _vp, C.c_int, _vp]
        L.oracle_window_table.restype = None
        L.oracle_coverage.argtypes = [C.c_int, C.c_int, _vp, C.c_int, C.c_int, C.c_int, C.c_int, _vp, _vp]
        L.oracle_coverage.restype = _i64
        L.oracle_cover_count.argtypes = [C.c_int, C.c_int, _vp, C.c_int, C.c_int, _vp]
        L.oracle_cover_count.restype = None
        L.oracle_modulus_project.argtypes = [C.c_int, C.c_int, _vp, _vp, rt, _vp, _vp]
        L.oracle_modulus_project.restype = None
        L.oracle_view_update.argtypes = [C.c_int] * 3 + [_vp, _vp] + [C.c_int] * 4 + [_vp, _vp, rt, rt, _vp, C.c_int]
        L.oracle_view_update.restype = None
        L.oracle_object_update.argtypes = [C.c_int] * 6 + [_vp] * 4 + [rt, _vp]
        L.oracle_object_update.restype = None
        L.oracle_probe_update.argtypes = [C.c_int] * 6 + [_vp] * 4 + [rt, _vp]
        L.oracle_probe_update.restype = None
        L.oracle_views_update.argtypes = [C.c_int] * 5 + [_vp, _vp, C.c_int, C.c_int, _vp, _vp, _vp, rt, rt, _vp]
        L.oracle_views_update.restype = None
        for f in ("oracle_object_accumulate", "oracle_probe_accumulate"):
            getattr(L, f).argtypes = [C.c_int] * 7 + [_vp] * 5
            getattr(L, f).restype = None
        L.oracle_object_finish.argtypes = [C.c_int] * 3 + [_vp] * 3 + [rt, _vp]
        L.oracle_object_finish.restype = None
        L.oracle_probe_finish.argtypes = [C.c_int] * 2 + [_vp] * 3 + [rt, _vp]
        L.oracle_probe_finish.restype = None
        L.oracle_frozen_alphas.argtypes = [C.c_int] * 6 + [_vp] * 3 + [rt, rt, _vp]
        L.oracle_frozen_alphas.restype = None
        L.oracle_rel_change.argtypes = [C.c_size_t, _vp, _vp]
        L.oracle_rel_change.restype = rt
        L.oracle_create.argtypes = [C.c_int] * 6 + [_vp]
        L.oracle_create.restype = _vp
        L.oracle_destroy.argtypes = [_vp]
        L.oracle_destroy.restype = None
        L.oracle_set_param.argtypes = [_vp, C.c_int, _dbl]
        L.oracle_set_param.restype = C.c_int
        L.oracle_set_data.argtypes = [_vp] * 4
        L.oracle_set_data.restype = C.c_int
        L.oracle_get_alphas.argtypes = [_vp, _vp]
        L.oracle_get_alphas.restype = None
        L.oracle_iterate.argtypes = [_vp, C.c_int]
        L.oracle_iterate.restype = C.c_int
        for f in ("oracle_get_probe", "oracle_get_object", "oracle_get_psi"):
            getattr(L, f).argtypes = [_vp, _vp]
            getattr(L, f).restype = None
        L.oracle_set_state.argtypes = [_vp] * 4
        L.oracle_set_state.restype = None
        L.oracle_get_errors.argtypes = [_vp, _vp, C.c_int]
        L.oracle_get_errors.restype = C.c_int
        L.oracle_num_threads.restype = C.c_int
        L.oracle_set_num_threads.argtypes = [C.c_int]
        L.oracle_real_bytes.restype = C.c_int
        _LIBS[real] = L
    return _LIBS[real]


def _p(a: np.ndarray):
    return a.ctypes.data_as(_vp)


def _types(real):
    return (np.float64, np.complex128) if real == "f64" else (np.float32, np.complex64)


def _c(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


PARAM = {"beta": 0, "alpha_obj": 1, "alpha_probe": 2, "eps_f": 3}


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_num_threads(n: int) -> None:
    lib().oracle_set_num_threads(int(n))
    if "f32" in _LIBS:
        _LIBS["f32"].oracle_set_num_threads(int(n))


def fft2(x, inverse: bool = False, real: str = "f64"):
    rt, ct = _types(real)
    x = _c(x, ct)
    out = np.empty_like(x)
    rc = lib(real).oracle_fft2(x.shape[-1], _p(x), _p(out), int(inverse))
    if rc != 0 or x.ndim != 2 or x.shape[0] != x.shape[1]:
        raise ValueError("oracle_fft2 needs a square power-of-two frame")
    return out


def window_table(positions, obj_w):
    pos = _c(positions, np.int32)
    out = np.empty((pos.shape[0], 3), np.int32)
    lib().oracle_window_table(pos.shape[0], _p(pos), int(obj_w), _p(out))
    return out


def coverage(N, positions, obj_h, obj_w, tile_h, tile_w):
    pos = _c(positions, np.int32)
    nty, ntx = -(-obj_h // tile_h), -(-obj_w // tile_w)
    nnz = lib().oracle_coverage(N, pos.shape[0], _p(pos), obj_h, obj_w, tile_h, tile_w, None, None)
    ptr = np.empty(nty * ntx + 1, np.int32)
    views = np.empty(max(int(nnz), 1), np.int32)
    lib().oracle_coverage(N, pos.shape[0], _p(pos), obj_h, obj_w, tile_h, tile_w, _p(ptr), _p(views))
    return ptr, views[:nnz]


def cover_count(N, positions, obj_h, obj_w):
    pos = _c(positions, np.int32)
    out = np.empty((obj_h, obj_w), np.int32)
    lib().oracle_cover_count(N, pos.shape[0], _p(pos), obj_h, obj_w, _p(out))
    return out


def modulus_project(F, amp, eps=1e-30, real="f64"):
    rt, ct = _types(real)
    F = _c(F, ct)
    amp = _c(amp, rt)
    M, N = F.shape[0], F.shape[-1]
    out = np.empty_like(F)
    err = np.zeros(1, rt)
    lib(real).oracle_modulus_project(N, M, _p(F), _p(amp), eps, _p(out), _p(err))
    return out, float(err[0])


def view_update(P, O, y0, x0, psi, amp, beta=1.0, eps=1e-30, fused=False, real="f64"):
    """One view of step A.  psi [K][L][N][N] -> (psi_new, acc[4])."""
    rt, ct = _types(real)
    P, O, amp = _c(P, ct), _c(O, ct), _c(amp, rt)
    psi = np.array(psi, dtype=ct, order="C", copy=True)
    K, N = P.shape[0], P.shape[-1]
    L, H, W = O.shape
    assert psi.shape == (K, L, N, N)
    acc = np.zeros(4, rt)
    lib(real).oracle_view_update(N, K, L, _p(P), _p(O), H, W, int(y0), int(x0), _p(psi), _p(amp),
                                 beta, eps, _p(acc), int(fused))
    return psi, acc.astype(np.float64)


def object_update(positions, P, psi, O_old, alpha=0.0, real="f64"):
    rt, ct = _types(real)
    pos, P, psi, O_old = _c(positions, np.int32), _c(P, ct), _c(psi, ct), _c(O_old, ct)
    K, N = P.shape[0], P.shape[-1]
    L, H, W = O_old.shape
    out = np.empty_like(O_old)
    lib(real).oracle_object_update(N, pos.shape[0], K, L, H, W, _p(pos), _p(P), _p(psi), _p(O_old),
                                   alpha, _p(out))
    return out


def probe_update(positions, O, psi, P_old, alpha=0.0, real="f64"):
    rt, ct = _types(real)
    pos, O, psi, P_old = _c(positions, np.int32), _c(O, ct), _c(psi, ct), _c(P_old, ct)
    K, N = P_old.shape[0], P_old.shape[-1]
    L, H, W = O.shape
    out = np.empty_like(P_old)
    lib(real).oracle_probe_update(N, pos.shape[0], K, L, H, W, _p(pos), _p(O), _p(psi), _p(P_old),
                                  alpha, _p(out))
    return out


# ---- view-range entry points: the same steps cut along the view axis (streaming of full-size problems) ----
def views_update(positions, j0, j1, P, O, psi_range, amp_range, beta=1.0, eps=1e-30, real="f64"):
    """Step A on views j0..j1-1 (oracle_view_update per view).  psi_range [j1-j0][K][L][N][N] ->
    (psi_new_range, acc [j1-j0][4])."""
    rt, ct = _types(real)
    pos, P, O, amp = _c(positions, np.int32), _c(P, ct), _c(O, ct), _c(amp_range, rt)
    psi = np.array(psi_range, dtype=ct, order="C", copy=True)
    K, N = P.shape[0], P.shape[-1]
    L, H, W = O.shape
    assert psi.shape == (j1 - j0, K, L, N, N) and amp.shape == (j1 - j0, N, N) and 0 <= j0 <= j1 <= pos.shape[0]
    acc = np.zeros((j1 - j0, 4), rt)
    lib(real).oracle_views_update(N, j0, j1, K, L, _p(P), _p(O), H, W, _p(pos), _p(psi), _p(amp), beta, eps, _p(acc))
    return psi, acc.astype(np.float64)


def object_accumulate(positions, j0, j1, P, psi_range, num, den, real="f64"):
    """eq. (6) sums of views j0..j1-1 added IN PLACE onto num (complex [L][H][W]) and den (real [H][W])."""
    rt, ct = _types(real)
    pos, P, psi = _c(positions, np.int32), _c(P, ct), _c(psi_range, ct)
    K, N = P.shape[0], P.shape[-1]
    L, H, W = num.shape
    assert num.dtype == ct and den.dtype == rt and num.flags.c_contiguous and den.flags.c_contiguous and den.shape == (H, W)
    assert psi.shape == (j1 - j0, K, L, N, N)
    lib(real).oracle_object_accumulate(N, j0, j1, K, L, H, W, _p(pos), _p(P), _p(psi), _p(num), _p(den))


def object_finish(num, den, O_old, alpha=0.0, real="f64"):
    rt, ct = _types(real)
    O_old = _c(O_old, ct)
    L, H, W = O_old.shape
    out = np.empty_like(O_old)
    lib(real).oracle_object_finish(L, H, W, _p(_c(num, ct)), _p(_c(den, rt)), _p(O_old), alpha, _p(out))
    return out


def probe_accumulate(positions, j0, j1, O, psi_range, num, den, real="f64"):
    """eq. (5) sums of views j0..j1-1 added IN PLACE onto num (complex [K][N][N]) and den (real [N][N])."""
    rt, ct = _types(real)
    pos, O, psi = _c(positions, np.int32), _c(O, ct), _c(psi_range, ct)
    L, H, W = O.shape
    K, N = num.shape[0], num.shape[-1]
    assert num.dtype == ct and den.dtype == rt and num.flags.c_contiguous and den.flags.c_contiguous and den.shape == (N, N)
    assert psi.shape == (j1 - j0, K, L, N, N)
    lib(real).oracle_probe_accumulate(N, j0, j1, K, L, H, W, _p(pos), _p(O), _p(psi), _p(num), _p(den))


def probe_finish(num, den, P_old, alpha=0.0, real="f64"):
    rt, ct = _types(real)
    P_old = _c(P_old, ct)
    K, N = P_old.shape[0], P_old.shape[-1]
    out = np.empty_like(P_old)
    lib(real).oracle_probe_finish(N, K, _p(_c(num, ct)), _p(_c(den, rt)), _p(P_old), alpha, _p(out))
    return out


def frozen_alphas(positions, P0, O0, a_obj=1e-3, a_probe=1e-3, real="f64"):
    """(alpha_obj, alpha_probe) as oracle_set_data freezes them (A8), without a state object."""
    rt, ct = _types(real)
    pos, P0, O0 = _c(positions, np.int32), _c(P0, ct), _c(O0, ct)
    K, N = P0.shape[0], P0.shape[-1]
    L, H, W = O0.shape
    out = np.zeros(2)
    lib(real).oracle_frozen_alphas(N, pos.shape[0], K, L, H, W, _p(pos), _p(P0), _p(O0), a_obj, a_probe, _p(out))
    return tuple(out)


def mode_power(modes):
    """Power fraction of every mode, sum_r |X_m|^2 / sum_m sum_r |X_m|^2 (a probe mode
    is kept while its contribution to the total intensity exceeds 1 %); 0/0 := 0.  Plain numpy, FP64."""
    x = np.asarray(modes).astype(np.complex128)
    p = np.array([float(np.sum(m.real ** 2 + m.imag ** 2)) for m in x])
    t = p.sum()
    return p / t if t > 0 else np.zeros_like(p)


def rel_change(new, old, real="f64"):
    rt, ct = _types(real)
    new, old = _c(new, ct), _c(old, ct)
    return float(lib(real).oracle_rel_change(new.size, _p(new), _p(old)))


class OracleDM:
    """Stateful oracle: same surface as the C-ABI of include/dm.h with host pointers."""

    def __init__(self, N, K, L, obj_h, obj_w, positions, real="f64", **params):
        self.real = real
        self.rt, self.ct = _types(real)
        self._lib = lib(real)
        pos = _c(positions, np.int32)
        self.N, self.K, self.L, self.H, self.W, self.n_views = N, K, L, obj_h, obj_w, pos.shape[0]
        self._h = self._lib.oracle_create(N, self.n_views, K, L, obj_h, obj_w, _p(pos))
        if not self._h:
            raise ValueError("oracle_create rejected the arguments (size, power of two, window bounds)")
        for k, v in params.items():
            self.set_param(k, v)

    def set_param(self, name, value):
        if self._lib.oracle_set_param(self._h, PARAM[name], float(value)) != 0:
            raise ValueError(f"bad value for {name}: {value}")

    def set_data(self, intensities, probe0, object0):
        I = _c(intensities, np.float32)
        P = _c(probe0, np.complex64)
        O = _c(object0, np.complex64)
        assert I.shape == (self.n_views, self.N, self.N) and P.shape == (self.K, self.N, self.N)
        assert O.shape == (self.L, self.H, self.W)
        self._lib.oracle_set_data(self._h, _p(I), _p(P), _p(O))

    def iterate(self, n_iter=1):
        if self._lib.oracle_iterate(self._h, int(n_iter)) != 0:
            raise RuntimeError("oracle_iterate: no data or bad n_iter")

    @property
    def alphas(self):
        out = np.zeros(2)
        self._lib.oracle_get_alphas(self._h, _p(out))
        return tuple(out)

    def probe(self):
        out = np.empty((self.K, self.N, self.N), self.ct)
        self._lib.oracle_get_probe(self._h, _p(out))
        return out

    def object(self):
        out = np.empty((self.L, self.H, self.W), self.ct)
        self._lib.oracle_get_object(self._h, _p(out))
        return out

    def psi(self):
        out = np.empty((self.n_views, self.K, self.L, self.N, self.N), self.ct)
        self._lib.oracle_get_psi(self._h, _p(out))
        return out

    def set_state(self, probe=None, object=None, psi=None):
        a = [None if x is None else _c(x, self.ct) for x in (probe, object, psi)]
        self._lib.oracle_set_state(self._h, *[None if x is None else _p(x) for x in a])

    def errors(self, max_rows=100000):
        out = np.empty((max_rows, 2 + self.K + self.L))
        n = self._lib.oracle_get_errors(self._h, _p(out), max_rows)
        return out[:n].copy()

    def close(self):
        if self._h:
            self._lib.oracle_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
