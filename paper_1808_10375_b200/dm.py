"""Thin ctypes binding of the C-ABI library (include/dm.h): argument marshalling only.

Every step of the difference-map iteration (arXiv:1808.10375 Sec. II) runs
in the CUDA kernels of csrc/; PyTorch is used for device memory and streams, nothing else.
There is no CPU fallback: if the library is missing, loading raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdm_b200.so")

DM_OK = 0
STATUS = {0: "DM_OK", 1: "DM_ERR_INVALID_ARG", 2: "DM_ERR_OUT_OF_BOUNDS", 3: "DM_ERR_UNSUPPORTED",
          4: "DM_ERR_NO_DATA", 5: "DM_ERR_WORKSPACE", 6: "DM_ERR_CUDA"}
PARAM = {"beta": 0, "alpha_obj": 1, "alpha_probe": 2, "eps_f": 3, "path": 4, "lag": 5, "precision": 6}

# every symbol include/dm.h declares (tests check the library exports exactly these)
SYMBOLS = (
    "dm_plan_create", "dm_plan_set_param", "dm_plan_workspace_bytes", "dm_plan_set_workspace",
    "dm_set_data", "dm_iterate", "dm_get_probe", "dm_get_object", "dm_get_psi", "dm_get_errors",
    "dm_set_state", "dm_get_window_table", "dm_get_coverage", "dm_get_alphas", "dm_get_mode_power", "dm_solve_host",
    "dm_plan_info", "dm_plan_geometry", "dm_plan_set_profiling", "dm_get_phase_ms", "dm_measure_peaks", "dm_host_fft2", "dm_host_fft2_path",
    "dm_probe_update_noalloc", "dm_status_string", "dm_last_error", "dm_plan_destroy",
)

_vp, _int, _dbl = C.c_void_p, C.c_int, C.c_double
_lib = None


class DMError(RuntimeError):
    def __init__(self, status: int, text: str):
        super().__init__(f"{STATUS.get(status, status)}: {text}")
        self.status = status
        self.text = text


def lib() -> C.CDLL:
    """Load libdm_b200.so (built by paper_1808_10375_b200.build).  Raises if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1808_10375_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.dm_plan_create.argtypes = [C.POINTER(_vp)] + [_int] * 6 + [_vp]
        L.dm_plan_set_param.argtypes = [_vp, _int, _dbl]
        L.dm_plan_workspace_bytes.argtypes = [_vp, C.POINTER(C.c_size_t)]
        L.dm_plan_set_workspace.argtypes = [_vp, _vp, C.c_size_t]
        L.dm_set_data.argtypes = [_vp] * 5
        L.dm_iterate.argtypes = [_vp, _int, _vp]
        for f in ("dm_get_probe", "dm_get_object", "dm_get_psi"):
            getattr(L, f).argtypes = [_vp, _vp, _vp]
        L.dm_get_errors.argtypes = [_vp, _vp, _int, C.POINTER(_int)]
        L.dm_set_state.argtypes = [_vp] * 5
        L.dm_get_window_table.argtypes = [_vp, _vp]
        L.dm_get_coverage.argtypes = [_vp, C.POINTER(_int), C.POINTER(_int), _vp, _vp, C.POINTER(C.c_int64)]
        L.dm_get_alphas.argtypes = [_vp, _vp]
        L.dm_get_mode_power.argtypes = [_vp, _vp]
        L.dm_solve_host.argtypes = [_vp, _vp, _vp, _vp, _int, _vp, _vp, _vp]
        L.dm_plan_info.argtypes = [_vp, C.POINTER(_int), C.POINTER(_int)]
        L.dm_plan_geometry.argtypes = [_vp, _vp, _int]
        L.dm_plan_set_profiling.argtypes = [_vp, _int]
        L.dm_get_phase_ms.argtypes = [_vp, _vp, C.POINTER(_int)]
        L.dm_measure_peaks.argtypes = [_vp, C.c_size_t, _vp, _int, _vp]
        L.dm_host_fft2.argtypes = [_int, _vp, _vp, _int]
        L.dm_host_fft2_path.argtypes = [_int, _int, _vp, _vp, _int]
        L.dm_probe_update_noalloc.argtypes = [_int] * 6 + [_vp] * 4 + [C.c_float, _vp, _vp, C.c_char_p, C.c_size_t]
        L.dm_status_string.argtypes = [_int]
        L.dm_status_string.restype = C.c_char_p
        L.dm_last_error.argtypes = [_vp]
        L.dm_last_error.restype = C.c_char_p
        L.dm_plan_destroy.argtypes = [_vp]
        L.dm_plan_destroy.restype = None
        for s in SYMBOLS:
            if s not in ("dm_status_string", "dm_last_error", "dm_plan_destroy"):
                getattr(L, s).restype = _int
        _lib = L
    return _lib


def _np_ptr(a: np.ndarray):
    return a.ctypes.data_as(_vp)


PEAK_FIELDS = ("fp32_lane_ops_per_s_ffma", "fp32_lane_ops_per_s_ffma2", "hbm_read_gbs", "hbm_copy_gbs", "l2_read_gbs",
               "smem_read_gbs", "sms")


def measure_peaks(scratch_bytes: int = 2 << 30) -> dict:
    """dm_measure_peaks: FP32 / HBM / L2 / shared-memory rates of the current CUDA device (syncs)."""
    import torch
    buf = torch.empty(scratch_bytes, dtype=torch.uint8, device="cuda")
    out = np.zeros(len(PEAK_FIELDS), dtype=np.float64)
    st = lib().dm_measure_peaks(_vp(buf.data_ptr()), scratch_bytes, _np_ptr(out), len(out), _vp(torch.cuda.current_stream().cuda_stream))
    if st != 0:
        raise DMError(st, "dm_measure_peaks")
    return dict(zip(PEAK_FIELDS, (float(v) for v in out)))


def host_fft2(x: np.ndarray, inverse: bool = False, path: int = 0) -> np.ndarray:
    """dm_host_fft2[_path]: the kernels' own FFT pass code run on the host (test hook, no CUDA)."""
    x = np.ascontiguousarray(x, np.complex64)
    out = np.empty_like(x)
    if path:
        st = lib().dm_host_fft2_path(x.shape[-1], path, _np_ptr(x), _np_ptr(out), int(inverse))
    else:
        st = lib().dm_host_fft2(x.shape[-1], _np_ptr(x), _np_ptr(out), int(inverse))
    if st != DM_OK:
        raise DMError(st, "dm_host_fft2")
    return out


NOALLOC_SCRATCH_BYTES = 16 << 20


def probe_update_noalloc(positions, object_, psi, probe_old, alpha_probe, out=None, stream=None):
    """dm_probe_update_noalloc: eq. (5) on device tensors the caller already holds, for callers that
    cannot allocate device memory (an application whose pool owns the whole card, a loop where cudaMalloc's
    device-wide stall is not acceptable): the partial sums go to a fixed NOALLOC_SCRATCH_BYTES array inside the
    library instead of a workspace.  positions int32 [n_views][2] (device), object_ c64 [L][H][W], psi c64
    [n_views][K][L][N][N], probe_old c64 [K][N][N]; returns P_new (written into `out` when given, so that this
    wrapper allocates nothing either).  Calls share the array: do not overlap two of them on one GPU.  The first
    call on a device does a one-time address look-up; keep it outside stream capture."""
    import torch
    n_views, K, L, N = psi.shape[0], psi.shape[1], psi.shape[2], psi.shape[-1]
    H, W = object_.shape[-2:]
    assert positions.is_cuda and positions.dtype == torch.int32 and positions.is_contiguous() and tuple(positions.shape) == (n_views, 2)
    for t, shape in ((object_, (L, H, W)), (psi, (n_views, K, L, N, N)), (probe_old, (K, N, N))):
        assert t.is_cuda and t.dtype == torch.complex64 and t.is_contiguous() and tuple(t.shape) == shape
    if out is None:
        out = torch.empty_like(probe_old)
    assert out.is_cuda and out.dtype == torch.complex64 and out.is_contiguous() and tuple(out.shape) == (K, N, N)
    err = C.create_string_buffer(512)
    st = lib().dm_probe_update_noalloc(N, n_views, K, L, H, W, _vp(positions.data_ptr()), _vp(object_.data_ptr()),
                                       _vp(psi.data_ptr()), _vp(probe_old.data_ptr()), float(alpha_probe),
                                       _vp(out.data_ptr()), DMPlan._stream(stream), err, len(err))
    if st != DM_OK:
        raise DMError(st, err.value.decode())
    return out


class DMPlan:
    """Owner of one dm_plan and (optionally) of its torch-allocated device workspace."""

    def __init__(self, N, n_views, K, L, obj_h, obj_w, positions, **params):
        self._lib = lib()
        self._h = _vp()
        pos = np.ascontiguousarray(positions, np.int32)
        if pos.shape != (n_views, 2):
            raise ValueError("positions must be int32 [n_views][2]")
        st = self._lib.dm_plan_create(C.byref(self._h), N, n_views, K, L, obj_h, obj_w, _np_ptr(pos))
        if st != DM_OK:
            self._h = _vp()
            raise DMError(st, self._lib.dm_last_error(None).decode())
        self.N, self.n_views, self.K, self.L, self.H, self.W = N, n_views, K, L, obj_h, obj_w
        self._ws = None
        for k, v in params.items():
            self.set_param(k, v)

    # -- plumbing ---------------------------------------------------------------------
    def _check(self, st):
        if st != DM_OK:
            raise DMError(st, self._lib.dm_last_error(self._h).decode())

    @staticmethod
    def _stream(stream):
        if stream is None:
            import torch
            return _vp(torch.cuda.current_stream().cuda_stream)
        return _vp(getattr(stream, "cuda_stream", stream))

    @staticmethod
    def _dev(t):
        return _vp(t.data_ptr())

    def set_param(self, name, value):
        self._check(self._lib.dm_plan_set_param(self._h, PARAM[name], float(value)))

    def workspace_bytes(self) -> int:
        n = C.c_size_t()
        self._check(self._lib.dm_plan_workspace_bytes(self._h, C.byref(n)))
        return int(n.value)

    def set_workspace(self, dev_ptr: int, nbytes: int):
        self._check(self._lib.dm_plan_set_workspace(self._h, _vp(dev_ptr), nbytes))

    def alloc_workspace(self, device="cuda"):
        """Allocate the workspace with torch (device memory only) and lend it to the plan."""
        import torch
        n = self.workspace_bytes()
        self._ws = torch.empty(n + 256, dtype=torch.uint8, device=device)
        base = (self._ws.data_ptr() + 255) // 256 * 256
        self.set_workspace(base, n)
        return self

    # -- the hot path -----------------------------------------------------------------
    def set_data(self, intensities, probe0, object0, stream=None):
        """Device tensors: f32 [n_views][N][N], c64 [K][N][N], c64 [L][H][W]."""
        import torch
        assert intensities.is_cuda and intensities.dtype == torch.float32 and intensities.is_contiguous()
        assert tuple(intensities.shape) == (self.n_views, self.N, self.N)
        assert probe0.dtype == torch.complex64 and probe0.is_contiguous() and tuple(probe0.shape) == (self.K, self.N, self.N)
        assert object0.dtype == torch.complex64 and object0.is_contiguous() and tuple(object0.shape) == (self.L, self.H, self.W)
        self._check(self._lib.dm_set_data(self._h, self._dev(intensities), self._dev(probe0), self._dev(object0),
                                          self._stream(stream)))

    def iterate(self, n_iter=1, stream=None):
        self._check(self._lib.dm_iterate(self._h, int(n_iter), self._stream(stream)))

    def solve_host(self, intensities, probe0, object0, n_iter, out_probe=None, out_object=None, stream=None):
        """dm_solve_host: HOST numpy / pinned torch buffers in, HOST buffers out, syncs."""
        def hp(a):
            if a is None:
                return None
            return _vp(a.data_ptr()) if hasattr(a, "data_ptr") else _np_ptr(a)
        self._check(self._lib.dm_solve_host(self._h, hp(intensities), hp(probe0), hp(object0), int(n_iter),
                                            hp(out_probe), hp(out_object), self._stream(stream)))

    def _get(self, fn, shape, stream):
        import torch
        out = torch.empty(shape, dtype=torch.complex64, device="cuda")
        self._check(fn(self._h, self._dev(out), self._stream(stream)))
        return out

    def probe(self, stream=None):
        return self._get(self._lib.dm_get_probe, (self.K, self.N, self.N), stream)

    def object(self, stream=None):
        return self._get(self._lib.dm_get_object, (self.L, self.H, self.W), stream)

    def psi(self, stream=None):
        return self._get(self._lib.dm_get_psi, (self.n_views, self.K, self.L, self.N, self.N), stream)

    def set_state(self, probe=None, object=None, psi=None, stream=None):
        args = [None if t is None else self._dev(t) for t in (probe, object, psi)]
        self._check(self._lib.dm_set_state(self._h, *args, self._stream(stream)))

    def errors(self, max_rows=16384) -> np.ndarray:
        out = np.empty((max_rows, 2 + self.K + self.L), np.float64)
        n = _int()
        self._check(self._lib.dm_get_errors(self._h, _np_ptr(out), max_rows, C.byref(n)))
        return out[: n.value].copy()

    @property
    def alphas(self):
        out = np.zeros(2)
        self._check(self._lib.dm_get_alphas(self._h, _np_ptr(out)))
        return tuple(out)

    def mode_power(self):
        """(probe fractions [K], object fractions [L]) of the current state."""
        out = np.zeros(self.K + self.L)
        self._check(self._lib.dm_get_mode_power(self._h, _np_ptr(out)))
        return out[: self.K].copy(), out[self.K:].copy()

    def info(self):
        p, n = _int(), _int()
        self._check(self._lib.dm_plan_info(self._h, C.byref(p), C.byref(n)))
        return {"path": p.value, "launches_per_iter": n.value}

    GEOMETRY = ("path", "sms", "prb_chunks", "prb_chunk_len", "obj_max_list", "obj_batch", "reg_grid",
                "reg_ctas_per_view", "reg_views_per_group", "wf_slots", "wf_lag", "wf_grid", "wf_warps", "reg_sw_barrier")

    def geometry(self):
        """dm_plan_geometry: the launch geometry as a dict (valid after set_data)."""
        out = np.zeros(len(self.GEOMETRY), np.int32)
        self._check(self._lib.dm_plan_geometry(self._h, _np_ptr(out), len(out)))
        return dict(zip(self.GEOMETRY, (int(v) for v in out)))

    def set_profiling(self, on=True):
        self._check(self._lib.dm_plan_set_profiling(self._h, int(bool(on))))

    def phase_ms(self):
        """Summed device milliseconds of (psi update, object, probe, errors) and the iteration count."""
        out = np.zeros(4, np.float32)
        n = _int()
        self._check(self._lib.dm_get_phase_ms(self._h, _np_ptr(out), C.byref(n)))
        return out.astype(np.float64), n.value

    # -- integer tables (host) ----------------------------------------------------------
    def window_table(self) -> np.ndarray:
        out = np.empty((self.n_views, 3), np.int32)
        self._check(self._lib.dm_get_window_table(self._h, _np_ptr(out)))
        return out

    def coverage(self):
        th, tw, nnz = _int(), _int(), C.c_int64()
        self._check(self._lib.dm_get_coverage(self._h, C.byref(th), C.byref(tw), None, None, C.byref(nnz)))
        nt = -(-self.H // th.value) * -(-self.W // tw.value)
        ptr = np.empty(nt + 1, np.int32)
        views = np.empty(max(nnz.value, 1), np.int32)
        self._check(self._lib.dm_get_coverage(self._h, C.byref(th), C.byref(tw), _np_ptr(ptr), _np_ptr(views),
                                              C.byref(nnz)))
        return th.value, tw.value, ptr, views[: nnz.value]

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            self._lib.dm_plan_destroy(self._h)
            self._h = _vp()
        self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
