"""Thin ctypes binding of include/hk.h: argument marshalling only.

Every step of the hot path runs in the CUDA library (csrc/); PyTorch is used for
device memory and streams.  There is no CPU fallback: if libhk.so is missing or
cannot be loaded, importing this module raises.
"""
import ctypes as C
import math
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libhk.so")

if not os.path.exists(LIB_PATH):
    raise ImportError(
        f"{LIB_PATH} not found: build the CUDA library first "
        "(python -m paper_2101_02005_b200.build, or __graft_entry__.build()); there is no CPU fallback")
_lib = C.CDLL(LIB_PATH)

HK_OK, HK_EINVAL, HK_ESTATE, HK_ENOSPC, HK_ECUDA, HK_ENOMEM = 0, -1, -2, -3, -4, -5
HK_Z1, HK_Z2, HK_Z4, HK_Z3 = 90000.0, 625.0, 49.0, 30.25
HK_STATIC_WS_BYTES = 32 << 20     # include/hk.h: the static device workspace of hk_compute_static
FIELDS = ("nu0", "A", "g_up", "E_low", "gamma_ref", "n_exp")

EXPORTS = ("hk_create", "hk_destroy", "hk_grid_size", "hk_set_conditions", "hk_workspace_bytes",
           "hk_set_workspace", "hk_compute", "hk_accumulate", "hk_compute_static", "hk_compute_batch", "hk_workspace_bytes_host", "hk_compute_host",
           "hk_get_extents", "hk_get_line_params", "hk_get_stats", "hk_get_phase_ms", "hk_probe_fp32_peak", "hk_probe_fp32_ops",
           "hk_eval_voigt_f32", "hk_set_debug_mode", "hk_set_tile_bins", "hk_set_node_separation", "hk_set_edge_nodes", "hk_set_node_kernel", "hk_set_core_nodes", "hk_set_single_pass", "hk_set_plinth", "hk_set_profile", "hk_set_cut_mode", "hk_compute_bands",
           "hk_set_conditions_hitran", "hk_compute_hitran", "hk_get_line_params_hitran",
           "hk_last_cuda_error", "hk_strerror")
PHASES = ("preprocess", "sort", "ranges", "node", "far", "mid", "edge", "centre", "lane", "near", "down")


class hk_lines(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in FIELDS]


HITRAN_FIELDS = ("nu0", "A", "g_up", "E_low", "gamma_air", "gamma_self", "n_exp", "delta")


class hk_lines_hitran(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in HITRAN_FIELDS] + [("iso", C.c_void_p)]


class hk_stats(C.Structure):
    _fields_ = [(k, C.c_int64) for k in ("n_lines", "n_skipped", "n_off_grid", "n_evals", "n_evals_far",
                                         "n_evals_mid", "n_evals_core", "n_evals_gh6", "n_evals_trap", "n_units_far", "n_units_mid", "n_units_near",
                                         "n_pairs_far", "n_pairs_mid", "n_pairs_near", "n_units_node", "n_units_edge",
                                         "n_units_centre", "n_pairs_edge", "n_pairs_centre", "n_pairs_node",
                                         "n_bins_node", "n_evals_gh10", "n_pairs_edge_node", "n_launches",
                                         "n_plinth_illcond", "n_evals_gh10_row", "n_pairs_node_eval", "n_pairs_node_far", "n_unsorted", "n_evals_core_nodes", "n_pairs_node_core")] + \
               [("scale_exp", C.c_int32), ("sort_bits", C.c_int32), ("bins_per_lane", C.c_int32), ("n_levels", C.c_int32),
                ("single_pass", C.c_int32), ("reserved0", C.c_int32)]


_vp, _d, _i64 = C.c_void_p, C.c_double, C.c_int64
_lib.hk_create.argtypes = [_d, _d, _d, C.POINTER(_vp)]
_lib.hk_destroy.argtypes = [_vp]
_lib.hk_grid_size.argtypes = [_vp]
_lib.hk_grid_size.restype = _i64
_lib.hk_set_conditions.argtypes = [_vp, _d, _d, _d, _d]
_lib.hk_workspace_bytes.argtypes = [_vp, _i64]
_lib.hk_workspace_bytes.restype = C.c_size_t
_lib.hk_set_workspace.argtypes = [_vp, _vp, C.c_size_t]
_lib.hk_compute.argtypes = [_vp, C.POINTER(hk_lines), _i64, _d, _vp, _vp]
_lib.hk_accumulate.argtypes = [_vp, C.POINTER(hk_lines), _i64, _d, _vp, _vp]
_lib.hk_compute_static.argtypes = [_vp, C.POINTER(hk_lines), _i64, _d, _vp, _vp]
_lib.hk_compute_static.restype = C.c_int
_lib.hk_compute_batch.argtypes = [_vp, C.POINTER(hk_lines), _i64, _d, C.c_int32, C.POINTER(_d), C.POINTER(_d), C.POINTER(_d),
                                  _vp, _vp]
_lib.hk_compute_batch.restype = C.c_int
_lib.hk_set_conditions_hitran.argtypes = [_vp, _d, _d, _d, C.c_int32, C.POINTER(_d), C.POINTER(_d), C.POINTER(_d)]
_lib.hk_set_conditions_hitran.restype = C.c_int
_lib.hk_compute_hitran.argtypes = [_vp, C.POINTER(hk_lines_hitran), _i64, _d, _vp, _vp]
_lib.hk_compute_hitran.restype = C.c_int
_lib.hk_get_line_params_hitran.argtypes = [_vp, C.POINTER(hk_lines_hitran), _i64, _d, _vp, _vp, _vp, _vp, _vp, _vp, _vp]
_lib.hk_get_line_params_hitran.restype = C.c_int
_lib.hk_workspace_bytes_host.argtypes = [_vp, _i64, _i64]
_lib.hk_workspace_bytes_host.restype = C.c_size_t
_lib.hk_compute_host.argtypes = [_vp, C.POINTER(hk_lines), _i64, _d, _vp, _i64, _vp]
_lib.hk_get_phase_ms.argtypes = [_vp, C.POINTER(C.c_float)]
_lib.hk_probe_fp32_peak.argtypes = [C.c_int, C.c_int, C.POINTER(_d), C.POINTER(C.c_float), _vp]
_lib.hk_probe_fp32_ops.argtypes = [C.c_int, C.c_int, C.POINTER(_d), C.POINTER(_d), C.POINTER(C.c_float), _vp]
_lib.hk_probe_fp32_ops.restype = C.c_int
_lib.hk_get_extents.argtypes = [_vp, C.POINTER(hk_lines), _i64, _vp, _vp, _vp, _vp]
_lib.hk_get_line_params.argtypes = [_vp, C.POINTER(hk_lines), _i64, _vp, _vp, _vp, _vp]
_lib.hk_get_stats.argtypes = [_vp, C.POINTER(hk_stats)]
_lib.hk_eval_voigt_f32.argtypes = [_vp, _vp, _i64, _vp, _vp, _vp]
_lib.hk_set_debug_mode.argtypes = [_vp, C.c_int]
_lib.hk_set_tile_bins.argtypes = [_vp, C.c_int]
_lib.hk_set_node_separation.argtypes = [_vp, _d]
_lib.hk_set_node_separation.restype = C.c_int
_lib.hk_set_edge_nodes.argtypes = [_vp, C.c_int]
_lib.hk_set_edge_nodes.restype = C.c_int
_lib.hk_set_node_kernel.argtypes = [_vp, C.c_int]
_lib.hk_set_node_kernel.restype = C.c_int
_lib.hk_set_core_nodes.argtypes = [_vp, C.c_int]
_lib.hk_set_core_nodes.restype = C.c_int
_lib.hk_set_single_pass.argtypes = [_vp, C.c_int]
_lib.hk_set_single_pass.restype = C.c_int
_lib.hk_set_plinth.argtypes = [_vp, C.c_int]
_lib.hk_set_plinth.restype = C.c_int
_lib.hk_set_profile.argtypes = [_vp, C.c_int]
_lib.hk_set_profile.restype = C.c_int
_lib.hk_set_cut_mode.argtypes = [_vp, C.c_int]
_lib.hk_set_cut_mode.restype = C.c_int
_lib.hk_compute_bands.argtypes = [C.POINTER(_vp), C.c_int32, C.POINTER(hk_lines), _i64, _d, C.POINTER(_vp), _vp]
_lib.hk_compute_bands.restype = C.c_int
_lib.hk_last_cuda_error.argtypes = [_vp]
_lib.hk_strerror.argtypes = [C.c_int]
_lib.hk_strerror.restype = C.c_char_p
for _name in ("hk_create", "hk_destroy", "hk_set_conditions", "hk_set_workspace", "hk_compute", "hk_get_extents",
              "hk_accumulate", "hk_compute_host", "hk_get_phase_ms", "hk_probe_fp32_peak", "hk_set_tile_bins",
              "hk_get_line_params", "hk_get_stats", "hk_eval_voigt_f32", "hk_set_debug_mode", "hk_set_tile_bins", "hk_last_cuda_error"):
    getattr(_lib, _name).restype = C.c_int


class HKError(RuntimeError):
    def __init__(self, status, where, cuda_err=0):
        self.status = status
        msg = _lib.hk_strerror(status).decode()
        super().__init__(f"{where}: {msg} (status {status}, cuda error {cuda_err})")


def hk_strerror(status: int) -> str:
    return _lib.hk_strerror(status).decode()


def _stream_ptr(stream=None):
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


def _lines_struct(lines, host=False):
    ls = hk_lines()
    n = None
    for k in FIELDS:
        t = lines[k]
        if not (t.is_cuda != host and t.dtype == torch.float64 and t.is_contiguous()):
            raise ValueError(f"lines[{k!r}] must be a contiguous {'CPU' if host else 'CUDA'} float64 tensor")
        if n is None:
            n = t.numel()
        elif t.numel() != n:
            raise ValueError("line arrays differ in length")
        setattr(ls, k, t.data_ptr())
    return ls, n


def _hitran_struct(lines):
    ls = hk_lines_hitran()
    n = None
    for k in HITRAN_FIELDS + ("iso",):
        t = lines[k]
        want = torch.int32 if k == "iso" else torch.float64
        if not (t.is_cuda and t.dtype == want and t.is_contiguous()):
            raise ValueError(f"lines[{k!r}] must be a contiguous CUDA {want} tensor")
        if n is None:
            n = t.numel()
        elif t.numel() != n:
            raise ValueError("line arrays differ in length")
        setattr(ls, k, t.data_ptr())
    return ls, n


class Opacity:
    """One grid (hk_create) + conditions + a torch-owned workspace; call compute()."""

    def __init__(self, numin: float, numax: float, dnu: float):
        self._ctx = _vp()
        st = _lib.hk_create(numin, numax, dnu, C.byref(self._ctx))
        if st != HK_OK:
            self._ctx = None
            raise HKError(st, "hk_create")
        self.N = int(_lib.hk_grid_size(self._ctx))
        self._ws = None

    def _check(self, st, where):
        if st != HK_OK:
            raise HKError(st, where, _lib.hk_last_cuda_error(self._ctx))

    def close(self):
        if getattr(self, "_ctx", None) and _lib is not None:      # (_lib is gone when the interpreter shuts down)
            _lib.hk_destroy(self._ctx)
            self._ctx = None

    __del__ = close

    def set_conditions(self, T, P_atm, mass_amu, Q):
        self._check(_lib.hk_set_conditions(self._ctx, T, P_atm, mass_amu, Q), "hk_set_conditions")

    def set_debug_mode(self, mode: int):
        self._check(_lib.hk_set_debug_mode(self._ctx, mode), "hk_set_debug_mode")

    def set_tile_bins(self, bins_per_lane: int):
        self._check(_lib.hk_set_tile_bins(self._ctx, bins_per_lane), "hk_set_tile_bins")

    def set_node_separation(self, sep: float):
        self._check(_lib.hk_set_node_separation(self._ctx, sep), "hk_set_node_separation")

    def set_profile(self, profile):
        """'voigt' (default), 'lorentz', 'doppler' or 'binned_gaussian' (hk_set_profile)."""
        code = {"voigt": 0, "lorentz": 1, "doppler": 2, "binned_gaussian": 3}.get(profile, profile)
        self._check(_lib.hk_set_profile(self._ctx, int(code)), "hk_set_profile")

    def set_cut_mode(self, mode):
        """'fixed' (default), 'lorentz' or 'doppler': cut = a multiple of each line's half-width (hk_set_cut_mode)."""
        code = {"fixed": 0, "lorentz": 1, "doppler": 2}.get(mode, mode)
        self._check(_lib.hk_set_cut_mode(self._ctx, int(code)), "hk_set_cut_mode")

    def set_plinth(self, on: bool):
        self._check(_lib.hk_set_plinth(self._ctx, 1 if on else 0), "hk_set_plinth")

    def set_node_kernel(self, entry_stationary: bool):
        self._check(_lib.hk_set_node_kernel(self._ctx, 1 if entry_stationary else 0), "hk_set_node_kernel")

    def set_core_nodes(self, on: bool):
        self._check(_lib.hk_set_core_nodes(self._ctx, 1 if on else 0), "hk_set_core_nodes")

    def set_single_pass(self, on: bool):
        self._check(_lib.hk_set_single_pass(self._ctx, 1 if on else 0), "hk_set_single_pass")

    def set_edge_nodes(self, on: bool):
        self._check(_lib.hk_set_edge_nodes(self._ctx, 1 if on else 0), "hk_set_edge_nodes")

    def workspace_bytes(self, n_lines: int) -> int:
        return int(_lib.hk_workspace_bytes(self._ctx, n_lines))

    def ensure_workspace(self, n_lines: int, need: int = None):
        if need is None:
            need = self.workspace_bytes(n_lines)
        if self._ws is None or self._ws.numel() < need:
            self._ws = None
            self._ws = torch.empty(need, dtype=torch.uint8, device="cuda")
            self._check(_lib.hk_set_workspace(self._ctx, self._ws.data_ptr(), self._ws.numel()), "hk_set_workspace")

    def compute(self, lines, cut, out=None, stream=None, accumulate=False):
        """Enqueue lines -> k(nu) on the current (or given) torch stream; returns the fp64 CUDA tensor.
        accumulate=True adds into `out` (hk_accumulate) instead of overwriting it."""
        ls, n = _lines_struct(lines)
        self.ensure_workspace(n)
        if out is None:
            assert not accumulate
            out = torch.empty(self.N, dtype=torch.float64, device="cuda")
        assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == self.N
        cut = float(cut) if cut is not None else 0.0
        fn = _lib.hk_accumulate if accumulate else _lib.hk_compute
        self._check(fn(self._ctx, C.byref(ls), n, cut, out.data_ptr(), _stream_ptr(stream)), "hk_compute")
        return out

    def compute_static(self, lines, cut, out, stream=None):
        """hk_compute_static: hk_compute on the library's static device workspace (HK_STATIC_WS_BYTES): no allocation on
        the call path -- `out` is the caller's, no workspace tensor is created.  HKError(HK_ENOSPC) beyond the limit."""
        ls, n = _lines_struct(lines)
        assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == self.N
        cut = float(cut) if cut is not None else 0.0
        self._check(_lib.hk_compute_static(self._ctx, C.byref(ls), n, cut, out.data_ptr(), _stream_ptr(stream)),
                    "hk_compute_static")
        return out

    def compute_batch(self, lines, cut, T, P_atm, Q, out=None, stream=None):
        """hk_compute_batch: k(nu) at every (T[c], P_atm[c], Q[c]) on the resident lines -> [n_cond, N] fp64 CUDA tensor."""
        ls, n = _lines_struct(lines)
        self.ensure_workspace(n)
        nc = len(T)
        assert len(P_atm) == nc and len(Q) == nc
        if out is None:
            out = torch.empty((nc, self.N), dtype=torch.float64, device="cuda")
        assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == nc * self.N
        arr = lambda v: (_d * nc)(*[float(x) for x in v])
        cut = float(cut) if cut is not None else 0.0
        self._check(_lib.hk_compute_batch(self._ctx, C.byref(ls), n, cut, nc, arr(T), arr(P_atm), arr(Q), out.data_ptr(),
                                          _stream_ptr(stream)), "hk_compute_batch")
        return out

    def set_conditions_hitran(self, T, P_atm, P_self_atm, isos):
        """isos: [(mass_amu, Q, abundance), ...] (hk_set_conditions_hitran)."""
        n = len(isos)
        arr = lambda j: (_d * n)(*[float(x[j]) for x in isos])
        self._check(_lib.hk_set_conditions_hitran(self._ctx, T, P_atm, P_self_atm, n, arr(0), arr(1), arr(2)),
                    "hk_set_conditions_hitran")

    def compute_hitran(self, lines, cut, out=None, stream=None):
        """hk_compute_hitran: HITRAN-style lines (HITRAN_FIELDS + int32 'iso') -> k(nu)."""
        ls, n = _hitran_struct(lines)
        self.ensure_workspace(n)
        if out is None:
            out = torch.empty(self.N, dtype=torch.float64, device="cuda")
        assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == self.N
        cut = float(cut) if cut is not None else 0.0
        self._check(_lib.hk_compute_hitran(self._ctx, C.byref(ls), n, cut, out.data_ptr(), _stream_ptr(stream)),
                    "hk_compute_hitran")
        return out

    def line_params_hitran(self, lines, cut, stream=None):
        """-> S, gammaL, alphaD (fp64), ilo, ihi, jc (int32) of HITRAN-style lines."""
        ls, n = _hitran_struct(lines)
        S, gL, aD = (torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
        ilo, ihi, jc = (torch.empty(n, dtype=torch.int32, device="cuda") for _ in range(3))
        cut = float(cut) if cut is not None else 0.0
        self._check(_lib.hk_get_line_params_hitran(self._ctx, C.byref(ls), n, cut, S.data_ptr(), gL.data_ptr(), aD.data_ptr(),
                                                   ilo.data_ptr(), ihi.data_ptr(), jc.data_ptr(), _stream_ptr(stream)),
                    "hk_get_line_params_hitran")
        return S, gL, aD, ilo, ihi, jc

    def compute_host(self, host_lines, cut, out=None, block_lines=0, stream=None):
        """Host-buffer entry (hk_compute_host): CPU fp64 tensors in (pinned for async copies), CPU fp64
        tensor out; blocks are copied host->device while the previous block computes.  Synchronous."""
        ls, n = _lines_struct(host_lines, host=True)
        self.ensure_workspace(n, int(_lib.hk_workspace_bytes_host(self._ctx, n, block_lines)))
        if out is None:
            out = torch.empty(self.N, dtype=torch.float64, pin_memory=True)
        assert (not out.is_cuda) and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == self.N
        cut = float(cut) if cut is not None else 0.0
        self._check(_lib.hk_compute_host(self._ctx, C.byref(ls), n, cut, out.data_ptr(), block_lines,
                                         _stream_ptr(stream)), "hk_compute_host")
        return out

    def phase_ms(self) -> dict:
        arr = (C.c_float * len(PHASES))()
        self._check(_lib.hk_get_phase_ms(self._ctx, arr), "hk_get_phase_ms")
        return {k: float(arr[i]) for i, k in enumerate(PHASES)}

    def extents(self, lines=None, n=None, stream=None):
        """hk_get_extents: (ilo, ihi, jc) of the last compute.  `lines` may be None (pass n = the last compute's line
        count) when that compute ran as one pass: the library then returns what it wrote."""
        if lines is not None:
            ls, n = _lines_struct(lines)
            lp = C.byref(ls)
        else:
            lp = None
        ilo, ihi, jc = (torch.empty(int(n), dtype=torch.int32, device="cuda") for _ in range(3))
        self._check(_lib.hk_get_extents(self._ctx, lp, int(n), ilo.data_ptr(), ihi.data_ptr(), jc.data_ptr(),
                                        _stream_ptr(stream)), "hk_get_extents")
        return ilo, ihi, jc

    def line_params(self, lines, stream=None):
        ls, n = _lines_struct(lines)
        S, gL, aD = (torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
        self._check(_lib.hk_get_line_params(self._ctx, C.byref(ls), n, S.data_ptr(), gL.data_ptr(), aD.data_ptr(),
                                            _stream_ptr(stream)), "hk_get_line_params")
        return S, gL, aD

    def stats(self) -> dict:
        s = hk_stats()
        self._check(_lib.hk_get_stats(self._ctx, C.byref(s)), "hk_get_stats")
        return {k: int(getattr(s, k)) for k, _ in hk_stats._fields_}


def compute_bands(ops, lines, cut, outs=None, stream=None):
    """hk_compute_bands: `ops` is a list of Opacity objects, one per band of the wavenumber axis (each with its own
    resolution and conditions set); -> list of fp64 CUDA tensors, one per band."""
    ls, n = _lines_struct(lines)
    nb = len(ops)
    if outs is None:
        outs = [torch.empty(op.N, dtype=torch.float64, device="cuda") for op in ops]
    for op, o in zip(ops, outs):
        op.ensure_workspace(n)
        assert o.is_cuda and o.dtype == torch.float64 and o.is_contiguous() and o.numel() == op.N
    ctxs = (_vp * nb)(*[op._ctx for op in ops])
    ptrs = (_vp * nb)(*[o.data_ptr() for o in outs])
    st = _lib.hk_compute_bands(ctxs, nb, C.byref(ls), n, float(cut) if cut is not None else 0.0, ptrs, _stream_ptr(stream))
    if st != HK_OK:
        raise HKError(st, "hk_compute_bands")
    return outs


PROBE_KINDS = ("ffma2", "ffma", "ffma2_bcast", "fadd2", "fmul2", "mufu_rcp")


def probe_fp32_ops(kind, iters=4096, stream=None):
    """hk_probe_fp32_ops -> (fp32 lane operations per second, SM clock in MHz measured inside the kernel, ms)."""
    code = PROBE_KINDS.index(kind) if isinstance(kind, str) else int(kind)
    ops, mhz, ms = _d(0.0), _d(0.0), C.c_float(0.0)
    st = _lib.hk_probe_fp32_ops(code, iters, C.byref(ops), C.byref(mhz), C.byref(ms), _stream_ptr(stream))
    if st != HK_OK:
        raise HKError(st, "hk_probe_fp32_ops")
    return ops.value, mhz.value, ms.value


def probe_fp32_peak(packed=True, iters=4096, stream=None):
    """Achieved FLOP/s of a register-resident FMA chain (hk_probe_fp32_peak) -> (flops, ms)."""
    f, ms = _d(0.0), C.c_float(0.0)
    st = _lib.hk_probe_fp32_peak(1 if packed else 0, iters, C.byref(f), C.byref(ms), _stream_ptr(stream))
    if st != HK_OK:
        raise HKError(st, "hk_probe_fp32_peak")
    return f.value, ms.value


def eval_voigt_f32(x: torch.Tensor, y: torch.Tensor, with_region=False, stream=None):
    """Re w(x + i y) through the shipped fp32 evaluator (accuracy probe, hk_eval_voigt_f32)."""
    assert x.is_cuda and y.is_cuda and x.dtype == torch.float32 and y.dtype == torch.float32
    x = x.contiguous()
    y = y.contiguous()
    out = torch.empty_like(x)
    reg = torch.empty(x.shape, dtype=torch.int32, device=x.device) if with_region else None
    st = _lib.hk_eval_voigt_f32(x.data_ptr(), y.data_ptr(), x.numel(), out.data_ptr(),
                                reg.data_ptr() if with_region else None, _stream_ptr(stream))
    if st != HK_OK:
        raise HKError(st, "hk_eval_voigt_f32")
    return (out, reg) if with_region else out
