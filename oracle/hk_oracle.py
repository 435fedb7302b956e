"""ctypes front end of the fp64 CPU oracle (oracle/hk_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, bench.py's cpu_baseline /
``--impl reference`` legs and ``__graft_entry__.smoke()`` may import this.  It
imports nothing from the CUDA package and the CUDA package imports nothing from
here.  All arithmetic of the method lives in hk_oracle.c; this file only
marshals numpy arrays and, for ``opacity_grid``, narrows the line range per
block of bins (a caller's knowledge the C routine documents: with a fixed cut
no line whose centre is further than the cut from a block can reach it).
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = C.CDLL(_build.build())

_d = C.c_double
_i64 = C.c_int64
_pd = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_pi64 = np.ctypeslib.ndpointer(dtype=np.int64, flags="C_CONTIGUOUS")
_pi32 = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")

_lib.hko_num_threads.restype = C.c_int
_lib.hko_voigt_K.restype = _d
_lib.hko_voigt_K.argtypes = [_d, _d]
_lib.hko_voigt_K_array.restype = None
_lib.hko_voigt_K_array.argtypes = [_i64, _pd, _pd, _pd]
_lib.hko_grid_size.restype = _i64
_lib.hko_grid_size.argtypes = [_d, _d, _d]
_lib.hko_line_params.restype = None
_lib.hko_line_params.argtypes = [_i64, _pd, _pd, _pd, _pd, _pd, _pd, _d, _d, _d, _d,
                                 _pd, _pd, _pd, _pi32]
_lib.hko_extents.restype = None
_lib.hko_extents.argtypes = [_i64, _pd, C.c_void_p, _d, _d, _i64, _d, _pi64, _pi64, _pi64]
_lib.hko_profile.restype = _d
_lib.hko_profile.argtypes = [_d, _d, _d, _d]
_lib.hko_opacity_bins.restype = None
_lib.hko_opacity_bins.argtypes = [_i64, _pd, _pd, _pd, _pd, _pd, _pd, _d, _d, _d, _d,
                                  _d, _d, _i64, _d, _i64, _pi64, _i64, _i64, _pd,
                                  C.POINTER(_i64)]

_lib.hko_opacity_bins_ex.restype = None
_lib.hko_opacity_bins_ex.argtypes = [_i64, _pd, _pd, _pd, _pd, _pd, _pd, _d, _d, _d, _d,
                                     _d, _d, _i64, _d, C.c_int, C.c_int, C.c_int, _i64, _pi64, _i64, _i64, _pd,
                                     C.POINTER(_i64)]

FIELDS = ("nu0", "A", "g_up", "E_low", "gamma_ref", "n_exp")


def num_threads() -> int:
    return int(_lib.hko_num_threads())


def _f64(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def voigt_K(x, y):
    """Re w(x + i y), element-wise (broadcast)."""
    x, y = np.broadcast_arrays(np.asarray(x, dtype=np.float64), np.asarray(y, dtype=np.float64))
    shape = x.shape
    x = np.ascontiguousarray(x).reshape(-1)
    y = np.ascontiguousarray(y).reshape(-1)
    out = np.empty(x.size, dtype=np.float64)
    _lib.hko_voigt_K_array(x.size, x, y, out)
    return out.reshape(shape)


def grid_size(numin, numax, dnu) -> int:
    return int(_lib.hko_grid_size(numin, numax, dnu))


def line_params(lines, T, P_atm, mass_amu, Q):
    """-> S, gammaL, alphaD (fp64) and valid (int32) per line."""
    a = [_f64(lines[k]) for k in FIELDS]
    n = a[0].size
    S = np.empty(n)
    gL = np.empty(n)
    aD = np.empty(n)
    valid = np.empty(n, dtype=np.int32)
    _lib.hko_line_params(n, *a, T, P_atm, mass_amu, Q, S, gL, aD, valid)
    return S, gL, aD, valid


def extents(nu0, valid, numin, dnu, N, cut):
    """-> i_lo, i_hi, j_c (int64).  cut <= 0 or inf means uncut."""
    nu0 = _f64(nu0)
    n = nu0.size
    ilo = np.empty(n, dtype=np.int64)
    ihi = np.empty(n, dtype=np.int64)
    jc = np.empty(n, dtype=np.int64)
    vp = None
    if valid is not None:
        valid = np.ascontiguousarray(valid, dtype=np.int32)
        vp = valid.ctypes.data_as(C.c_void_p)
    _lib.hko_extents(n, nu0, vp, numin, dnu, N, float(cut), ilo, ihi, jc)
    return ilo, ihi, jc


def profile(nu, nu0, gammaL, alphaD) -> float:
    return float(_lib.hko_profile(nu, nu0, gammaL, alphaD))


PROFILES = {"voigt": 0, "lorentz": 1, "doppler": 2, "binned_gaussian": 3}


CUT_MODES = {"fixed": 0, "lorentz": 1, "doppler": 2}


def opacity_bins(lines, cond, grid, cut, bins, l0=0, l1=None, plinth=False, profile="voigt", cut_mode="fixed"):
    """k at the listed bins, brute force over lines [l0, l1).  -> (k, n_evals).
    plinth=True removes every line's value at the cutting length from its bins (section 2.1.1)."""
    a = [_f64(lines[k]) for k in FIELDS]
    n = a[0].size
    if l1 is None:
        l1 = n
    bins = np.ascontiguousarray(bins, dtype=np.int64)
    out = np.empty(bins.size)
    ev = _i64(0)
    numin, numax, dnu = grid
    N = grid_size(numin, numax, dnu)
    _lib.hko_opacity_bins_ex(n, *a, cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"],
                             numin, dnu, N, float(cut), 1 if plinth else 0, PROFILES[profile], CUT_MODES[cut_mode], bins.size, bins, int(l0), int(l1),
                             out, C.byref(ev))
    return out, int(ev.value)


def _uncut(cut) -> bool:
    return not (cut > 0.0 and np.isfinite(cut))


def opacity_window(lines_sorted, cond, grid, cut, b0, b1, plinth=False, profile="voigt", cut_mode="fixed", reach=None):
    """k on bins [b0, b1) for lines SORTED by nu0 (fixed cut: only lines within
    cut + one bin of the window are passed to the brute-force routine)."""
    numin, numax, dnu = grid
    bins = np.arange(b0, b1, dtype=np.int64)
    nu0 = lines_sorted["nu0"]
    if _uncut(cut):
        return opacity_bins(lines_sorted, cond, grid, cut, bins, plinth=plinth, profile=profile, cut_mode=cut_mode)
    reach = cut if reach is None else reach          # the largest cutting length of any line (a caller's knowledge)
    lo = numin + b0 * dnu - reach - 2.0 * dnu
    hi = numin + (b1 - 1) * dnu + reach + 2.0 * dnu
    l0 = int(np.searchsorted(nu0, lo, side="left"))
    l1 = int(np.searchsorted(nu0, hi, side="right"))
    return opacity_bins(lines_sorted, cond, grid, cut, bins, l0, l1, plinth=plinth, profile=profile, cut_mode=cut_mode)


def sort_lines(lines):
    """Lines reordered by ascending nu0 (NaN centres last).  The sum over lines
    does not depend on their order (R16)."""
    nu0 = _f64(lines["nu0"])
    order = np.argsort(nu0, kind="stable")
    return {k: _f64(lines[k])[order] for k in FIELDS}


def opacity_grid(lines, cond, grid, cut, block=512, presorted=False, plinth=False, profile="voigt", cut_mode="fixed"):
    """k on every bin of the grid.  -> (k[N], n_evals)."""
    numin, numax, dnu = grid
    N = grid_size(numin, numax, dnu)
    ls = lines if presorted else sort_lines(lines)
    k = np.zeros(N)
    evals = 0
    reach = None
    if cut_mode != "fixed" and not _uncut(cut):
        _, gL, aD, valid = line_params(ls, cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
        w = gL if cut_mode == "lorentz" else aD * np.sqrt(np.log(2.0))
        reach = float(cut) * float(np.max(np.where(valid > 0, w, 0.0), initial=0.0))
    if _uncut(cut):
        block = N
    for b0 in range(0, N, block):
        b1 = min(N, b0 + block)
        kk, ev = opacity_window(ls, cond, grid, cut, b0, b1, plinth=plinth, profile=profile, cut_mode=cut_mode, reach=reach)
        k[b0:b1] = kk
        evals += ev
    return k, evals


# ---- HITRAN-style inputs -------------------------------------------------
HITRAN_FIELDS = ("nu0", "A", "g_up", "E_low", "gamma_air", "gamma_self", "n_exp", "delta")
_lib.hko_line_params_hitran.restype = None
_lib.hko_line_params_hitran.argtypes = [_i64] + [_pd] * 8 + [_pi32, _d, _d, _d, C.c_int32, _pd, _pd, _pd,
                                                          _pd, _pd, _pd, _pd, _pi32]
_lib.hko_opacity_bins_params.restype = None
_lib.hko_opacity_bins_params.argtypes = [_i64, _pd, _pd, _pd, _pd, _pi32, _d, _d, _i64, _d, _i64, _pi64, _pd,
                                         C.POINTER(_i64)]


def line_params_hitran(lines, cond):
    """cond: T, P_atm, P_self_atm, isos = [(mass_amu, Q, abundance), ...].
    -> S, gammaL, alphaD, centre (= nu0 + delta P), valid."""
    a = [_f64(lines[k]) for k in HITRAN_FIELDS]
    iso = np.ascontiguousarray(lines["iso"], dtype=np.int32)
    n = a[0].size
    isos = np.asarray(cond["isos"], dtype=np.float64).reshape(-1, 3)
    S, gL, aD, ctr = (np.empty(n) for _ in range(4))
    valid = np.empty(n, dtype=np.int32)
    _lib.hko_line_params_hitran(n, *a, iso, cond["T"], cond["P_atm"], cond["P_self_atm"], isos.shape[0],
                                _f64(isos[:, 0]), _f64(isos[:, 1]), _f64(isos[:, 2]), S, gL, aD, ctr, valid)
    return S, gL, aD, ctr, valid


def opacity_grid_hitran(lines, cond, grid, cut, block=512):
    """k on every bin for HITRAN-style lines.  -> (k[N], n_evals)."""
    numin, numax, dnu = grid
    N = grid_size(numin, numax, dnu)
    S, gL, aD, ctr, valid = line_params_hitran(lines, cond)
    order = np.argsort(np.where(valid > 0, ctr, np.inf), kind="stable")
    S, gL, aD, ctr, valid = (np.ascontiguousarray(v[order]) for v in (S, gL, aD, ctr, valid))
    nv = int((valid > 0).sum())
    k = np.zeros(N)
    evals = 0
    step = N if _uncut(cut) else block
    for b0 in range(0, N, step):
        b1 = min(N, b0 + step)
        if _uncut(cut):
            l0, l1 = 0, nv
        else:                      # a caller's knowledge: no line further than the cut (+ a bin) from the block reaches it
            l0 = int(np.searchsorted(ctr[:nv], numin + b0 * dnu - cut - 2.0 * dnu, side="left"))
            l1 = int(np.searchsorted(ctr[:nv], numin + (b1 - 1) * dnu + cut + 2.0 * dnu, side="right"))
        bins = np.arange(b0, b1, dtype=np.int64)
        out = np.empty(bins.size)
        ev = _i64(0)
        sl = slice(l0, l1)
        _lib.hko_opacity_bins_params(l1 - l0, _f64(ctr[sl]), _f64(S[sl]), _f64(gL[sl]), _f64(aD[sl]),
                                     np.ascontiguousarray(valid[sl]), numin, dnu, N, float(cut), bins.size, bins, out,
                                     C.byref(ev))
        k[b0:b1] = out
        evals += int(ev.value)
    return k, evals
