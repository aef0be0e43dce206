"""Thin ctypes binding of libgbk (include/gbk.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of csrc/; PyTorch is used by callers for
device memory and streams.  There is no CPU fallback: if libgbk.so is missing the import of
the library fails loudly, and without a CUDA device every compute call raises GbkError.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgbk.so")

GBK_P = 10
GBK_P_EPINAT = 12   # GBK_P + the Epinat slopes a, g (eq. 7)
GBK_P_MAX = 12
GBK_OK, GBK_ERR_ARG, GBK_ERR_ALLOC, GBK_ERR_CUDA, GBK_ERR_UNSUPPORTED = range(5)
GBK_RC_ARCTAN, GBK_RC_RAMP, GBK_RC_EPINAT = 0, 1, 2
GBK_STRATEGY_CUBE, GBK_STRATEGY_VFIELD = 0, 1
GBK_PSF_GAUSSIAN, GBK_PSF_IMAGE = 0, 1
GBK_EXTRACT_MOMENTS, GBK_EXTRACT_GAUSSFIT = 0, 1

EXPORTS = (   # every symbol include/gbk.h declares (tests/test_abi_and_dist.py checks them all)
    "gbk_create_problem", "gbk_get_info", "gbk_set_strategy", "gbk_set_extraction", "gbk_reserve", "gbk_eval_batch",
    "gbk_eval_batch_counted", "gbk_eval_batch_static",
    "gbk_eval_batch_unfused", "gbk_eval_vfield_batch", "gbk_eval_batch_host", "gbk_destroy",
    "gbk_last_error", "gbk_probe_pipe", "gbk_probe_umma", "gbk_fit_ng", "gbk_fit_lm", "gbk_fit_ns",
)


class GbkError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libgbk error {code}: {msg}")
        self.code = code


class gbk_problem_desc(C.Structure):
    _fields_ = [
        ("nx", C.c_int32), ("ny", C.c_int32), ("nv", C.c_int32), ("u", C.c_int32),
        ("v_center", C.c_float), ("dv", C.c_float),
        ("rc_model", C.c_int32), ("n_gal", C.c_int32),
        ("vobs", C.c_void_p), ("verr", C.c_void_p), ("sobs", C.c_void_p), ("serr", C.c_void_p),
        ("mask", C.c_void_p),
        ("psf_kind", C.c_int32),
        ("psf_fwhm", C.c_void_p), ("psf_image", C.c_void_p), ("psf_n", C.c_int32),
        ("psf_per_gal", C.c_int32),
        ("lsf_sigma", C.c_float),
        ("tile_w", C.c_int32), ("tile_h", C.c_int32),
        ("device", C.c_int32),
        ("intensity_table", C.c_void_p), ("intensity_n", C.c_int32), ("intensity_dx", C.c_float),
    ]


class gbk_problem_info(C.Structure):
    _fields_ = [
        ("nx", C.c_int32), ("ny", C.c_int32), ("nv", C.c_int32), ("u", C.c_int32),
        ("n_gal", C.c_int32), ("r_v", C.c_int32), ("r_p_max", C.c_int32),
        ("tile_w", C.c_int32), ("tile_h", C.c_int32), ("tiles_x", C.c_int32),
        ("tiles_y", C.c_int32), ("block_threads", C.c_int32), ("smem_bytes", C.c_int32),
        ("blocks_per_sm", C.c_int32), ("sm_count", C.c_int32),
        ("ext_voxels_per_eval", C.c_int64),
        ("device", C.c_int32),
        ("strategy", C.c_int32),
        ("unfused_bytes_per_eval", C.c_int64),
        ("row_stride", C.c_int32), ("extraction", C.c_int32),
    ]


class gbk_fit_stats(C.Structure):
    _fields_ = [
        ("evals", C.c_int64), ("launches", C.c_int32), ("iterations", C.c_int32),
        ("converged", C.c_int32), ("ms_total", C.c_float), ("failed", C.c_int32),
    ]


_lib = None


def lib():
    """The loaded C-ABI library; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(
                f"{LIB_PATH} is missing: build it with `python -m paper_1510_01815_b200.build` "
                "(or __graft_entry__.build()); there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        vp = C.c_void_p
        L.gbk_create_problem.argtypes = [C.POINTER(gbk_problem_desc), C.POINTER(vp)]
        L.gbk_create_problem.restype = C.c_int
        L.gbk_get_info.argtypes = [vp, C.POINTER(gbk_problem_info)]
        L.gbk_get_info.restype = C.c_int
        for name in ("gbk_eval_batch", "gbk_eval_batch_unfused", "gbk_eval_batch_static"):
            f = getattr(L, name)
            f.argtypes = [vp, vp, vp, C.c_int64, vp, vp, vp, vp, vp, vp]
            f.restype = C.c_int
        L.gbk_eval_batch_counted.argtypes = [vp, vp, vp, C.c_int64, vp, vp, vp]
        L.gbk_eval_batch_counted.restype = C.c_int
        L.gbk_reserve.argtypes = [vp, C.c_int64, vp]
        L.gbk_reserve.restype = C.c_int
        L.gbk_set_extraction.argtypes = [vp, C.c_int32]
        L.gbk_set_extraction.restype = C.c_int
        L.gbk_set_strategy.argtypes = [vp, C.c_int32]
        L.gbk_set_strategy.restype = C.c_int
        L.gbk_eval_vfield_batch.argtypes = [vp, vp, vp, C.c_int64, vp, vp, vp, vp]
        L.gbk_eval_vfield_batch.restype = C.c_int
        L.gbk_eval_batch_host.argtypes = [vp, vp, vp, C.c_int64, vp, vp]
        L.gbk_eval_batch_host.restype = C.c_int
        L.gbk_destroy.argtypes = [vp]
        L.gbk_destroy.restype = C.c_int
        L.gbk_last_error.argtypes = []
        L.gbk_last_error.restype = C.c_char_p
        L.gbk_probe_pipe.argtypes = [C.c_int, C.c_int64, C.c_int, C.c_int, vp,
                                     C.POINTER(C.c_double), vp]
        L.gbk_probe_pipe.restype = C.c_int
        L.gbk_probe_umma.argtypes = [C.c_int, C.c_int, vp, C.POINTER(C.c_double), vp]
        L.gbk_probe_umma.restype = C.c_int
        sp = C.POINTER(gbk_fit_stats)
        L.gbk_fit_ng.argtypes = [vp, vp, C.c_int32, C.c_int32, vp, vp, vp, vp, vp, C.c_int32, vp,
                                 vp, sp, vp]
        L.gbk_fit_ng.restype = C.c_int
        L.gbk_fit_lm.argtypes = [vp, C.c_int32, vp, vp, C.c_int32, vp, vp, vp, C.c_float, C.c_int32,
                                 C.c_float, vp, vp, vp, sp, vp]
        L.gbk_fit_lm.restype = C.c_int
        L.gbk_fit_ns.argtypes = [vp, vp, C.c_int32, C.c_int32, vp, vp, vp, C.c_int32, C.c_int32,
                                 C.c_int32, C.c_float, C.c_float, C.c_uint64, vp, vp, vp,
                                 C.POINTER(C.c_double), sp, vp]
        L.gbk_fit_ns.restype = C.c_int
        _lib = L
    return _lib


def gbk_last_error() -> str:
    return lib().gbk_last_error().decode()


def _check(rc: int):
    if rc != GBK_OK:
        raise GbkError(rc, gbk_last_error())


def _ptr(t) -> Optional[int]:
    """Device/host address of a torch tensor or numpy array (None -> NULL)."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return t.data_ptr()


def _host_f32(a, shape=None):
    if a is None:
        return None
    a = np.ascontiguousarray(a, dtype=np.float32)
    if shape is not None and a.size != int(np.prod(shape)):
        raise ValueError(f"expected {shape} elements, got {a.shape}")
    return a


# ------------------------------------------------------------------ C calls, same names ----

def gbk_create_problem(*, nx, ny, nv, u=1, v_center=0.0, dv, rc_model=GBK_RC_ARCTAN, n_gal=1,
                       vobs, verr, sobs=None, serr=None, mask=None,
                       psf_kind=GBK_PSF_GAUSSIAN, psf_fwhm=None, psf_image=None, psf_per_gal=False,
                       lsf_sigma=0.0, tile_w=0, tile_h=0, device=-1, intensity_table=None,
                       intensity_dx=0.0) -> int:
    """Returns the opaque handle (an integer address).  Host arrays are copied by the library."""
    shape = (n_gal, ny, nx)
    keep = [_host_f32(vobs, shape), _host_f32(verr, shape), _host_f32(sobs, shape),
            _host_f32(serr, shape)]
    mk = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    if mk is not None and mk.size != n_gal * ny * nx:
        raise ValueError("mask has the wrong size")
    n_psf = n_gal if psf_per_gal else 1
    fw = None
    img = None
    psf_n = 0
    if psf_kind == GBK_PSF_GAUSSIAN:
        fw = np.ascontiguousarray(np.broadcast_to(np.asarray(psf_fwhm, dtype=np.float32).reshape(-1),
                                                  (n_psf,)))
    else:
        img = np.ascontiguousarray(psf_image, dtype=np.float32)
        psf_n = img.shape[-1]
        if img.size != n_psf * psf_n * psf_n:
            raise ValueError("psf_image has the wrong size")
    tab = _host_f32(intensity_table)
    d = gbk_problem_desc(nx, ny, nv, u, v_center, dv, rc_model, n_gal,
                         _ptr(keep[0]), _ptr(keep[1]), _ptr(keep[2]), _ptr(keep[3]), _ptr(mk),
                         psf_kind, _ptr(fw), _ptr(img), psf_n, 1 if psf_per_gal else 0,
                         lsf_sigma, tile_w, tile_h, device,
                         _ptr(tab), 0 if tab is None else tab.size, intensity_dx)
    out = C.c_void_p()
    _check(lib().gbk_create_problem(C.byref(d), C.byref(out)))
    return out.value


def gbk_get_info(handle: int) -> gbk_problem_info:
    info = gbk_problem_info()
    _check(lib().gbk_get_info(handle, C.byref(info)))
    return info


def gbk_eval_batch(handle, params, gal_index, K, chi2, m0=None, m1=None, m2=None, resid=None,
                   stream=0, unfused=False):
    """Device buffers (torch CUDA tensors or raw addresses); asynchronous on `stream`."""
    f = lib().gbk_eval_batch_unfused if unfused else lib().gbk_eval_batch
    _check(f(handle, _ptr(params), _ptr(gal_index), int(K), _ptr(chi2), _ptr(m0), _ptr(m1),
             _ptr(m2), _ptr(resid), stream or None))


def gbk_eval_batch_unfused(handle, params, gal_index, K, chi2, m0=None, m1=None, m2=None,
                           resid=None, stream=0):
    gbk_eval_batch(handle, params, gal_index, K, chi2, m0, m1, m2, resid, stream, unfused=True)


GBK_CNT_ITEMS, GBK_CNT_POLY_BLOCKS, GBK_CNT_DIRECT_CHANNELS, GBK_CNT_PRECISE_ITEMS, GBK_N_COUNTERS = range(5)


def gbk_eval_batch_counted(handle, params, gal_index, K, chi2, counters, stream=0):
    """gbk_eval_batch (chi^2 only) adding the voxel loop's work counts to `counters` (device int64 [4])."""
    _check(lib().gbk_eval_batch_counted(handle, _ptr(params), _ptr(gal_index), int(K), _ptr(chi2),
                                        _ptr(counters), stream or None))


GBK_STATIC_MAX_ROWS, GBK_STATIC_MAX_PARTIALS = 1 << 16, 1 << 20


def gbk_eval_batch_static(handle, params, gal_index, K, chi2, m0=None, m1=None, m2=None, resid=None, stream=0):
    """gbk_eval_batch that allocates nothing: cross-tile scratch in the library's static device array
    (K <= GBK_STATIC_MAX_ROWS, K x tiles <= GBK_STATIC_MAX_PARTIALS; overlapping calls race on it)."""
    _check(lib().gbk_eval_batch_static(handle, _ptr(params), _ptr(gal_index), int(K), _ptr(chi2), _ptr(m0),
                                       _ptr(m1), _ptr(m2), _ptr(resid), stream or None))


def gbk_reserve(handle, K_max: int, stream=0):
    """Sizes the scratch of `stream` for batches of up to K_max rows (required before a capture)."""
    _check(lib().gbk_reserve(handle, int(K_max), stream or None))


def gbk_set_strategy(handle, strategy: int):
    """Strategy the host drivers evaluate with (GBK_STRATEGY_CUBE / GBK_STRATEGY_VFIELD)."""
    _check(lib().gbk_set_strategy(handle, int(strategy)))


def gbk_set_extraction(handle, extraction: int):
    """Moments (GBK_EXTRACT_MOMENTS) or Gaussian-profile fits (GBK_EXTRACT_GAUSSFIT) for the maps."""
    _check(lib().gbk_set_extraction(handle, int(extraction)))


def gbk_eval_vfield_batch(handle, params, gal_index, K, chi2, vmap=None, resid=None, stream=0):
    """Velocity-field strategy (device buffers; asynchronous on `stream`)."""
    _check(lib().gbk_eval_vfield_batch(handle, _ptr(params), _ptr(gal_index), int(K), _ptr(chi2),
                                       _ptr(vmap), _ptr(resid), stream or None))


def gbk_eval_batch_host(handle, params, gal_index, K, chi2, stream=0):
    """Host buffers (numpy arrays or pinned torch CPU tensors); returns when chi2 is on the host."""
    _check(lib().gbk_eval_batch_host(handle, _ptr(params), _ptr(gal_index), int(K), _ptr(chi2),
                                     stream or None))


def gbk_destroy(handle):
    if handle:
        _check(lib().gbk_destroy(handle))


def gbk_probe_pipe(which: int, iters: int, blocks: int, threads: int, sink, stream=0) -> float:
    ops = C.c_double()
    _check(lib().gbk_probe_pipe(which, iters, blocks, threads, _ptr(sink), C.byref(ops),
                                stream or None))
    return ops.value


def gbk_probe_umma(iters: int, blocks: int, check, stream=0) -> float:
    """The tcgen05.mma sequence of the 15 x 15 pass as a banded contraction; returns 2 x multiply-adds issued."""
    fl = C.c_double()
    _check(lib().gbk_probe_umma(int(iters), int(blocks), _ptr(check), C.byref(fl), stream or None))
    return fl.value


def _stats_dict(st: gbk_fit_stats) -> dict:
    return {k: getattr(st, k) for k, _ in gbk_fit_stats._fields_}


def _box(params, lo, hi):
    idx = np.ascontiguousarray(params, dtype=np.int32)
    lo = np.ascontiguousarray(lo, dtype=np.float32)
    hi = np.ascontiguousarray(hi, dtype=np.float32)
    if not (idx.size == lo.size == hi.size):
        raise ValueError("params, lo and hi must have the same length")
    return idx, lo, hi


def _stride(handle) -> int:
    return gbk_get_info(handle).row_stride


def gbk_fit_ng(handle, base_row, gal, axis_param, axis_lo, axis_hi, nodes, levels, accuracy=None, stream=0):
    """Nested grids (host arrays in, host results out) -> (best_row [row_stride], best_chi2, stats).
    `nodes`: one count for all axes or one per axis; `levels`: the most levels to run; `accuracy`:
    per-axis spacing thresholds that end the refinement (None: run exactly `levels` levels)."""
    S = _stride(handle)
    base = _host_f32(base_row, (S,))
    idx, lo, hi = _box(axis_param, axis_lo, axis_hi)
    nn = np.ascontiguousarray(np.broadcast_to(np.asarray(nodes, dtype=np.int32).reshape(-1), (idx.size,)))
    acc = None if accuracy is None else np.ascontiguousarray(
        np.broadcast_to(np.asarray(accuracy, dtype=np.float32).reshape(-1), (idx.size,)))
    best = np.empty(S, np.float32)
    chi = np.empty(1, np.float32)
    st = gbk_fit_stats()
    _check(lib().gbk_fit_ng(handle, _ptr(base), int(gal), idx.size, _ptr(idx), _ptr(lo), _ptr(hi),
                            _ptr(nn), _ptr(acc), int(levels), _ptr(best), _ptr(chi), C.byref(st),
                            stream or None))
    return best, float(chi[0]), _stats_dict(st)


def gbk_fit_lm(handle, start_rows, gal, free_param, lo, hi, rel_step=1e-3, max_iter=50, ftol=1e-6,
               stream=0):
    """Levenberg-Marquardt for n_fits rows at once -> (fit_rows [n, P], chi2 [n], iters [n], stats)."""
    S = _stride(handle)
    start = np.ascontiguousarray(start_rows, dtype=np.float32).reshape(-1, S)
    n = start.shape[0]
    g = None if gal is None else np.ascontiguousarray(gal, dtype=np.int32)
    if g is not None and g.size != n:
        raise ValueError("gal must have one entry per fit")
    idx, lo, hi = _box(free_param, lo, hi)
    rows = np.empty((n, S), np.float32)
    chi = np.empty(n, np.float32)
    iters = np.empty(n, np.int32)
    st = gbk_fit_stats()
    _check(lib().gbk_fit_lm(handle, n, _ptr(start), _ptr(g), idx.size, _ptr(idx), _ptr(lo), _ptr(hi),
                            float(rel_step), int(max_iter), float(ftol), _ptr(rows), _ptr(chi),
                            _ptr(iters), C.byref(st), stream or None))
    return rows, chi, iters, _stats_dict(st)


def gbk_fit_ns(handle, base_row, gal, free_param, lo, hi, n_live=256, batch=256, max_batches=200,
               enlarge=0.2, tol=0.01, seed=1, stream=0):
    """Nested sampling -> dict(best_row, best_chi2, mean_row, log_evidence, stats)."""
    S = _stride(handle)
    base = _host_f32(base_row, (S,))
    idx, lo, hi = _box(free_param, lo, hi)
    best = np.empty(S, np.float32)
    mean = np.empty(S, np.float32)
    chi = np.empty(1, np.float32)
    lnz = C.c_double()
    st = gbk_fit_stats()
    _check(lib().gbk_fit_ns(handle, _ptr(base), int(gal), idx.size, _ptr(idx), _ptr(lo), _ptr(hi),
                            int(n_live), int(batch), int(max_batches), float(enlarge), float(tol),
                            int(seed), _ptr(best), _ptr(chi), _ptr(mean), C.byref(lnz), C.byref(st),
                            stream or None))
    return dict(best_row=best, best_chi2=float(chi[0]), mean_row=mean, log_evidence=lnz.value,
                stats=_stats_dict(st))


# ------------------------------------------------------------------------ convenience ----

class Problem:
    """Owns a gbk_problem handle; `eval` allocates outputs with torch on the problem's device."""

    def __init__(self, **desc):
        self.handle = gbk_create_problem(**desc)
        self.info = gbk_get_info(self.handle)

    def close(self):
        if getattr(self, "handle", None):
            gbk_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def set_strategy(self, strategy: int):
        """gbk_set_strategy, keeping `info` (which reports the strategy) up to date."""
        gbk_set_strategy(self.handle, strategy)
        self.info = gbk_get_info(self.handle)

    def set_extraction(self, extraction: int):
        gbk_set_extraction(self.handle, extraction)
        self.info = gbk_get_info(self.handle)

    def eval_vfield(self, params, gal_index=None, want_maps=False, want_resid=False, stream=None):
        """Velocity-field strategy: torch CUDA float32 [K, row_stride] -> dict(chi2[, vmap][, resid])."""
        import torch
        assert params.is_cuda and params.dtype == torch.float32 and params.is_contiguous()
        assert params.ndim == 2 and params.shape[1] == self.info.row_stride
        K = params.shape[0]
        i = self.info
        out = {"chi2": torch.empty(K, dtype=torch.float32, device=params.device)}
        if want_maps:
            out["vmap"] = torch.empty((K, i.ny, i.nx), dtype=torch.float32, device=params.device)
        if want_resid:
            out["resid"] = torch.empty((K, i.ny, i.nx), dtype=torch.float32, device=params.device)
        if gal_index is not None:
            assert gal_index.is_cuda and gal_index.dtype == torch.int32 and gal_index.is_contiguous()
        st = (stream or torch.cuda.current_stream(params.device)).cuda_stream
        gbk_eval_vfield_batch(self.handle, params, gal_index, K, out["chi2"], out.get("vmap"),
                              out.get("resid"), st)
        return out

    def eval(self, params, gal_index=None, want_maps=False, want_resid=False, unfused=False,
             stream=None):
        """params: torch CUDA float32 [K, row_stride] -> dict of torch tensors (chi2[, m0, m1, m2][, resid])."""
        import torch
        assert params.is_cuda and params.dtype == torch.float32 and params.is_contiguous()
        assert params.ndim == 2 and params.shape[1] == self.info.row_stride
        K = params.shape[0]
        dev = params.device
        i = self.info
        out = {"chi2": torch.empty(K, dtype=torch.float32, device=dev)}
        if want_maps:
            for k in ("m0", "m1", "m2"):
                out[k] = torch.empty((K, i.ny, i.nx), dtype=torch.float32, device=dev)
        if want_resid:
            out["resid"] = torch.empty((K, 2, i.ny, i.nx), dtype=torch.float32, device=dev)
        if gal_index is not None:
            assert gal_index.is_cuda and gal_index.dtype == torch.int32 and gal_index.is_contiguous()
        st = (stream or torch.cuda.current_stream(dev)).cuda_stream
        gbk_eval_batch(self.handle, params, gal_index, K, out["chi2"], out.get("m0"), out.get("m1"),
                       out.get("m2"), out.get("resid"), st, unfused=unfused)
        return out
