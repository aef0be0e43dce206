"""ctypes loader for the CPU oracle (oracle/gbk_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It
never imports the product package `paper_1510_01815_b200`.

Argument marshalling only; every number is computed by the C file, which cites
the passages of PAPER.md it follows.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gbk_oracle.c")
_LIB = os.path.join(_HERE, "libgbk_oracle.so")

P = 10  # xo, yo, pa_deg, inc_deg, vsys, vt, rt, sigma0, r0, i0
P_EPINAT = 12  # ... + a, g (eq. 7)
RC_ARCTAN, RC_RAMP, RC_EPINAT = 0, 1, 2


def row_len(rc_model: int) -> int:
    return P_EPINAT if rc_model == RC_EPINAT else P


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C, double precision, OpenMP over rows)."""
    if force or (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


class _Grid(C.Structure):
    _fields_ = [
        ("nx", C.c_int32), ("ny", C.c_int32), ("nv", C.c_int32), ("u", C.c_int32),
        ("v_center", C.c_double), ("dv", C.c_double),
        ("rc_model", C.c_int32), ("psf_n", C.c_int32), ("psf", C.POINTER(C.c_double)),
        ("lsf_n", C.c_int32), ("lsf", C.POINTER(C.c_double)),
        ("halo_zero", C.c_int32),
        ("tab_n", C.c_int32), ("tab", C.POINTER(C.c_double)), ("tab_dx", C.c_double),
        ("extract", C.c_int32),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp, fp, u8p = C.POINTER(C.c_double), C.POINTER(C.c_float), C.POINTER(C.c_uint8)
        gp = C.POINTER(_Grid)
        L.gbko_gaussian_taps.argtypes = [C.c_double, dp, C.c_int]
        L.gbko_gaussian_taps.restype = C.c_int
        L.gbko_fwhm_to_sigma.argtypes = [C.c_double]
        L.gbko_fwhm_to_sigma.restype = C.c_double
        L.gbko_psf_gaussian_image.argtypes = [C.c_double, C.c_int, dp, C.c_int]
        L.gbko_psf_gaussian_image.restype = C.c_int
        L.gbko_psf_moffat_image.argtypes = [C.c_double, C.c_double, C.c_int, dp]
        L.gbko_psf_moffat_image.restype = C.c_int
        L.gbko_row_valid.argtypes = [dp]
        L.gbko_row_valid.restype = C.c_int
        L.gbko_row_valid_rc.argtypes = [dp, C.c_int]
        L.gbko_row_valid_rc.restype = C.c_int
        L.gbko_table_profile.argtypes = [dp, C.c_int, C.c_double, C.c_double]
        L.gbko_table_profile.restype = C.c_double
        L.gbko_disc_point.argtypes = [dp, C.c_int, C.c_double, C.c_double, dp, dp]
        L.gbko_disc_point.restype = None
        L.gbko_channel_velocity.argtypes = [gp, C.c_int]
        L.gbko_channel_velocity.restype = C.c_double
        L.gbko_fine_coord.argtypes = [C.c_int, C.c_int]
        L.gbko_fine_coord.restype = C.c_double
        L.gbko_model_cube.argtypes = [gp, dp, dp]
        L.gbko_model_cube.restype = None
        L.gbko_conv_lsf.argtypes = [dp, C.c_int, C.c_size_t, dp, C.c_int, dp]
        L.gbko_conv_lsf.restype = None
        L.gbko_conv_psf.argtypes = [dp, C.c_int, C.c_int, C.c_int, dp, C.c_int, dp]
        L.gbko_conv_psf.restype = None
        L.gbko_downsample.argtypes = [dp, C.c_int, C.c_int, C.c_int, C.c_int, dp]
        L.gbko_downsample.restype = None
        L.gbko_moments.argtypes = [dp, C.c_int, C.c_size_t, dp, dp, dp, dp]
        L.gbko_moments.restype = None
        L.gbko_gaussfit.argtypes = [dp, C.c_int, C.c_size_t, dp, dp, dp, dp]
        L.gbko_gaussfit.restype = None
        L.gbko_chi2.argtypes = [dp, dp, dp, fp, fp, fp, fp, u8p, C.c_size_t, C.c_double, dp]
        L.gbko_chi2.restype = C.c_double
        L.gbko_model_maps.argtypes = [gp, dp, dp, dp, dp]
        L.gbko_model_maps.restype = C.c_int
        L.gbko_eval_rows.argtypes = [gp, fp, fp, fp, fp, u8p, fp, C.c_int64, dp, dp, dp, dp, dp,
                                     C.c_int]
        L.gbko_eval_rows.restype = C.c_int
        L.gbko_vfield_rows.argtypes = [gp, fp, fp, u8p, fp, C.c_int64, dp, dp, dp, C.c_int]
        L.gbko_vfield_rows.restype = C.c_int
        L.gbko_max_threads.argtypes = []
        L.gbko_max_threads.restype = C.c_int
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


def _fp(a):
    return a.ctypes.data_as(C.POINTER(C.c_float)) if a is not None else None


def _u8p(a):
    return a.ctypes.data_as(C.POINTER(C.c_uint8)) if a is not None else None


def _c64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _c32(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float32)


# ----------------------------------------------------------------- taps ----

def fwhm_to_sigma(fwhm: float) -> float:
    return float(lib().gbko_fwhm_to_sigma(float(fwhm)))


def gaussian_taps(sigma: float) -> np.ndarray:
    buf = np.zeros(4096, dtype=np.float64)
    R = lib().gbko_gaussian_taps(float(sigma), _dp(buf), buf.size)
    if R < 0:
        raise ValueError("sigma too large for the tap buffer")
    return buf[: 2 * R + 1].copy()


def psf_gaussian_image(fwhm_data_px: float, u: int) -> np.ndarray:
    buf = np.zeros(1023 * 1023, dtype=np.float64)
    n = lib().gbko_psf_gaussian_image(float(fwhm_data_px), int(u), _dp(buf), 1023)
    if n < 0:
        raise ValueError("PSF too large")
    return buf[: n * n].reshape(n, n).copy()


def psf_moffat_image(fwhm_fine_px: float, beta: float, n: int) -> np.ndarray:
    buf = np.zeros(n * n, dtype=np.float64)
    if lib().gbko_psf_moffat_image(float(fwhm_fine_px), float(beta), int(n), _dp(buf)) < 0:
        raise ValueError("psf_n must be odd and positive")
    return buf.reshape(n, n)


# ----------------------------------------------------------------- grid ----

@dataclass
class Grid:
    """Geometry of one observation + the PSF / LSF taps (all float64)."""
    nx: int
    ny: int
    nv: int
    u: int = 1
    v_center: float = 0.0
    dv: float = 1.0
    rc_model: int = RC_ARCTAN
    psf: np.ndarray = field(default_factory=lambda: np.ones((1, 1)))
    lsf: np.ndarray = field(default_factory=lambda: np.ones(1))
    halo_zero: bool = False
    tab: np.ndarray | None = None      # tabulated radial profile T(x_j), x_j = j * tab_dx
    tab_dx: float = 0.0
    extract: int = 0                   # 0: moments; 1: Gaussian-profile fit of every spectrum

    def c(self) -> _Grid:
        self._psf = _c64(self.psf)
        self._lsf = _c64(self.lsf)
        assert self._psf.ndim == 2 and self._psf.shape[0] == self._psf.shape[1]
        assert self._psf.shape[0] % 2 == 1 and self._lsf.size % 2 == 1
        self._tab = None if self.tab is None else _c64(self.tab)
        assert self._tab is None or (self._tab.size >= 2 and self.tab_dx > 0)
        return _Grid(self.nx, self.ny, self.nv, self.u, self.v_center, self.dv, self.rc_model,
                     self._psf.shape[0], _dp(self._psf), self._lsf.size, _dp(self._lsf),
                     1 if self.halo_zero else 0,
                     0 if self._tab is None else self._tab.size, _dp(self._tab), float(self.tab_dx),
                     int(self.extract))

    @property
    def P(self) -> int:
        return row_len(self.rc_model)

    @property
    def ext_shape(self):
        n = self.psf.shape[0]
        return (self.nv + self.lsf.size - 1, self.u * self.ny + n - 1, self.u * self.nx + n - 1)

    def channel_velocities(self) -> np.ndarray:
        g = self.c()
        return np.array([lib().gbko_channel_velocity(C.byref(g), k) for k in range(self.nv)])


# ------------------------------------------------------------ the steps ----

def row_valid(p) -> bool:
    p = _c64(p)
    return bool(lib().gbko_row_valid(_dp(p)))


def row_valid_rc(p, rc_model: int) -> bool:
    p = _c64(p)
    assert p.size >= row_len(rc_model)
    return bool(lib().gbko_row_valid_rc(_dp(p), int(rc_model)))


def table_profile(tab, dx: float, x: float) -> float:
    tab = _c64(tab)
    return float(lib().gbko_table_profile(_dp(tab), tab.size, float(dx), float(x)))


def disc_point(p, rc_model: int, x: float, y: float):
    p = _c64(p)
    assert p.size >= row_len(rc_model)
    I, v = C.c_double(), C.c_double()
    lib().gbko_disc_point(_dp(p), int(rc_model), float(x), float(y), C.byref(I), C.byref(v))
    return I.value, v.value


def fine_coord(a: int, u: int) -> float:
    return float(lib().gbko_fine_coord(int(a), int(u)))


def model_cube(grid: Grid, p) -> np.ndarray:
    p = _c64(p)
    g = grid.c()
    out = np.empty(grid.ext_shape, dtype=np.float64)
    lib().gbko_model_cube(C.byref(g), _dp(p), _dp(out))
    return out


def conv_lsf(cube: np.ndarray, taps: np.ndarray) -> np.ndarray:
    cube, taps = _c64(cube), _c64(taps)
    nc = cube.shape[0]
    plane = int(np.prod(cube.shape[1:]))
    out = np.empty((nc - taps.size + 1,) + cube.shape[1:], dtype=np.float64)
    lib().gbko_conv_lsf(_dp(cube), nc, plane, _dp(taps), taps.size, _dp(out))
    return out


def conv_psf(cube: np.ndarray, img: np.ndarray) -> np.ndarray:
    cube, img = _c64(cube), _c64(img)
    nch, eh, ew = cube.shape
    n = img.shape[0]
    out = np.empty((nch, eh - n + 1, ew - n + 1), dtype=np.float64)
    lib().gbko_conv_psf(_dp(cube), nch, eh, ew, _dp(img), n, _dp(out))
    return out


def downsample(cube: np.ndarray, u: int) -> np.ndarray:
    cube = _c64(cube)
    nch, fh, fw = cube.shape
    assert fh % u == 0 and fw % u == 0
    out = np.empty((nch, fh // u, fw // u), dtype=np.float64)
    lib().gbko_downsample(_dp(cube), nch, fh // u, fw // u, int(u), _dp(out))
    return out


def moments(cube: np.ndarray, vel: np.ndarray):
    cube, vel = _c64(cube), _c64(vel)
    nv = cube.shape[0]
    shp = cube.shape[1:]
    npix = int(np.prod(shp))
    m0, m1, m2 = (np.empty(shp, dtype=np.float64) for _ in range(3))
    lib().gbko_moments(_dp(cube), nv, npix, _dp(vel), _dp(m0), _dp(m1), _dp(m2))
    return m0, m1, m2


def gaussfit(cube: np.ndarray, vel: np.ndarray):
    """Gaussian-profile fit of every spectrum -> (m0, mu, sigma); NaN where the fit fails."""
    cube, vel = _c64(cube), _c64(vel)
    nv = cube.shape[0]
    shp = cube.shape[1:]
    npix = int(np.prod(shp))
    m0, mu, sg = (np.empty(shp, dtype=np.float64) for _ in range(3))
    lib().gbko_gaussfit(_dp(cube), nv, npix, _dp(vel), _dp(m0), _dp(mu), _dp(sg))
    return m0, mu, sg


def chi2(m0, m1, m2, vobs, verr, sobs=None, serr=None, mask=None, dark_level=0.0,
         want_resid=False):
    m0, m1, m2 = _c64(m0), _c64(m1), _c64(m2)
    vobs, verr, sobs, serr = _c32(vobs), _c32(verr), _c32(sobs), _c32(serr)
    mask = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    npix = m0.size
    resid = np.empty((2,) + m0.shape, dtype=np.float64) if want_resid else None
    val = lib().gbko_chi2(_dp(m0), _dp(m1), _dp(m2), _fp(vobs), _fp(verr), _fp(sobs), _fp(serr),
                          _u8p(mask), npix, float(dark_level), _dp(resid))
    return (val, resid) if want_resid else val


def model_maps(grid: Grid, p):
    """Steps 1-5 for one row -> (m0, m1, m2), float64 [ny, nx]."""
    p = _c64(p)
    assert p.size == grid.P
    g = grid.c()
    m0, m1, m2 = (np.empty((grid.ny, grid.nx), dtype=np.float64) for _ in range(3))
    if lib().gbko_model_maps(C.byref(g), _dp(p), _dp(m0), _dp(m1), _dp(m2)) < 0:
        raise MemoryError("oracle allocation failed")
    return m0, m1, m2


def eval_rows(grid: Grid, vobs, verr, sobs, serr, mask, params, want_maps=False,
              want_resid=False, nthreads: int = 0):
    """K float32 rows against one data set -> dict(chi2[, m0, m1, m2][, resid])."""
    params = np.ascontiguousarray(params, dtype=np.float32).reshape(-1, grid.P)
    K = params.shape[0]
    vobs, verr, sobs, serr = _c32(vobs), _c32(verr), _c32(sobs), _c32(serr)
    mask = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    g = grid.c()
    out = {"chi2": np.empty(K, dtype=np.float64)}
    shp = (K, grid.ny, grid.nx)
    if want_maps:
        for k in ("m0", "m1", "m2"):
            out[k] = np.empty(shp, dtype=np.float64)
    if want_resid:
        out["resid"] = np.empty((K, 2, grid.ny, grid.nx), dtype=np.float64)
    rc = lib().gbko_eval_rows(C.byref(g), _fp(vobs), _fp(verr), _fp(sobs), _fp(serr), _u8p(mask),
                              _fp(params), K, _dp(out["chi2"]), _dp(out.get("m0")),
                              _dp(out.get("m1")), _dp(out.get("m2")), _dp(out.get("resid")),
                              int(nthreads))
    if rc != 0:
        raise MemoryError("oracle allocation failed")
    return out


def vfield_rows(grid: Grid, vobs, verr, mask, params, want_maps=False, want_resid=False,
                nthreads: int = 0):
    """Velocity-field strategy: K rows -> dict(chi2[, vmap][, resid])."""
    params = np.ascontiguousarray(params, dtype=np.float32).reshape(-1, grid.P)
    K = params.shape[0]
    vobs, verr = _c32(vobs), _c32(verr)
    mask = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    g = grid.c()
    out = {"chi2": np.empty(K, dtype=np.float64)}
    if want_maps:
        out["vmap"] = np.empty((K, grid.ny, grid.nx), dtype=np.float64)
    if want_resid:
        out["resid"] = np.empty((K, grid.ny, grid.nx), dtype=np.float64)
    lib().gbko_vfield_rows(C.byref(g), _fp(vobs), _fp(verr), _u8p(mask), _fp(params), K,
                           _dp(out["chi2"]), _dp(out.get("vmap")), _dp(out.get("resid")),
                           int(nthreads))
    return out


def max_threads() -> int:
    return int(lib().gbko_max_threads())
