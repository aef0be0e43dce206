"""Seeded synthetic workloads for the five BASELINE.json configs.

This module is the ONE piece shared by the oracle-side tests and the CUDA-side
tests / bench: it draws parameters, noise, error maps and masks from seeded
numpy generators and describes grids.  It holds none of the method's arithmetic
(no disc model, no line profile, no convolution, no moments, no chi^2): clean
model maps are always handed in by the caller (the oracle in tests, the CUDA
path in bench.py's GPU leg).  It imports neither the oracle nor the binding.

The data behind the paper's measurements (its own 1000 mock cubes, GHASP,
DYNAMO) are not available; the inputs below take the shapes,
sizes and value ranges of those workloads (Tables 1-2; the
section 5.2 test sizes; section 6.5) and
stand in for them.  Recipe: DESIGN.md "Input recipe".
"""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import Optional

import numpy as np

SEED = 151001815
P = 10  # xo, yo, pa_deg, inc_deg, vsys, vt, rt, sigma0, r0, i0
IX_XO, IX_YO, IX_PA, IX_INC, IX_VSYS, IX_VT, IX_RT, IX_SIG, IX_R0, IX_I0 = range(10)
RC_ARCTAN, RC_RAMP, RC_EPINAT = 0, 1, 2
PSF_GAUSSIAN, PSF_IMAGE = 0, 1


@dataclass(frozen=True)
class Workload:
    name: str
    nx: int
    ny: int
    nv: int
    u: int
    dv: float
    v_center: float
    rc_model: int
    psf_kind: int
    psf_fwhm: float            # data pixels (Gaussian), or fine pixels (Moffat image)
    lsf_sigma: float           # km/s
    K: int                     # rows per launch
    n_gal: int = 1
    moffat_beta: float = 0.0   # > 0 with PSF_IMAGE
    psf_n: int = 0             # side of the PSF image (PSF_IMAGE)
    sigma0: float = 40.0
    r0_lo: float = 8.0
    r0_hi: float = 8.0
    noise: float = 5.0
    err_lo: float = 5.0
    err_hi: float = 5.0
    mask_rule: str = "m0_rel"  # "m0_rel": m0 >= 1e-3 max;  "m0_q30": m0 >= 30 % quantile
    psf_fwhm_hi: float = 0.0   # > 0: per-galaxy FWHM ~ U[psf_fwhm, psf_fwhm_hi]

    @property
    def npix(self) -> int:
        return self.nx * self.ny

    def scaled(self, **kw) -> "Workload":
        return replace(self, **kw)


def config(n: int) -> Workload:
    """BASELINE.json configs 1..5 (items the JSON leaves open: DESIGN.md)."""
    if n == 1:   # DYNAMO-like low-resolution IFS cube, single evaluation
        return Workload("cfg1", 32, 32, 64, 1, 30.0, 0.0, RC_ARCTAN, PSF_GAUSSIAN, 2.5, 25.0, K=1,
                        sigma0=40.0, r0_lo=4.0, r0_hi=4.0)
    if n == 2:   # LM fit, 2x spatial super-sampling
        return Workload("cfg2", 64, 64, 128, 2, 15.0, 0.0, RC_ARCTAN, PSF_GAUSSIAN, 2.5, 25.0, K=8)
    if n == 3:   # nested-grid brute force -- the headline config
        return Workload("cfg3", 64, 64, 64, 1, 30.0, 0.0, RC_ARCTAN, PSF_GAUSSIAN, 3.0, 30.0,
                        K=4096)
    if n == 4:   # Fabry-Perot-like field, Moffat PSF image, ramp curve
        return Workload("cfg4", 256, 256, 48, 1, 10.0, 0.0, RC_RAMP, PSF_IMAGE, 4.0, 8.0, K=256,
                        moffat_beta=2.5, psf_n=15, sigma0=20.0, r0_lo=10.0, r0_hi=40.0,
                        mask_rule="m0_q30")
    if n == 5:   # 1000-galaxy survey, mixed-galaxy batches
        return Workload("cfg5", 48, 48, 96, 1, 20.0, 0.0, RC_ARCTAN, PSF_GAUSSIAN, 1.5, 25.0,
                        K=16384, n_gal=1000, r0_lo=4.0, r0_hi=10.0, err_lo=3.0, err_hi=15.0,
                        psf_fwhm_hi=4.0)
    raise ValueError("config number must be 1..5")


def rng_for(cfg_number: int, stream: int = 0) -> np.random.Generator:
    return np.random.default_rng([SEED + cfg_number, stream])


# --------------------------------------------------------------- PSF image --

def moffat_image(fwhm_fine_px: float, beta: float, n: int) -> np.ndarray:
    """The PSF *image* a caller supplies for config 4 (an input, like an observed
    PSF frame): Moffat profile point-sampled on an n x n fine grid, float32,
    not normalised here (the library normalises at create)."""
    R = n // 2
    alpha = fwhm_fine_px / (2.0 * np.sqrt(2.0 ** (1.0 / beta) - 1.0))
    j = np.arange(-R, R + 1, dtype=np.float64)
    rr = j[:, None] ** 2 + j[None, :] ** 2
    return ((1.0 + rr / alpha ** 2) ** (-beta)).astype(np.float32)


# --------------------------------------------------------------- parameters --

def box(w: Workload) -> np.ndarray:
    """Prior box [P, 2] (Table 2 style, widened as BASELINE.json says)."""
    b = np.zeros((P, 2))
    b[IX_XO] = (0.4 * w.nx, 0.6 * w.nx)
    b[IX_YO] = (0.4 * w.ny, 0.6 * w.ny)
    b[IX_PA] = (0.0, 360.0)
    b[IX_INC] = (20.0, 80.0)
    b[IX_VSYS] = (-50.0, 50.0)
    b[IX_VT] = (50.0, 300.0)
    b[IX_RT] = (1.0, 8.0)
    b[IX_SIG] = (w.sigma0, w.sigma0)
    b[IX_R0] = (w.r0_lo, w.r0_hi)
    b[IX_I0] = (1.0, 1.0)
    return b


def draw_rows(w: Workload, rng: np.random.Generator, n: int) -> np.ndarray:
    """n rows uniform in the prior box, float32 [n, P]."""
    b = box(w)
    r = b[:, 0] + (b[:, 1] - b[:, 0]) * rng.random((n, P))
    return r.astype(np.float32)


def cfg1_trial_row() -> np.ndarray:
    return np.array([[16.3, 15.8, 37.0, 55.0, 12.0, 200.0, 3.0, 40.0, 4.0, 1.0]], dtype=np.float32)


def cfg1_true_row(rng: np.random.Generator) -> np.ndarray:
    t = cfg1_trial_row().astype(np.float64)
    half = np.array([0.5, 0.5, 5.0, 5.0, 5.0, 20.0, 0.5])
    t[0, :7] += half * rng.uniform(-1.0, 1.0, 7)
    return t.astype(np.float32)


def nested_grid_rows(w: Workload, true_row: np.ndarray, level: int = 0,
                     centre: Optional[np.ndarray] = None, nodes: int = 8) -> np.ndarray:
    """Config 3: nodes^4 rows over (PA, i, V_t, r_t); centre, V_sys, sigma0, r0, I0 at truth.
    Level l spacing h = (hi-lo)/(nodes*2^l); nodes at c + (j - (nodes-1)/2) h (DESIGN A19)."""
    b = box(w)
    free = [IX_PA, IX_INC, IX_VT, IX_RT]
    c = np.array([0.5 * (b[i, 0] + b[i, 1]) for i in free]) if centre is None else np.asarray(centre)
    axes = []
    for n_i, i in enumerate(free):
        h = (b[i, 1] - b[i, 0]) / (nodes * 2 ** level)
        ax = c[n_i] + (np.arange(nodes) - 0.5 * (nodes - 1)) * h
        if i == IX_PA:
            ax = np.mod(ax, 360.0)
        else:
            lo_shift = max(0.0, b[i, 0] - ax[0])
            hi_shift = max(0.0, ax[-1] - b[i, 1])
            ax = ax + lo_shift - hi_shift
        axes.append(ax)
    mesh = np.stack(np.meshgrid(*axes, indexing="ij"), axis=-1).reshape(-1, 4)
    rows = np.repeat(np.asarray(true_row, dtype=np.float64).reshape(1, P), mesh.shape[0], axis=0)
    rows[:, free] = mesh
    return rows.astype(np.float32)


def lm_rows(w: Workload, base: np.ndarray, rel_step: float = 1e-3) -> np.ndarray:
    """Config 2/5: base row + 7 forward differences (step = rel_step x box width) -> [8, P]."""
    b = box(w)
    free = [IX_XO, IX_YO, IX_PA, IX_INC, IX_VSYS, IX_VT, IX_RT]
    rows = np.repeat(np.asarray(base, dtype=np.float64).reshape(1, P), 8, axis=0)
    for j, i in enumerate(free):
        rows[j + 1, i] += rel_step * (b[i, 1] - b[i, 0])
    return rows.astype(np.float32)


# ------------------------------------------------------------ observations --

@dataclass
class Observed:
    vobs: np.ndarray   # float32 [n_gal, ny, nx]
    verr: np.ndarray
    sobs: np.ndarray
    serr: np.ndarray
    mask: np.ndarray   # uint8, 0 = masked


def observe(w: Workload, m0: np.ndarray, m1: np.ndarray, m2: np.ndarray,
            rng: np.random.Generator) -> Observed:
    """Turn clean model maps [.., ny, nx] (supplied by the caller) into an observation:
    per-spaxel errors ~ U[err_lo, err_hi], Gaussian noise (sigma = w.noise, or the
    per-spaxel error when err_lo != err_hi), mask from an m0 threshold."""
    m0 = np.asarray(m0, dtype=np.float64)
    shp = m0.shape
    if w.err_lo == w.err_hi:
        verr = np.full(shp, w.err_lo)
        serr = np.full(shp, w.err_lo)
        nv_, ns_ = w.noise, w.noise
    else:
        verr = rng.uniform(w.err_lo, w.err_hi, shp)
        serr = rng.uniform(w.err_lo, w.err_hi, shp)
        nv_, ns_ = verr, serr
    vobs = np.asarray(m1, dtype=np.float64) + nv_ * rng.standard_normal(shp)
    sobs = np.asarray(m2, dtype=np.float64) + ns_ * rng.standard_normal(shp)
    flat = m0.reshape(-1, shp[-2] * shp[-1]) if m0.ndim > 2 else m0.reshape(1, -1)
    if w.mask_rule == "m0_rel":
        thr = 1e-3 * np.nanmax(flat, axis=1)
    elif w.mask_rule == "m0_q30":
        thr = np.nanquantile(flat, 0.30, axis=1)
    else:
        raise ValueError(w.mask_rule)
    mask = (flat >= thr[:, None]).reshape(shp)
    mask &= np.isfinite(vobs) & np.isfinite(sobs)
    vobs = np.where(mask, vobs, 0.0)
    sobs = np.where(mask, sobs, 0.0)
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    return Observed(f32(vobs), f32(verr), f32(sobs), f32(serr),
                    np.ascontiguousarray(mask, dtype=np.uint8))


def galaxy_fwhms(w: Workload, rng: np.random.Generator) -> np.ndarray:
    """Per-galaxy Gaussian PSF FWHM in data pixels, float32 [n_gal]."""
    if w.psf_fwhm_hi > 0.0:
        return rng.uniform(w.psf_fwhm, w.psf_fwhm_hi, w.n_gal).astype(np.float32)
    return np.full(w.n_gal, w.psf_fwhm, dtype=np.float32)


def shard_rows(K: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous block of rows [lo, hi) owned by `rank` (rows are independent: no
    collective on the data path)."""
    base, rem = divmod(K, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)
