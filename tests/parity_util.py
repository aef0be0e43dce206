"""Helpers shared by the parity tests: build the same problem for the oracle and for libgbk
from a seeded Workload, and compare outputs with the tolerances of BASELINE.json.

Tolerances (north_star): m0 1e-4 relative, m1 and m2 0.05 km/s absolute, chi^2 1e-4 relative.
"""
from __future__ import annotations

import numpy as np

from paper_1510_01815_b200 import workloads as wl

TOL_M0_REL = 1e-4
TOL_M12_ABS = 0.05
TOL_CHI2_REL = 1e-4
DARK_GUARD = 100.0   # skip spaxels / rows within 100x of the 1e-30 I0 model-dark threshold (A15)


def f32(x) -> float:
    return float(np.float32(x))


def oracle_grid(oracle, w: wl.Workload, fwhm=None, tab=None, tab_dx=0.0, extract=0):
    """Oracle Grid for workload w (Gaussian PSF of `fwhm` data pixels, or w's Moffat image; `tab`:
    a tabulated radial intensity profile, float32 values promoted like every other input)."""
    if w.psf_kind == wl.PSF_GAUSSIAN:
        psf = oracle.psf_gaussian_image(f32(w.psf_fwhm if fwhm is None else fwhm), w.u)
    else:
        img = wl.moffat_image(w.psf_fwhm, w.moffat_beta, w.psf_n).astype(np.float64)
        psf = img / img.sum()
    lsf = oracle.gaussian_taps(f32(w.lsf_sigma) / f32(w.dv) if w.lsf_sigma > 0 else 0.0)
    return oracle.Grid(nx=w.nx, ny=w.ny, nv=w.nv, u=w.u, v_center=f32(w.v_center), dv=f32(w.dv),
                       rc_model=w.rc_model, psf=psf, lsf=lsf,
                       tab=None if tab is None else np.asarray(tab, dtype=np.float32).astype(np.float64),
                       tab_dx=f32(tab_dx), extract=extract)


def gbk_desc(w: wl.Workload, obs: wl.Observed, fwhms=None, **extra):
    """Keyword arguments of gbk.gbk_create_problem for workload w and observation obs."""
    d = dict(nx=w.nx, ny=w.ny, nv=w.nv, u=w.u, v_center=w.v_center, dv=w.dv, rc_model=w.rc_model,
             n_gal=obs.vobs.shape[0] if obs.vobs.ndim == 3 else 1,
             vobs=obs.vobs, verr=obs.verr, sobs=obs.sobs, serr=obs.serr, mask=obs.mask,
             psf_kind=w.psf_kind, lsf_sigma=w.lsf_sigma)
    if w.psf_kind == wl.PSF_GAUSSIAN:
        d["psf_fwhm"] = np.asarray([w.psf_fwhm] if fwhms is None else fwhms, dtype=np.float32)
        d["psf_per_gal"] = fwhms is not None
    else:
        d["psf_image"] = wl.moffat_image(w.psf_fwhm, w.moffat_beta, w.psf_n)
    d.update(extra)
    return d


def single_galaxy_case(oracle, w: wl.Workload, true_row, rng, fwhm=None, tab=None, tab_dx=0.0):
    """Observation of one galaxy: oracle maps of `true_row` + seeded noise / errors / mask."""
    g = oracle_grid(oracle, w, fwhm, tab, tab_dx)
    m0, m1, m2 = oracle.model_maps(g, np.asarray(true_row, dtype=np.float32).astype(np.float64))
    obs = wl.observe(w, m0[None], m1[None], m2[None], rng)
    return g, obs


def compare(oracle_out: dict, gpu_out: dict, rows: np.ndarray, want_maps: bool, label=""):
    """Element-by-element comparison; returns a dict of the worst errors (for reporting)."""
    chi_o = np.asarray(oracle_out["chi2"], dtype=np.float64)
    chi_g = np.asarray(gpu_out["chi2"], dtype=np.float64)
    worst = {"chi2_rel": 0.0, "m0_rel": 0.0, "m1_abs": 0.0, "m2_abs": 0.0, "rows": len(chi_o),
             "skipped_rows": 0}
    inf_o, inf_g = np.isinf(chi_o), np.isinf(chi_g)
    near_dark = np.zeros(len(chi_o), dtype=bool)
    if want_maps:
        i0 = rows[:, wl.IX_I0].astype(np.float64)
        with np.errstate(invalid="ignore"):
            mn = np.nanmin(np.where(np.isfinite(oracle_out["m0"]), oracle_out["m0"], np.inf),
                           axis=(1, 2))
        near_dark = (mn < DARK_GUARD * 1e-30 * i0) & (mn > 1e-30 * i0 / DARK_GUARD)
    assert not np.isnan(chi_g).any(), f"{label}: NaN chi2 from the GPU"
    ok = ~near_dark
    worst["skipped_rows"] = int(near_dark.sum())
    assert np.array_equal(inf_o[ok], inf_g[ok]), f"{label}: +INF rows differ"
    fin = ok & ~inf_o
    if fin.any():
        rel = np.abs(chi_g[fin] - chi_o[fin]) / np.maximum(np.abs(chi_o[fin]), 1e-300)
        worst["chi2_rel"] = float(rel.max())
        assert rel.max() <= TOL_CHI2_REL, f"{label}: chi2 rel err {rel.max():.3e}"
    if want_maps:
        for k in np.nonzero(ok)[0]:
            o0, o1, o2 = (np.asarray(oracle_out[m][k], dtype=np.float64) for m in ("m0", "m1", "m2"))
            g0, g1, g2 = (np.asarray(gpu_out[m][k], dtype=np.float64) for m in ("m0", "m1", "m2"))
            if np.isnan(o0).all():
                assert np.isnan(g0).all() and np.isnan(g1).all() and np.isnan(g2).all()
                continue
            bright = o0 > DARK_GUARD * 1e-30 * float(rows[k, wl.IX_I0])
            if not bright.any():        # the whole map is model-dark (line outside the band)
                continue
            r0 = np.abs(g0 - o0)[bright] / o0[bright]
            d1 = np.abs(g1 - o1)[bright]
            d2 = np.abs(g2 - o2)[bright]
            worst["m0_rel"] = max(worst["m0_rel"], float(r0.max()))
            worst["m1_abs"] = max(worst["m1_abs"], float(d1.max()))
            worst["m2_abs"] = max(worst["m2_abs"], float(d2.max()))
            assert r0.max() <= TOL_M0_REL, f"{label} row {k}: m0 rel err {r0.max():.3e}"
            assert d1.max() <= TOL_M12_ABS, f"{label} row {k}: m1 abs err {d1.max():.3e}"
            assert d2.max() <= TOL_M12_ABS, f"{label} row {k}: m2 abs err {d2.max():.3e}"
    return worst
