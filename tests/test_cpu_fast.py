"""The optimised CPU restatement that bench.py times as a second CPU baseline (oracle/gbk_cpu_fast.c)
computes what the oracle computes: chi^2 within BASELINE.json's 1e-4 relative, on config-1-like and
up-sampled cases, +INF rows included.  (It is float32 and moment-first; the oracle is the literal
pipeline in float64.)"""
import numpy as np
import pytest

from paper_1510_01815_b200 import workloads as wl

import parity_util as pu


@pytest.mark.parametrize("kw", [dict(), dict(u=2, nx=18, ny=15, nv=40), dict(rc_model=wl.RC_RAMP, nx=20, ny=17)])
def test_fast_cpu_baseline_agrees_with_the_oracle(oracle, kw):
    from oracle import gbk_cpu_fast as fast
    w = wl.config(1).scaled(**kw)
    rng = wl.rng_for(1, 77)
    true = wl.cfg1_true_row(rng)[0]
    true[[wl.IX_XO, wl.IX_YO]] = (0.5 * w.nx + 0.3, 0.5 * w.ny - 0.2)
    g, obs = pu.single_galaxy_case(oracle, w, true, rng)
    rows = np.repeat(true[None].astype(np.float64), 12, axis=0)
    b = wl.box(w)
    rows[1:] += 0.1 * (b[:, 1] - b[:, 0]) * rng.uniform(-1, 1, (11, wl.P))
    rows[:, wl.IX_INC] = np.clip(rows[:, wl.IX_INC], 5.0, 85.0)
    rows[:, wl.IX_RT] = np.clip(rows[:, wl.IX_RT], 0.5, None)
    rows = rows.astype(np.float32)
    rows[5, wl.IX_SIG] = -1.0                        # out of domain: +INF on both sides
    ref = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], obs.sobs[0], obs.serr[0], obs.mask[0], rows)["chi2"]
    psf1d = oracle.gaussian_taps(w.u * oracle.fwhm_to_sigma(pu.f32(w.psf_fwhm)))
    lsf = oracle.gaussian_taps(pu.f32(w.lsf_sigma) / pu.f32(w.dv))
    got = fast.eval_rows(nx=w.nx, ny=w.ny, nv=w.nv, u=w.u, v_center=w.v_center, dv=w.dv, rc_model=w.rc_model,
                         psf_taps=psf1d, lsf_taps=lsf, vobs=obs.vobs[0], verr=obs.verr[0], sobs=obs.sobs[0],
                         serr=obs.serr[0], mask=obs.mask[0], params=rows, nthreads=2)
    assert np.array_equal(np.isinf(ref), np.isinf(got)) and np.isinf(got[5])
    fin = np.isfinite(ref)
    assert np.max(np.abs(got[fin] / ref[fin] - 1.0)) <= pu.TOL_CHI2_REL
