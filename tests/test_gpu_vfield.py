"""Parity of gbk_eval_vfield_batch (velocity-field modelling strategy) with the
CPU oracle, element by element on the same seeded inputs.  Tolerances: velocity 0.05 km/s absolute
(BASELINE.json's m1 tolerance), chi^2 1e-4 relative.
"""
import numpy as np
import pytest

from paper_1510_01815_b200 import workloads as wl

import parity_util as pu

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("the gpu tests need a CUDA device")
    return torch


@pytest.fixture(scope="module")
def gbk():
    from paper_1510_01815_b200 import gbk as g
    g.lib()
    return g


def _compare(ref, got, label):
    chi_o, chi_g = np.asarray(ref["chi2"]), np.asarray(got["chi2"], dtype=np.float64)
    assert not np.isnan(chi_g).any(), label
    assert np.array_equal(np.isinf(chi_o), np.isinf(chi_g)), f"{label}: +INF rows differ"
    fin = np.isfinite(chi_o)
    rel = np.abs(chi_g[fin] - chi_o[fin]) / np.maximum(chi_o[fin], 1e-300)
    assert rel.size == 0 or rel.max() <= pu.TOL_CHI2_REL, f"{label}: chi2 rel err {rel.max():.3e}"
    worst_v = 0.0
    if "vmap" in ref:
        v_o, v_g = ref["vmap"], got["vmap"].astype(np.float64)
        assert np.array_equal(np.isnan(v_o), np.isnan(v_g)), label
        ok = ~np.isnan(v_o)
        worst_v = float(np.max(np.abs(v_o[ok] - v_g[ok]))) if ok.any() else 0.0
        assert worst_v <= pu.TOL_M12_ABS, f"{label}: velocity abs err {worst_v:.3e}"
    if "resid" in ref:
        r_o, r_g = ref["resid"], got["resid"].astype(np.float64)
        assert np.array_equal(np.isnan(r_o), np.isnan(r_g)), label
        ok = ~np.isnan(r_o)
        assert np.max(np.abs(r_o[ok] - r_g[ok])) <= 0.02, label     # 0.05 km/s / min error 3 km/s
    return dict(chi2_rel=float(rel.max()) if rel.size else 0.0, v_abs=worst_v)


def _case(oracle, cfg, **scale):
    w = wl.config(cfg).scaled(**scale)
    rng = wl.rng_for(cfg, 21)
    true = wl.draw_rows(w, rng, 1)[0]
    g, obs = pu.single_galaxy_case(oracle, w, true, rng)
    return w, g, obs, true, rng


@pytest.mark.parametrize("cfg,scale,K", [(1, {}, 9), (3, dict(nx=37, ny=29), 130),
                                         (4, dict(nx=96, ny=80, nv=16), 33)])
def test_vfield_maps_residuals_and_chi2(oracle, torch_cuda, gbk, cfg, scale, K):
    torch = torch_cuda
    w, g, obs, true, rng = _case(oracle, cfg, **scale)
    rows = wl.draw_rows(w, rng, K)
    rows[0] = true
    rows[1, wl.IX_XO], rows[1, wl.IX_YO] = 5.0, 7.0        # centre exactly on a spaxel: r = 0 (A8)
    rows[2, wl.IX_SIG:] = np.nan                           # sigma_0, r_0, I_0 are not part of eq. 8
    ref = oracle.vfield_rows(g, obs.vobs[0], obs.verr[0], obs.mask[0], rows, want_maps=True,
                             want_resid=True)
    with gbk.Problem(**pu.gbk_desc(w, obs)) as prob:
        p = torch.from_numpy(rows).cuda()
        out = prob.eval_vfield(p, want_maps=True, want_resid=True)
        chi_only = prob.eval_vfield(p)["chi2"]
        torch.cuda.synchronize()
        got = {k: v.cpu().numpy() for k, v in out.items()}
        assert np.array_equal(got["chi2"], chi_only.cpu().numpy())      # both instantiations agree
        again = prob.eval_vfield(p)["chi2"].cpu().numpy()
        assert np.array_equal(again, got["chi2"])                       # bit-reproducible
    print("vfield", cfg, _compare(ref, got, f"vfield cfg{cfg}"))


def test_vfield_domain_rule_and_empty_batch(oracle, torch_cuda, gbk):
    torch = torch_cuda
    w, g, obs, true, rng = _case(oracle, 1, nx=13, ny=9)
    rows = np.repeat(true[None], 7, axis=0)
    rows[1, wl.IX_RT] = 0.0
    rows[2, wl.IX_INC] = 90.0
    rows[3, wl.IX_VT] = np.nan
    rows[4, wl.IX_XO] = np.inf
    rows[5, wl.IX_VT] = 1e6             # absurd but finite in FP32 and FP64 alike
    rows[6, wl.IX_PA] = -725.0          # any angle is fine
    ref = oracle.vfield_rows(g, obs.vobs[0], obs.verr[0], obs.mask[0], rows, want_maps=True,
                             want_resid=True)
    assert np.isinf(ref["chi2"][1:5]).all() and np.isfinite(ref["chi2"][[0, 5, 6]]).all()
    with gbk.Problem(**pu.gbk_desc(w, obs)) as prob:
        out = prob.eval_vfield(torch.from_numpy(rows).cuda(), want_maps=True, want_resid=True)
        got = {k: v.cpu().numpy() for k, v in out.items()}
        empty = prob.eval_vfield(torch.empty((0, wl.P), dtype=torch.float32, device="cuda"))
        assert empty["chi2"].numel() == 0
    chi_o, chi_g = ref["chi2"], got["chi2"]
    assert np.array_equal(np.isinf(chi_o), np.isinf(chi_g))
    assert chi_g[5] == pytest.approx(chi_o[5], rel=1e-4)
    for k in (0, 6):
        assert chi_g[k] == pytest.approx(chi_o[k], rel=1e-4)
        assert np.max(np.abs(got["vmap"][k] - ref["vmap"][k])) <= pu.TOL_M12_ABS
    for k in (1, 2, 3, 4):
        assert np.isnan(got["vmap"][k]).all()


def test_vfield_mixed_galaxies(oracle, torch_cuda, gbk):
    torch = torch_cuda
    n_gal = 5
    w = wl.config(5).scaled(n_gal=n_gal, nx=31, ny=26, nv=32)
    rng = wl.rng_for(5, 22)
    trues = wl.draw_rows(w, rng, n_gal)
    g = pu.oracle_grid(oracle, w, 2.0)
    maps = [oracle.model_maps(g, t.astype(np.float64)) for t in trues]
    obs = wl.observe(w, *(np.stack([m[i] for m in maps]) for i in range(3)), rng)
    K = 41
    rows = wl.draw_rows(w, rng, K)
    gal = rng.integers(0, n_gal, K).astype(np.int32)
    with gbk.Problem(**pu.gbk_desc(w, obs, fwhms=np.full(n_gal, 2.0, np.float32))) as prob:
        out = prob.eval_vfield(torch.from_numpy(rows).cuda(), torch.from_numpy(gal).cuda(),
                               want_maps=True, want_resid=True)
        got = {k: v.cpu().numpy() for k, v in out.items()}
    for gi in range(n_gal):
        sel = np.nonzero(gal == gi)[0]
        if sel.size == 0:
            continue
        ref = oracle.vfield_rows(g, obs.vobs[gi], obs.verr[gi], obs.mask[gi], rows[sel],
                                 want_maps=True, want_resid=True)
        _compare(ref, {k: v[sel] for k, v in got.items()}, f"vfield gal {gi}")


def test_vfield_full_size_sampled_rows(oracle, torch_cuda, gbk):
    """Config-3 shape at the launch size bench.py's velocity-field leg times (K = 4096)."""
    torch = torch_cuda
    w, g, obs, true, rng = _case(oracle, 3)
    rows = wl.nested_grid_rows(w, true, level=1, centre=true[[wl.IX_PA, wl.IX_INC, wl.IX_VT, wl.IX_RT]])
    with gbk.Problem(**pu.gbk_desc(w, obs)) as prob:
        chi = prob.eval_vfield(torch.from_numpy(rows).cuda())["chi2"].cpu().numpy()
    sel = np.concatenate([[0, 1, 4095], rng.integers(0, 4096, 29)])
    ref = oracle.vfield_rows(g, obs.vobs[0], obs.verr[0], obs.mask[0], rows[sel])
    _compare(ref, {"chi2": chi[sel]}, "vfield cfg3 full")


def test_vfield_epinat_curve(oracle, torch_cuda, gbk):
    """Eq. 7 with the velocity-field strategy, the GHASP model:
    rows of 12 floats, the slopes a, g in slots 10 and 11."""
    torch = torch_cuda
    w, g, obs, true, rng = _case(oracle, 3, nx=45, ny=38)
    w = w.scaled(rc_model=wl.RC_EPINAT)
    g = pu.oracle_grid(oracle, w)
    K = 64
    rows = np.concatenate([wl.draw_rows(w, rng, K), rng.uniform(0.5, 2.5, (K, 2)).astype(np.float32)], axis=1)
    rows[0, wl.IX_XO], rows[0, wl.IX_YO] = 20.0, 17.0   # r = 0 on a spaxel
    rows[1, 10] = 0.0                                  # a <= 0: out of domain
    rows[2, 11] = np.nan
    rows[3, 10:] = (1.0, 1.0)                          # the paper's initial slopes
    rows[4, wl.IX_SIG] = np.nan                        # sigma_0 is not part of eq. 8: harmless here
    ref = oracle.vfield_rows(g, obs.vobs[0], obs.verr[0], obs.mask[0], rows, want_maps=True,
                             want_resid=True)
    assert np.isinf(ref["chi2"][[1, 2]]).all() and np.isfinite(np.delete(ref["chi2"], [1, 2])).all()
    with gbk.Problem(**pu.gbk_desc(w, obs)) as prob:
        assert prob.info.row_stride == gbk.GBK_P_EPINAT == 12
        p = torch.from_numpy(rows).cuda()
        out = prob.eval_vfield(p, want_maps=True, want_resid=True)
        got = {k: v.cpu().numpy() for k, v in out.items()}
    print("vfield epinat", _compare(ref, got, "vfield epinat"))
