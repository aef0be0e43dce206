"""SURVEY.md section 8(f) item 3 on the GPU: the Epinat rotation curve (eq. 7) inside
the intensity-cube strategy, and a tabulated "user-specified" radial intensity profile (PAPER.md:106,
reading A22) -- fused and unfused paths against the oracle, at config-1 and config-3 size, element by
element at BASELINE.json's tolerances (parity_util.compare).
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


def _eval(torch, gbk, desc, rows, unfused=False, want_maps=True):
    with gbk.Problem(**desc) as prob:
        out = prob.eval(torch.from_numpy(np.ascontiguousarray(rows, dtype=np.float32)).cuda(),
                        want_maps=want_maps, unfused=unfused)
        torch.cuda.synchronize()
        return {k: v.cpu().numpy() for k, v in out.items()}


def _epinat_rows(w, rng, K, true12):
    rows = np.repeat(np.asarray(true12, dtype=np.float64)[None], K, axis=0)
    b = wl.box(w)
    width = np.concatenate([b[:, 1] - b[:, 0], [2.0, 2.0]])
    rows[1:] += 0.1 * width * rng.uniform(-1, 1, (K - 1, 12))
    rows[:, wl.IX_INC] = np.clip(rows[:, wl.IX_INC], 5.0, 85.0)
    rows[:, wl.IX_RT] = np.clip(rows[:, wl.IX_RT], 0.5, None)
    rows[:, 10:] = np.clip(rows[:, 10:], 0.3, 3.0)
    return rows.astype(np.float32)


@pytest.mark.parametrize("cfg,tile", [(1, (0, 0)), (1, (12, 10)), (3, (0, 0))])
def test_cube_with_the_epinat_curve(oracle, torch_cuda, gbk, cfg, tile):
    w = wl.config(cfg).scaled(rc_model=wl.RC_EPINAT)
    rng = wl.rng_for(cfg, 31)
    true = np.concatenate([wl.cfg1_true_row(rng)[0] if cfg == 1 else wl.draw_rows(w, rng, 1)[0], [1.4, 0.9]])
    g, obs = pu.single_galaxy_case(oracle, w, true, rng)
    rows = _epinat_rows(w, rng, 10 if cfg == 1 else 6, true)
    rows[2, 10:] = (0.8, 1.6)           # g > a: the curve keeps rising
    rows[3, 10:] = (1.0, 1.0)           # the paper's starting slopes
    ref = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], obs.sobs[0], obs.serr[0], obs.mask[0], rows,
                           want_maps=True)
    desc = pu.gbk_desc(w, obs, tile_w=tile[0], tile_h=tile[1])
    print("epinat cube", cfg, tile, pu.compare(ref, _eval(torch_cuda, gbk, desc, rows), rows, True,
                                               f"epinat cube cfg{cfg} tile={tile}"))
    if cfg == 1:
        print("epinat cube unfused", pu.compare(ref, _eval(torch_cuda, gbk, desc, rows, unfused=True), rows,
                                                True, "epinat cube unfused"))
        bad = rows[:3].copy()
        bad[1, 10] = 0.0
        bad[2, 11] = np.nan
        got = _eval(torch_cuda, gbk, desc, bad)
        assert np.isfinite(got["chi2"][0]) and np.isposinf(got["chi2"][1:]).all()
        assert np.isnan(got["m1"][1:]).all()


def test_epinat_cube_full_launch_and_far_wing(oracle, torch_cuda, gbk):
    """K = 4096 Epinat rows of config-3 shape in one launch (sampled against the oracle), plus rows whose
    lines leave a short band (the FP64 geometry path with eq. 7)."""
    torch = torch_cuda
    w = wl.config(3).scaled(rc_model=wl.RC_EPINAT)
    rng = wl.rng_for(3, 32)
    true = np.concatenate([wl.draw_rows(w, rng, 1)[0], [1.2, 1.0]])
    g, obs = pu.single_galaxy_case(oracle, w, true, rng)
    rows = np.concatenate([wl.draw_rows(w, rng, 4096), rng.uniform(0.5, 2.5, (4096, 2)).astype(np.float32)], axis=1)
    got = _eval(torch, gbk, pu.gbk_desc(w, obs), rows, want_maps=False)
    pick = rng.choice(4096, size=24, replace=False)
    ref = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], obs.sobs[0], obs.serr[0], obs.mask[0], rows[pick])
    print("epinat cfg3 full", pu.compare(ref, {"chi2": got["chi2"][pick]}, rows[pick], False, "epinat cfg3 full"))
    ws = wl.config(1).scaled(rc_model=wl.RC_EPINAT, nx=18, ny=15, nv=20, dv=10.0, lsf_sigma=6.0, psf_fwhm=1.7)
    trues = np.array([8.3, 7.1, 140.0, 50.0, 8.0, 180.0, 2.0, 12.0, 3.0, 1.5, 1.3, 0.9], dtype=np.float32)
    gs, obss = pu.single_galaxy_case(oracle, ws, trues, rng)
    far = []
    for nsig in (0.0, 4.0, 8.0, 10.5):
        for a_, g_ in ((1.3, 0.9), (0.7, 1.8)):
            r = trues.copy()
            r[wl.IX_VSYS] = 100.0 + nsig * 12.0
            r[wl.IX_VT] = 280.0
            r[10:] = (a_, g_)
            far.append(r)
    far = np.stack(far)
    ref = oracle.eval_rows(gs, obss.vobs[0], obss.verr[0], obss.sobs[0], obss.serr[0], obss.mask[0], far,
                           want_maps=True)
    print("epinat far wing", pu.compare(ref, _eval(torch, gbk, pu.gbk_desc(ws, obss), far), far, True,
                                        "epinat far wing"))


def _tables(rng):
    x = np.arange(0.0, 9.0, 0.05)
    return [("sersic-like exp(-x^0.7)", np.exp(-x ** 0.7).astype(np.float32), 0.05),
            ("ring", (np.exp(-0.5 * ((x - 1.5) / 0.6) ** 2) + 0.05 * np.exp(-x / 3)).astype(np.float32), 0.05),
            ("coarse random", rng.uniform(0.2, 1.0, 7).astype(np.float32), 0.9)]


@pytest.mark.parametrize("cfg,tile", [(1, (0, 0)), (1, (9, 16)), (3, (0, 0))])
def test_cube_with_a_tabulated_intensity_profile(oracle, torch_cuda, gbk, cfg, tile):
    w = wl.config(cfg)
    rng = wl.rng_for(cfg, 33)
    true = wl.cfg1_true_row(rng)[0] if cfg == 1 else wl.draw_rows(w, rng, 1)[0]
    for name, tab, dx in _tables(rng):
        g, obs = pu.single_galaxy_case(oracle, w, true, rng, tab=tab, tab_dx=dx)
        rows = np.repeat(true[None].astype(np.float64), 8 if cfg == 1 else 5, axis=0)
        b = wl.box(w)
        rows[1:] += 0.1 * (b[:, 1] - b[:, 0]) * rng.uniform(-1, 1, (rows.shape[0] - 1, wl.P))
        rows[:, wl.IX_R0] = true[wl.IX_R0] * rng.uniform(0.6, 1.6, rows.shape[0])     # the table's scale length
        rows[:, wl.IX_INC] = np.clip(rows[:, wl.IX_INC], 5.0, 85.0)
        rows[:, wl.IX_RT] = np.clip(rows[:, wl.IX_RT], 0.5, None)
        rows[-1, wl.IX_VSYS] = 0.5 * w.nv * w.dv + 7.0 * true[wl.IX_SIG]    # line centred 7 sigma_0 outside the band:
        rows = rows.astype(np.float32)                                       # the FP64 geometry path with the table
        ref = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], obs.sobs[0], obs.serr[0], obs.mask[0], rows,
                               want_maps=True)
        desc = pu.gbk_desc(w, obs, tile_w=tile[0], tile_h=tile[1], intensity_table=tab, intensity_dx=dx)
        print("table", name, cfg, tile, pu.compare(ref, _eval(torch_cuda, gbk, desc, rows), rows, True,
                                                   f"table {name} cfg{cfg} tile={tile}"))
        if cfg == 1 and tile == (0, 0):
            print("table unfused", name, pu.compare(ref, _eval(torch_cuda, gbk, desc, rows, unfused=True),
                                                    rows, True, f"table {name} unfused"))


def test_create_rejects_bad_tables(oracle, torch_cuda, gbk):
    w = wl.config(1)
    rng = wl.rng_for(1, 34)
    g, obs = pu.single_galaxy_case(oracle, w, wl.cfg1_true_row(rng)[0], rng)
    for tab, dx in ((np.array([1.0], np.float32), 1.0), (np.array([1.0, np.nan], np.float32), 1.0),
                    (np.array([1.0, -0.5], np.float32), 1.0), (np.array([1.0, 0.5], np.float32), 0.0)):
        with pytest.raises(gbk.GbkError) as e:
            gbk.Problem(**pu.gbk_desc(w, obs, intensity_table=tab, intensity_dx=dx))
        assert e.value.code == gbk.GBK_ERR_ARG


# ------------------------ Gaussian-profile extraction ----

@pytest.mark.parametrize("cfg,kw", [(1, {}), (1, dict(u=2, nx=20, ny=18, nv=48)), (3, {})])
def test_gaussian_profile_extraction(oracle, torch_cuda, gbk, cfg, kw):
    """GBK_EXTRACT_GAUSSFIT: velocity and dispersion maps from a Gaussian fitted to every spectrum, through
    gbk_eval_batch (which then runs the multi-kernel pipeline) against the oracle's extract = 1.  Maps are
    compared at the unmasked spaxels (the observation's mask keeps m0 >= 1e-3 max); where the oracle's fit
    fails (NaN) the GPU's must fail too."""
    torch = torch_cuda
    w = wl.config(cfg).scaled(**kw)
    rng = wl.rng_for(cfg, 41)
    true = wl.cfg1_true_row(rng)[0] if cfg == 1 else wl.draw_rows(w, rng, 1)[0]
    g = pu.oracle_grid(oracle, w, extract=1)
    m0, m1, m2 = oracle.model_maps(g, true.astype(np.float64))
    obs = wl.observe(w, m0[None], m1[None], m2[None], rng)
    rows = np.repeat(true[None].astype(np.float64), 6 if cfg == 1 else 3, axis=0)
    b = wl.box(w)
    rows[1:] += 0.05 * (b[:, 1] - b[:, 0]) * rng.uniform(-1, 1, (rows.shape[0] - 1, wl.P))
    rows[:, wl.IX_INC] = np.clip(rows[:, wl.IX_INC], 5.0, 85.0)
    rows[:, wl.IX_RT] = np.clip(rows[:, wl.IX_RT], 0.5, None)
    rows = rows.astype(np.float32)
    ref = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], obs.sobs[0], obs.serr[0], obs.mask[0], rows,
                           want_maps=True)
    ref_mom = oracle.eval_rows(pu.oracle_grid(oracle, w), obs.vobs[0], obs.verr[0], obs.sobs[0], obs.serr[0],
                               obs.mask[0], rows, want_maps=True)
    with gbk.Problem(**pu.gbk_desc(w, obs)) as prob:
        prob.set_extraction(gbk.GBK_EXTRACT_GAUSSFIT)
        assert prob.info.extraction == gbk.GBK_EXTRACT_GAUSSFIT
        out = prob.eval(torch.from_numpy(rows).cuda(), want_maps=True)
        torch.cuda.synchronize()
        got = {k: v.cpu().numpy().astype(np.float64) for k, v in out.items()}
        prob.set_extraction(gbk.GBK_EXTRACT_MOMENTS)            # and back: the fused kernel again
        back = prob.eval(torch.from_numpy(rows).cuda(), want_maps=True)
        mom = {k: v.cpu().numpy().astype(np.float64) for k, v in back.items()}
    m = obs.mask[0] != 0
    worst = {}
    for k in range(rows.shape[0]):
        assert np.array_equal(np.isnan(ref["m1"][k][m]), np.isnan(got["m1"][k][m]))
        ok = m & np.isfinite(ref["m1"][k])
        worst["m0"] = max(worst.get("m0", 0), float(np.max(np.abs(got["m0"][k][ok] / ref["m0"][k][ok] - 1))))
        worst["m1"] = max(worst.get("m1", 0), float(np.max(np.abs(got["m1"][k][ok] - ref["m1"][k][ok]))))
        worst["m2"] = max(worst.get("m2", 0), float(np.max(np.abs(got["m2"][k][ok] - ref["m2"][k][ok]))))
    fin = np.isfinite(ref["chi2"])
    assert np.array_equal(fin, np.isfinite(got["chi2"]))
    worst["chi2"] = float(np.max(np.abs(got["chi2"][fin] / ref["chi2"][fin] - 1))) if fin.any() else 0.0
    print("gaussfit", cfg, kw, worst)
    assert worst["m0"] <= pu.TOL_M0_REL and worst["m1"] <= pu.TOL_M12_ABS and worst["m2"] <= pu.TOL_M12_ABS
    assert worst["chi2"] <= pu.TOL_CHI2_REL
    pu.compare(ref_mom, mom, rows, True, "moments after switching back")
    # the two extractions are different things: beam smearing separates them
    assert np.nanmax(np.abs(ref["m2"][0][m] - ref_mom["m2"][0][m])) > 0.05


def test_gaussian_profile_extraction_with_an_image_psf_and_two_galaxies(oracle, torch_cuda, gbk):
    """GBK_EXTRACT_GAUSSFIT on the other branches of the multi-kernel pipeline: a 9 x 9 image PSF (direct
    2-D sum from a shared-memory tile) and a batch that mixes two data sets."""
    torch = torch_cuda
    w = wl.config(4).scaled(nx=26, ny=22, nv=40, psf_n=9, sigma0=25.0, r0_lo=5.0, r0_hi=9.0, mask_rule="m0_rel")
    rng = wl.rng_for(4, 42)
    trues = wl.draw_rows(w, rng, 2)
    img = wl.moffat_image(w.psf_fwhm, w.moffat_beta, w.psf_n).astype(np.float64)
    g = oracle.Grid(nx=w.nx, ny=w.ny, nv=w.nv, u=1, v_center=0.0, dv=pu.f32(w.dv), rc_model=w.rc_model,
                    psf=img / img.sum(), lsf=oracle.gaussian_taps(pu.f32(w.lsf_sigma) / pu.f32(w.dv)), extract=1)
    clean = [oracle.model_maps(g, t.astype(np.float64)) for t in trues]
    obs = wl.observe(w, *(np.stack([c[i] for c in clean]) for i in range(3)), rng)
    rows = np.concatenate([np.repeat(t[None], 3, axis=0) for t in trues]).astype(np.float64)
    rows[[1, 2, 4, 5], wl.IX_VT] += rng.uniform(-15, 15, 4)
    rows = rows.astype(np.float32)
    gal = np.array([0, 0, 0, 1, 1, 1], dtype=np.int32)
    perm = rng.permutation(6)
    rows, gal = rows[perm], gal[perm]
    d = pu.gbk_desc(w, obs)
    d["psf_image"] = wl.moffat_image(w.psf_fwhm, w.moffat_beta, w.psf_n)
    with gbk.Problem(**d) as prob:
        prob.set_extraction(gbk.GBK_EXTRACT_GAUSSFIT)
        out = prob.eval(torch.from_numpy(rows).cuda(), torch.from_numpy(gal).cuda(), want_maps=True)
        got = {k: v.cpu().numpy().astype(np.float64) for k, v in out.items()}
    for gi in range(2):
        sel = np.nonzero(gal == gi)[0]
        ref = oracle.eval_rows(g, obs.vobs[gi], obs.verr[gi], obs.sobs[gi], obs.serr[gi], obs.mask[gi], rows[sel],
                               want_maps=True)
        m = obs.mask[gi] != 0
        for j, k in enumerate(sel):
            ok = m & np.isfinite(ref["m1"][j])
            assert np.array_equal(np.isnan(ref["m1"][j][m]), np.isnan(got["m1"][k][m]))
            assert np.max(np.abs(got["m1"][k][ok] - ref["m1"][j][ok])) <= pu.TOL_M12_ABS
            assert np.max(np.abs(got["m2"][k][ok] - ref["m2"][j][ok])) <= pu.TOL_M12_ABS
            assert np.max(np.abs(got["m0"][k][ok] / ref["m0"][j][ok] - 1.0)) <= pu.TOL_M0_REL
        fin = np.isfinite(ref["chi2"])
        assert np.array_equal(fin, np.isfinite(got["chi2"][sel]))
        assert np.max(np.abs(got["chi2"][sel][fin] / ref["chi2"][fin] - 1.0)) <= pu.TOL_CHI2_REL


@pytest.mark.parametrize("seed", range(int(__import__("os").environ.get("GBK_MODEL_FUZZ_CASES", "60"))))
def test_random_shapes_with_the_epinat_curve_and_tabulated_profiles(oracle, torch_cuda, gbk, seed):
    """Seeded random problems for the section-8(f) models: odd grid sizes, up-sampling, Gaussian or image PSFs,
    delta or wide LSFs, explicit or automatic tiles -- with the Epinat curve (random slopes), a random tabulated
    profile, or both; chi^2 and maps against the oracle, fused path (and the unfused one on every fourth case)."""
    rng = np.random.default_rng(7_1510_01815 + seed)
    nx, ny = int(rng.integers(4, 30)), int(rng.integers(4, 26))
    u = int(rng.choice([1, 1, 2, 3]))
    nv = int(rng.integers(14, 60))
    dv = float(rng.choice([10.0, 20.0, 30.0]))
    epinat = bool(rng.random() < 0.7)
    table = bool(rng.random() < 0.6) or not epinat
    image = bool(rng.random() < 0.35)
    kw = dict(nx=nx, ny=ny, nv=nv, u=u, dv=dv, rc_model=wl.RC_EPINAT if epinat else int(rng.integers(0, 2)),
              lsf_sigma=float(rng.choice([0.0, 0.7, 1.5])) * dv)
    if image:
        n = int(rng.choice([3, 5, 9, 13]))
        img = rng.random((n, n)).astype(np.float32) + 0.05
        w = wl.config(4).scaled(psf_n=n, sigma0=float(rng.uniform(0.6, 2.5)) * dv, r0_lo=4.0, r0_hi=9.0,
                                mask_rule="m0_rel", **kw)
        psf = img.astype(np.float64) / img.astype(np.float64).sum()
    else:
        fw = float(rng.choice([0.0, 0.9, 1.8, 2.7]))
        w = wl.config(1).scaled(psf_fwhm=fw, sigma0=float(rng.uniform(0.6, 2.5)) * dv, **kw)
        psf = oracle.psf_gaussian_image(pu.f32(fw), u)
    tab, tab_dx = None, 0.0
    if table:
        ntab = int(rng.integers(2, 40))
        tab_dx = float(rng.uniform(0.05, 0.8))
        tab = (rng.uniform(0.1, 1.0, ntab) * np.exp(-0.3 * tab_dx * np.arange(ntab))).astype(np.float32)
    lsf = oracle.gaussian_taps(pu.f32(w.lsf_sigma) / pu.f32(w.dv) if w.lsf_sigma > 0 else 0.0)
    g = oracle.Grid(nx=nx, ny=ny, nv=nv, u=u, v_center=0.0, dv=pu.f32(dv), rc_model=w.rc_model, psf=psf, lsf=lsf,
                    tab=None if tab is None else tab.astype(np.float64), tab_dx=pu.f32(tab_dx))
    true = [0.5 * nx + rng.uniform(-1, 1), 0.5 * ny + rng.uniform(-1, 1), rng.uniform(0, 360), rng.uniform(20, 75),
            rng.uniform(-40, 40), rng.uniform(60, 280), rng.uniform(1, 6), w.sigma0, rng.uniform(3, 8),
            rng.uniform(0.5, 3)]
    if epinat:
        true += [rng.uniform(0.5, 2.5), rng.uniform(0.5, 2.5)]
    true = np.asarray(true, dtype=np.float32)
    m0, m1, m2 = oracle.model_maps(g, true.astype(np.float64))
    obs = wl.observe(w, m0[None], m1[None], m2[None], rng)
    K = int(rng.choice([1, 4, 9]))
    rows = np.repeat(true[None].astype(np.float64), K, axis=0)
    width = np.array([0.2 * nx, 0.2 * ny, 360.0, 60.0, 100.0, 250.0, 7.0, 0.0, 0.0, 0.0] + ([2.0, 2.0] if epinat else []))
    rows[1:] += 0.1 * width * rng.uniform(-1, 1, (K - 1, rows.shape[1]))
    rows[:, wl.IX_INC] = np.clip(rows[:, wl.IX_INC], 5.0, 85.0)
    rows[:, wl.IX_RT] = np.clip(rows[:, wl.IX_RT], 0.5, None)
    if epinat:
        rows[:, 10:] = np.clip(rows[:, 10:], 0.3, 3.0)
    rows = rows.astype(np.float32)
    ref = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], obs.sobs[0], obs.serr[0], obs.mask[0], rows, want_maps=True)
    d = pu.gbk_desc(w, obs)
    if image:
        d["psf_image"] = img
    if table:
        d["intensity_table"], d["intensity_dx"] = tab, tab_dx
    if rng.random() < 0.5:
        d["tile_w"], d["tile_h"] = int(rng.integers(1, nx + 1)), int(rng.integers(1, ny + 1))
    label = f"model fuzz {seed}: {kw} epinat={epinat} table={table} image={image}"
    pu.compare(ref, _eval(torch_cuda, gbk, d, rows), rows, True, label)
    if seed % 4 == 0:
        pu.compare(ref, _eval(torch_cuda, gbk, d, rows, unfused=True), rows, True, label + " unfused")
