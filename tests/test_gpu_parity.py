"""Parity of the CUDA path (through the C ABI) with the CPU oracle, element by element, on the
same seeded inputs.  Tolerances are BASELINE.json's: m0 1e-4 relative, m1/m2 0.05 km/s absolute,
chi^2 1e-4 relative (see parity_util.compare).  All tests here need a GPU.
"""
import math

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


def _gpu_eval(torch, gbk, desc, rows, gal_index=None, want_maps=True, want_resid=False,
              unfused=False):
    with gbk.Problem(**desc) as prob:
        p = torch.from_numpy(np.ascontiguousarray(rows, dtype=np.float32)).cuda()
        gi = None if gal_index is None else torch.from_numpy(
            np.ascontiguousarray(gal_index, dtype=np.int32)).cuda()
        out = prob.eval(p, gi, want_maps=want_maps, want_resid=want_resid, unfused=unfused)
        torch.cuda.synchronize()
        res = {k: v.cpu().numpy() for k, v in out.items()}
        res["info"] = prob.info
    return res


def _rows_near(w, true_row, rng, n):
    """n trial rows scattered around the true row (10 % of the box width), plus the true row."""
    b = wl.box(w)
    width = b[:, 1] - b[:, 0]
    rows = np.repeat(np.asarray(true_row, dtype=np.float64).reshape(1, -1), n, axis=0)
    rows[1:] += 0.1 * width * rng.uniform(-1, 1, (n - 1, wl.P))
    rows[:, wl.IX_INC] = np.clip(rows[:, wl.IX_INC], 5.0, 85.0)
    rows[:, wl.IX_RT] = np.clip(rows[:, wl.IX_RT], 0.5, None)
    return rows.astype(np.float32)


# ------------------------------------------------------------------------- config 1 ----

@pytest.mark.parametrize("tile", [(0, 0), (16, 16), (12, 10), (8, 32)])
def test_cfg1_maps_and_chi2(oracle, torch_cuda, gbk, tile):
    w = wl.config(1)
    rng = wl.rng_for(1)
    true = wl.cfg1_true_row(rng)
    g, obs = pu.single_galaxy_case(oracle, w, true[0], rng)
    rows = np.concatenate([wl.cfg1_trial_row(), true, _rows_near(w, true[0], rng, 6)])
    ref = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], obs.sobs[0], obs.serr[0], obs.mask[0], rows,
                           want_maps=True, want_resid=True)
    got = _gpu_eval(torch_cuda, gbk, pu.gbk_desc(w, obs, tile_w=tile[0], tile_h=tile[1]), rows,
                    want_resid=True)
    worst = pu.compare(ref, got, rows, want_maps=True, label=f"cfg1 tile={tile}")
    m = obs.mask[0] != 0
    dres = np.abs(got["resid"] - ref["resid"])[:, :, m]
    assert dres.max() <= pu.TOL_M12_ABS / 5.0 + 1e-6          # residual = map difference / 5 km/s
    assert np.all(got["resid"][:, :, ~m] == 0)
    if tile != (0, 0):
        assert got["info"].tiles_x * got["info"].tiles_y > 1
    print("cfg1", tile, worst)


# ------------------------------------------------- config 2 (u = 2), reduced and sampled ----

def test_cfg2_reduced_supersampled(oracle, torch_cuda, gbk):
    w = wl.config(2).scaled(nx=22, ny=18, nv=48)
    rng = wl.rng_for(2)
    true = wl.draw_rows(w, rng, 1)[0]
    g, obs = pu.single_galaxy_case(oracle, w, true, rng)
    rows = wl.lm_rows(w, true)
    ref = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], obs.sobs[0], obs.serr[0], obs.mask[0], rows,
                           want_maps=True)
    for tile in [(0, 0), (8, 6)]:
        got = _gpu_eval(torch_cuda, gbk, pu.gbk_desc(w, obs, tile_w=tile[0], tile_h=tile[1]), rows)
        print("cfg2-reduced", tile, pu.compare(ref, got, rows, True, f"cfg2r tile={tile}"))


def test_cfg2_full_size_sampled_rows(oracle, torch_cuda, gbk):
    w = wl.config(2)
    rng = wl.rng_for(2, 1)
    true = wl.draw_rows(w, rng, 1)[0]
    g, obs = pu.single_galaxy_case(oracle, w, true, rng)
    rows = wl.lm_rows(w, true)                       # K = 8, the launch shape of the LM driver
    got = _gpu_eval(torch_cuda, gbk, pu.gbk_desc(w, obs), rows)
    pick = [0, 3, 7]
    ref = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], obs.sobs[0], obs.serr[0], obs.mask[0],
                           rows[pick], want_maps=True)
    sub = {k: v[pick] for k, v in got.items() if k != "info"}
    print("cfg2-full", pu.compare(ref, sub, rows[pick], True, "cfg2 full"))


# ----------------------------------------------------- config 3: the headline launch ----

def test_cfg3_full_launch_sampled_rows(oracle, torch_cuda, gbk):
    w = wl.config(3)
    rng = wl.rng_for(3)
    true = wl.draw_rows(w, rng, 1)[0]
    true[[wl.IX_XO, wl.IX_YO, wl.IX_VSYS]] = (31.7, 32.4, 0.0)
    g, obs = pu.single_galaxy_case(oracle, w, true, rng)
    rows = wl.nested_grid_rows(w, true, level=0)      # K = 4096, chi^2 only (bench configuration)
    assert rows.shape == (4096, wl.P)
    got = _gpu_eval(torch_cuda, gbk, pu.gbk_desc(w, obs), rows, want_maps=False)
    pick = rng.choice(4096, size=48, replace=False)
    ref = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], obs.sobs[0], obs.serr[0], obs.mask[0],
                           rows[pick])
    sub = {"chi2": got["chi2"][pick]}
    print("cfg3", pu.compare(ref, sub, rows[pick], False, "cfg3"))
    # the grid minimum found on the GPU is the oracle's minimum among the sampled rows
    assert pick[np.argmin(ref["chi2"])] == pick[np.argmin(sub["chi2"])]
    # maps for a few rows as well
    got_m = _gpu_eval(torch_cuda, gbk, pu.gbk_desc(w, obs), rows[pick[:6]])
    ref_m = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], obs.sobs[0], obs.serr[0], obs.mask[0],
                             rows[pick[:6]], want_maps=True)
    print("cfg3 maps", pu.compare(ref_m, got_m, rows[pick[:6]], True, "cfg3 maps"))


# ------------------------------------------------------- config 4: image PSF, ramp ----

def test_cfg4_reduced_moffat_ramp(oracle, torch_cuda, gbk):
    w = wl.config(4).scaled(nx=44, ny=36)
    rng = wl.rng_for(4)
    true = wl.draw_rows(w, rng, 1)[0]
    g, obs = pu.single_galaxy_case(oracle, w, true, rng)
    assert 0.25 < 1.0 - obs.mask.mean() < 0.35        # ~30 % masked
    rows = np.concatenate([true[None], wl.draw_rows(w, rng, 11)])
    ref = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], obs.sobs[0], obs.serr[0], obs.mask[0], rows,
                           want_maps=True)
    for tile in [(0, 0), (16, 12)]:
        got = _gpu_eval(torch_cuda, gbk, pu.gbk_desc(w, obs, tile_w=tile[0], tile_h=tile[1]), rows)
        print("cfg4-reduced", tile, pu.compare(ref, got, rows, True, f"cfg4r tile={tile}"))


def test_cfg4_full_size_sampled_rows(oracle, torch_cuda, gbk):
    w = wl.config(4)
    rng = wl.rng_for(4, 1)
    true = wl.draw_rows(w, rng, 1)[0]
    true[wl.IX_R0] = 30.0
    g, obs = pu.single_galaxy_case(oracle, w, true, rng)
    rows = wl.draw_rows(w, rng, w.K)
    rows[0] = true
    got = _gpu_eval(torch_cuda, gbk, pu.gbk_desc(w, obs), rows, want_maps=True)
    pick = [0, 17, 101]
    ref = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], obs.sobs[0], obs.serr[0], obs.mask[0],
                           rows[pick], want_maps=True)
    sub = {k: v[pick] for k, v in got.items() if k != "info"}
    print("cfg4-full", pu.compare(ref, sub, rows[pick], True, "cfg4 full"))


# ------------------------------------------------ config 5: mixed-galaxy batches ----

def test_cfg5_mixed_galaxies(oracle, torch_cuda, gbk):
    n_gal = 6
    w = wl.config(5).scaled(n_gal=n_gal)
    rng = wl.rng_for(5)
    fwhms = wl.galaxy_fwhms(w, rng)
    trues = wl.draw_rows(w, rng, n_gal)
    grids, clean = [], []
    for gi in range(n_gal):
        g = pu.oracle_grid(oracle, w, fwhms[gi])
        grids.append(g)
        clean.append(oracle.model_maps(g, trues[gi].astype(np.float64)))
    m0, m1, m2 = (np.stack([c[i] for c in clean]) for i in range(3))
    obs = wl.observe(w, m0, m1, m2, rng)
    rows, gal = [], []
    for gi in range(n_gal):                          # LM-shaped slots: base + 7 forward differences
        rows.append(wl.lm_rows(w, trues[gi]))
        gal += [gi] * 8
    rows = np.concatenate(rows)
    gal = np.asarray(gal, dtype=np.int32)
    perm = rng.permutation(len(gal))                  # mixed order
    rows, gal = rows[perm], gal[perm]
    got = _gpu_eval(torch_cuda, gbk, pu.gbk_desc(w, obs, fwhms=fwhms), rows, gal_index=gal)
    assert got["info"].r_p_max == max(int(math.ceil(4 * oracle.fwhm_to_sigma(pu.f32(f)))) for f in fwhms)
    for gi in range(n_gal):
        sel = np.nonzero(gal == gi)[0]
        ref = oracle.eval_rows(grids[gi], obs.vobs[gi], obs.verr[gi], obs.sobs[gi], obs.serr[gi],
                               obs.mask[gi], rows[sel], want_maps=True)
        sub = {k: v[sel] for k, v in got.items() if k != "info"}
        print("cfg5 gal", gi, float(fwhms[gi]), pu.compare(ref, sub, rows[sel], True, f"cfg5 gal {gi}"))


def test_cfg5_full_launch_sampled_rows(oracle, torch_cuda, gbk):
    """Config 5 at the size bench.py's survey leg launches: 1000 data sets with their own PSF, one
    mixed batch of K = 16384 rows.  The observation is seeded random data (chi^2 parity needs no
    realistic maps, and clean maps of 1000 galaxies would take the oracle minutes); 24 sampled rows
    are checked against the oracle with the sampled row's own PSF and data set."""
    torch = torch_cuda
    w = wl.config(5)
    rng = wl.rng_for(5, 9)
    n = w.n_gal
    fwhms = wl.galaxy_fwhms(w, rng)
    shp = (n, w.ny, w.nx)
    obs = wl.Observed(rng.normal(0.0, 80.0, shp).astype(np.float32),
                      rng.uniform(3.0, 15.0, shp).astype(np.float32),
                      rng.uniform(20.0, 80.0, shp).astype(np.float32),
                      rng.uniform(3.0, 15.0, shp).astype(np.float32),
                      (rng.random(shp) < 0.8).astype(np.uint8))
    K = w.K
    rows = wl.draw_rows(w, rng, K)
    gal = rng.integers(0, n, K).astype(np.int32)
    with gbk.Problem(**pu.gbk_desc(w, obs, fwhms=fwhms)) as prob:
        assert prob.info.n_gal == n
        out = prob.eval(torch.from_numpy(rows).cuda(), torch.from_numpy(gal).cuda())
        chi = out["chi2"].cpu().numpy()
    assert np.isfinite(chi).all()
    sel = np.concatenate([[0, K - 1], rng.integers(0, K, 22)])
    for k in sel:
        gi = int(gal[k])
        g = pu.oracle_grid(oracle, w, fwhms[gi])
        ref = oracle.eval_rows(g, obs.vobs[gi], obs.verr[gi], obs.sobs[gi], obs.serr[gi], obs.mask[gi],
                               rows[k:k + 1])
        pu.compare(ref, {"chi2": chi[k:k + 1]}, rows[k:k + 1], False, f"cfg5 full row {k} gal {gi}")


# ------------------------------------------------------------------- edge cases ----

def _tiny_case(oracle, **kw):
    w = wl.config(1).scaled(**{**dict(nx=14, ny=11, nv=40), **kw})
    rng = np.random.default_rng(11)
    true = np.array([6.2, 5.1, 140.0, 50.0, 8.0, 180.0, 2.0, 40.0, 3.0, 1.5], dtype=np.float32)
    g, obs = pu.single_galaxy_case(oracle, w, true, rng)
    return w, g, obs, true, rng


def test_out_of_domain_rows_and_empty_batch(oracle, torch_cuda, gbk):
    w, g, obs, true, rng = _tiny_case(oracle)
    rows = np.repeat(true[None], 8, axis=0)
    rows[1, wl.IX_SIG] = 0.0
    rows[2, wl.IX_R0] = -1.0
    rows[3, wl.IX_RT] = 0.0
    rows[4, wl.IX_INC] = 90.0
    rows[5, wl.IX_VT] = np.nan
    rows[6, wl.IX_I0] = 0.0
    rows[7, wl.IX_XO] = np.inf
    ref = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], obs.sobs[0], obs.serr[0], obs.mask[0], rows,
                           want_maps=True)
    for tile in [(0, 0), (5, 4)]:
        got = _gpu_eval(torch_cuda, gbk, pu.gbk_desc(w, obs, tile_w=tile[0], tile_h=tile[1]), rows,
                        want_resid=True)
        assert np.isfinite(got["chi2"][0]) and np.all(np.isposinf(got["chi2"][1:]))
        assert np.all(np.isposinf(ref["chi2"][1:]))
        assert np.isnan(got["m1"][1:]).all() and np.isnan(got["resid"][1:]).all()
        pu.compare(ref, got, rows, True, "domain")
    # K = 0 is a no-op
    with gbk.Problem(**pu.gbk_desc(w, obs)) as prob:
        p = torch_cuda.empty((0, 10), dtype=torch_cuda.float32, device="cuda")
        assert prob.eval(p)["chi2"].numel() == 0
    # a gal_index outside [0, n_gal) makes the row +INF instead of reading out of bounds
    got = _gpu_eval(torch_cuda, gbk, pu.gbk_desc(w, obs), rows[:2],
                    gal_index=np.array([0, 3], dtype=np.int32), want_maps=False)
    assert np.isfinite(got["chi2"][0]) and np.isposinf(got["chi2"][1])


def test_model_dark_unmasked_spaxel_gives_inf(oracle, torch_cuda, gbk):
    w, g, obs, true, rng = _tiny_case(oracle)
    rows = np.repeat(true[None], 2, axis=0)
    rows[1, wl.IX_R0] = 0.02         # exp(-r/r0) falls below 1e-30 inside the field
    obs.mask[:] = 1                   # nothing masked: dark spaxels count
    obs.verr[:] = 5.0
    ref = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], obs.sobs[0], obs.serr[0], obs.mask[0], rows)
    got = _gpu_eval(torch_cuda, gbk, pu.gbk_desc(w, obs), rows, want_maps=False)
    assert np.isposinf(ref["chi2"][1]) and np.isposinf(got["chi2"][1])
    assert np.isfinite(got["chi2"][0])


def test_masks_and_missing_dispersion_term(oracle, torch_cuda, gbk):
    w, g, obs, true, rng = _tiny_case(oracle)
    rows = _rows_near(w, true, rng, 4)
    # all masked: chi^2 = 0
    all_masked = wl.Observed(obs.vobs, obs.verr, obs.sobs, obs.serr, np.zeros_like(obs.mask))
    got = _gpu_eval(torch_cuda, gbk, pu.gbk_desc(w, all_masked), rows, want_maps=False)
    assert np.all(got["chi2"] == 0.0)
    # no dispersion map: second term of eq. 11 dropped
    d = pu.gbk_desc(w, obs)
    d["sobs"] = d["serr"] = None
    got = _gpu_eval(torch_cuda, gbk, d, rows, want_maps=False)
    ref = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], None, None, obs.mask[0], rows)
    pu.compare(ref, got, rows, False, "no dispersion")
    # mask = None: every spaxel counts
    d = pu.gbk_desc(w, obs)
    d["mask"] = None
    full = wl.Observed(obs.vobs, obs.verr, obs.sobs, obs.serr, np.ones_like(obs.mask))
    got = _gpu_eval(torch_cuda, gbk, d, rows, want_maps=False)
    ref = oracle.eval_rows(g, full.vobs[0], full.verr[0], full.sobs[0], full.serr[0], None, rows)
    pu.compare(ref, got, rows, False, "no mask")


@pytest.mark.parametrize("kw", [dict(psf_fwhm=0.0, lsf_sigma=0.0), dict(psf_fwhm=0.7),
                                dict(u=3, psf_fwhm=1.2), dict(u=4, nx=6, ny=5, psf_fwhm=1.6),
                                dict(v_center=1500.0), dict(rc_model=wl.RC_RAMP),
                                dict(psf_fwhm=6.7, nx=9, ny=7)])
def test_variants(oracle, torch_cuda, gbk, kw):
    w, g, obs, true, rng = _tiny_case(oracle, **kw)
    if "v_center" in kw:
        true = true.copy()
        true[wl.IX_VSYS] += kw["v_center"]
        g, obs = pu.single_galaxy_case(oracle, w, true, rng)
    rows = _rows_near(w, true, rng, 5)
    ref = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], obs.sobs[0], obs.serr[0], obs.mask[0], rows,
                           want_maps=True)
    got = _gpu_eval(torch_cuda, gbk, pu.gbk_desc(w, obs), rows)
    print("variant", kw, pu.compare(ref, got, rows, True, f"variant {kw}"))


@pytest.mark.parametrize("kw,tile", [
    (dict(psf_fwhm=0.0, lsf_sigma=0.0), (4, 4)), (dict(psf_fwhm=0.0, lsf_sigma=0.0), (2, 2)),
    (dict(psf_fwhm=0.0, lsf_sigma=0.0), (1, 1)), (dict(psf_fwhm=0.0), (3, 11)),
    (dict(psf_fwhm=1.1), (1, 2)), (dict(psf_fwhm=1.1), (2, 1)), (dict(psf_fwhm=1.1, u=2), (1, 1)),
    (dict(psf_fwhm=0.0, lsf_sigma=0.0), (0, 0))])
def test_tiny_tiles_and_delta_kernels(oracle, torch_cuda, gbk, kw, tile):
    """Tiles of one or two pixels and the delta PSF (tap radius 0): the degenerate sizes of the index
    arithmetic (a divisor of 1 in the multiply-high division once produced +INF rows).  K = 5 with
    automatic tiling (0, 0) also takes the small-batch tiling chosen at eval time."""
    w, g, obs, true, rng = _tiny_case(oracle, **kw)
    rows = _rows_near(w, true, rng, 5)
    ref = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], obs.sobs[0], obs.serr[0], obs.mask[0], rows,
                           want_maps=True)
    got = _gpu_eval(torch_cuda, gbk, pu.gbk_desc(w, obs, tile_w=tile[0], tile_h=tile[1]), rows)
    pu.compare(ref, got, rows, True, f"tiny tiles {kw} {tile}")


def test_batch_size_picks_the_tiling_but_not_the_result(oracle, torch_cuda, gbk):
    """Automatic tiling takes smaller tiles for batches too small to fill the GPU: the same row
    must agree with the oracle (and with itself to rounding) at K = 1, 8 and 600."""
    torch = torch_cuda
    w, g, obs, true, rng = _tiny_case(oracle, nx=40, ny=36)
    rows = _rows_near(w, true, rng, 600)
    ref = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], obs.sobs[0], obs.serr[0], obs.mask[0], rows[:8],
                           want_maps=True)
    with gbk.Problem(**pu.gbk_desc(w, obs)) as prob:
        p = torch.from_numpy(rows).cuda()
        outs = {}
        for K in (1, 8, 600):
            out = prob.eval(p[:K].contiguous(), want_maps=True)
            torch.cuda.synchronize()
            outs[K] = {k: v.cpu().numpy() for k, v in out.items()}
    pu.compare({k: v[:1] for k, v in ref.items()}, outs[1], rows[:1], True, "K=1")
    pu.compare(ref, outs[8], rows[:8], True, "K=8")
    pu.compare(ref, {k: v[:8] for k, v in outs[600].items()}, rows[:8], True, "K=600")
    np.testing.assert_allclose(outs[1]["chi2"], outs[600]["chi2"][:1], rtol=2e-6)


@pytest.mark.parametrize("rc_model", [wl.RC_ARCTAN, wl.RC_RAMP])
def test_line_width_sweep_covers_recurrence_and_direct_loops(oracle, torch_cuda, gbk, rc_model):
    """The voxel loop evaluates the line by a multiplicative recurrence when sigma_0/dv >= 1.06 and by
    one ex2 per voxel below that: one batch mixes both, on either side of the
    switch, with lines that leave the band (large V_sys offsets), very fast and very slow discs."""
    w, g, obs, true, rng = _tiny_case(oracle, nx=20, ny=17, nv=56, rc_model=rc_model)
    dv = w.dv
    rows = []
    for ratio in (0.45, 0.8, 1.0, 1.05, 1.0617, 1.07, 1.2, 2.0, 5.0):
        for dvsys, vt in ((0.0, 180.0), (400.0, 250.0), (-700.0, 60.0), (0.0, 1500.0)):
            r = true.copy()
            r[wl.IX_SIG] = ratio * dv
            r[wl.IX_VSYS] += dvsys
            r[wl.IX_VT] = vt
            rows.append(r)
    r = true.copy()
    r[wl.IX_VSYS] = 5000.0            # the whole line outside the band: model-dark everywhere
    rows.append(r)
    rows = np.stack(rows).astype(np.float32)
    ref = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], obs.sobs[0], obs.serr[0], obs.mask[0], rows,
                           want_maps=True)
    for tile in ((0, 0), (7, 6)):
        got = _gpu_eval(torch_cuda, gbk, pu.gbk_desc(w, obs, tile_w=tile[0], tile_h=tile[1]), rows)
        worst = pu.compare(ref, got, rows, True, f"line width sweep rc={rc_model} tile={tile}")
        assert worst["skipped_rows"] <= 4, worst
    assert np.isinf(ref["chi2"][-1])


@pytest.mark.parametrize("rc_model", [wl.RC_ARCTAN, wl.RC_RAMP])
@pytest.mark.parametrize("nv,dv", [(20, 10.0), (12, 30.0), (40, 5.0)])
def test_far_wing_lines_centred_outside_a_short_band(oracle, torch_cuda, gbk, rc_model, nv, dv):
    """Short bands with the line centred up to ~11 sigma_0 OUTSIDE them: every spaxel then sees only the
    far wing of its line (m0 down to 1e-28 I_0), where a voxel is 2^-(d^2) at |d| ~ 9 and an error of
    the line offset d is amplified 12-fold.  Those rows take the FP64 geometry (RowConst::precise); m0
    must still hold 1e-4 relative at every spaxel brighter than the model-dark guard.  Fast discs with
    narrow lines (|V_t sin i| / sigma_0 up to ~70) are the worst case for the FP32 offset."""
    w, g, obs, true, rng = _tiny_case(oracle, nx=18, ny=15, nv=nv, dv=dv, rc_model=rc_model,
                                      lsf_sigma=0.6 * dv, psf_fwhm=1.7)
    half = 0.5 * nv * dv
    rows = []
    for ratio in (0.45, 0.9, 1.1, 1.6, 3.0):                 # sigma_0 / dv: direct loop and block polynomial
        sig = ratio * dv
        for edge in (-1.0, 1.0):                             # below and above the band
            for nsig in (0.0, 2.0, 4.0, 6.0, 8.0, 9.5, 11.0):   # line centre this many sigma_0 outside
                for vt in (60.0, 300.0):
                    r = true.copy()
                    r[wl.IX_SIG] = sig
                    r[wl.IX_VSYS] = edge * (half + nsig * sig)
                    r[wl.IX_VT] = vt
                    rows.append(r)
    rows = np.stack(rows).astype(np.float32)
    ref = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], obs.sobs[0], obs.serr[0], obs.mask[0], rows,
                           want_maps=True)
    n_bright_faint = 0
    for k in range(len(rows)):                               # the case must really contain far-wing spaxels
        m = ref["m0"][k]
        n_bright_faint += int(((m > 1e-27 * rows[k, wl.IX_I0]) & (m < 1e-12 * rows[k, wl.IX_I0])).sum())
    assert n_bright_faint > 1000
    for tile in ((0, 0), (7, 5)):
        got = _gpu_eval(torch_cuda, gbk, pu.gbk_desc(w, obs, tile_w=tile[0], tile_h=tile[1]), rows)
        worst = pu.compare(ref, got, rows, True, f"far wing rc={rc_model} nv={nv} dv={dv} tile={tile}")
        print("far wing", rc_model, nv, dv, tile, worst)


def test_bitwise_reproducible_and_host_entry(oracle, torch_cuda, gbk):
    torch = torch_cuda
    w, g, obs, true, rng = _tiny_case(oracle)
    rows = _rows_near(w, true, rng, 64)
    with gbk.Problem(**pu.gbk_desc(w, obs, tile_w=5, tile_h=4)) as prob:
        p = torch.from_numpy(rows).cuda()
        a = prob.eval(p)["chi2"].cpu().numpy()
        b = prob.eval(p)["chi2"].cpu().numpy()
        assert np.array_equal(a, b)                      # fixed-order reductions, no float atomics
        host_params = torch.from_numpy(rows).pin_memory()
        host_chi2 = torch.empty(64, dtype=torch.float32).pin_memory()
        gbk.gbk_eval_batch_host(prob.handle, host_params, None, 64, host_chi2,
                                torch.cuda.current_stream().cuda_stream)
        assert np.array_equal(host_chi2.numpy(), a)
        pageable = np.empty(64, dtype=np.float32)
        gbk.gbk_eval_batch_host(prob.handle, rows, None, 64, pageable)
        assert np.array_equal(pageable, a)


def test_create_rejects_bad_descriptors(oracle, torch_cuda, gbk):
    w, g, obs, true, rng = _tiny_case(oracle)
    d = pu.gbk_desc(w, obs)
    bad = dict(d)
    bad["dv"] = 0.0
    with pytest.raises(gbk.GbkError) as e:
        gbk.Problem(**bad)
    assert e.value.code == gbk.GBK_ERR_ARG
    bad = dict(d)
    v = obs.vobs.copy()
    v[0][obs.mask[0] != 0] = np.nan
    bad["vobs"] = v
    with pytest.raises(gbk.GbkError):
        gbk.Problem(**bad)
    bad = dict(d)
    bad["psf_kind"], bad["psf_image"] = gbk.GBK_PSF_IMAGE, np.ones((4, 4), dtype=np.float32)
    with pytest.raises(gbk.GbkError):
        gbk.Problem(**bad)
    bad = dict(d)
    bad["psf_fwhm"] = np.array([40.0], dtype=np.float32)          # radius beyond the supported maximum
    with pytest.raises(gbk.GbkError) as e:
        gbk.Problem(**bad)
    assert e.value.code == gbk.GBK_ERR_UNSUPPORTED


def test_eval_batch_in_a_cuda_graph(oracle, torch_cuda, gbk):
    """gbk_eval_batch is asynchronous on the caller's stream and allocates nothing once its scratch
    is sized, so it can be captured in a CUDA graph and replayed on new parameters (bench-style
    inner loops, optimiser iterations)."""
    torch = torch_cuda
    w, g, obs, true, rng = _tiny_case(oracle, nx=40, ny=36)
    rows_a = _rows_near(w, true, rng, 300)
    rows_b = _rows_near(w, true, rng, 300)
    with gbk.Problem(**pu.gbk_desc(w, obs, tile_w=16, tile_h=12)) as prob:   # tiled: two kernels
        params = torch.from_numpy(rows_a).cuda()
        chi2 = torch.empty(300, dtype=torch.float32, device="cuda")
        side = torch.cuda.Stream()
        with torch.cuda.stream(side):
            gbk.gbk_eval_batch(prob.handle, params, None, 300, chi2, stream=side.cuda_stream)  # sizes scratch
        side.synchronize()
        eager = chi2.cpu().numpy().copy()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            gbk.gbk_eval_batch(prob.handle, params, None, 300, chi2, stream=side.cuda_stream)
        chi2.zero_()
        graph.replay()
        torch.cuda.synchronize()
        assert np.array_equal(chi2.cpu().numpy(), eager)
        params.copy_(torch.from_numpy(rows_b))
        graph.replay()
        torch.cuda.synchronize()
        got_b = chi2.cpu().numpy()
    ref = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], obs.sobs[0], obs.serr[0], obs.mask[0], rows_b[:16])
    pu.compare(ref, {"chi2": got_b[:16]}, rows_b[:16], False, "graph replay")


def test_two_streams_overlap_on_one_problem_and_capture_needs_reserve(oracle, torch_cuda, gbk):
    """Multi-tile launches of ONE problem on two streams at the same time: each stream has its own
    cross-tile scratch, so the results are those of sequential launches (bit for bit).  Growing the
    scratch during a stream capture is refused with GBK_ERR_ARG; after gbk_reserve the capture works."""
    torch = torch_cuda
    w, g, obs, true, rng = _tiny_case(oracle, nx=40, ny=36)
    Ka, Kb = 700, 900
    rows_a, rows_b = _rows_near(w, true, rng, Ka), _rows_near(w, true, rng, Kb)
    with gbk.Problem(**pu.gbk_desc(w, obs, tile_w=8, tile_h=6)) as prob:        # 35 tiles per row
        pa, pb = torch.from_numpy(rows_a).cuda(), torch.from_numpy(rows_b).cuda()
        seq_a = prob.eval(pa)["chi2"].cpu().numpy()
        seq_b = prob.eval(pb)["chi2"].cpu().numpy()
        s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
        ca = torch.empty(Ka, dtype=torch.float32, device="cuda")
        cb = torch.empty(Kb, dtype=torch.float32, device="cuda")
        torch.cuda.synchronize()
        for rep in range(6):                          # several rounds in flight on both streams
            gbk.gbk_eval_batch(prob.handle, pa, None, Ka, ca, stream=s1.cuda_stream)
            gbk.gbk_eval_batch(prob.handle, pb, None, Kb, cb, stream=s2.cuda_stream)
        torch.cuda.synchronize()
        assert np.array_equal(ca.cpu().numpy(), seq_a) and np.array_equal(cb.cpu().numpy(), seq_b)
        # capture on a fresh stream whose scratch has never been sized
        s3 = torch.cuda.Stream()
        graph = torch.cuda.CUDAGraph()
        with pytest.raises(gbk.GbkError) as e:
            with torch.cuda.graph(graph, stream=s3):
                gbk.gbk_eval_batch(prob.handle, pa, None, Ka, ca, stream=s3.cuda_stream)
        assert e.value.code == gbk.GBK_ERR_ARG and "gbk_reserve" in str(e.value)
        torch.cuda.synchronize()
        s4 = torch.cuda.Stream()
        gbk.gbk_reserve(prob.handle, Ka, s4.cuda_stream)
        s4.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=s4):
            gbk.gbk_eval_batch(prob.handle, pa, None, Ka, ca, stream=s4.cuda_stream)
        ca.zero_()
        graph.replay()
        torch.cuda.synchronize()
        assert np.array_equal(ca.cpu().numpy(), seq_a)
    ref = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], obs.sobs[0], obs.serr[0], obs.mask[0], rows_a[:8])
    pu.compare(ref, {"chi2": seq_a[:8]}, rows_a[:8], False, "two streams")


# seeds 431 and 589: lines centred outside a short band (far-wing spaxels, m0 ~ 1e-15 I) once lost their
# relative accuracy to the clamped block polynomial; seed 2313: a spaxel that sees only the far wing
# (m0 ~ 1e-24 I) was 1.36e-4 off in m0 while the line offset was carried in FP32
@pytest.mark.parametrize("seed", sorted(set(range(int(__import__("os").environ.get("GBK_FUZZ_CASES", "300"))))
                                        | {431, 589, 2313}))
def test_random_shapes_and_kernels(oracle, torch_cuda, gbk, seed):
    """Seeded random problems: odd grid sizes, any up-sampling, Gaussian or image PSFs of any small
    size (symmetric or not), delta or wide LSFs, explicit or automatic tiles, both rotation curves,
    with and without a dispersion map -- chi^2 and maps against the oracle."""
    rng = np.random.default_rng(1510_01815 + seed)
    nx, ny = int(rng.integers(3, 34)), int(rng.integers(3, 30))
    u = int(rng.choice([1, 1, 1, 2, 3]))
    nv = int(rng.integers(12, 70))
    dv = float(rng.choice([10.0, 20.0, 30.0]))
    image = bool(rng.random() < 0.4)
    kw = dict(nx=nx, ny=ny, nv=nv, u=u, dv=dv, rc_model=int(rng.integers(0, 2)),
              lsf_sigma=float(rng.choice([0.0, 0.6, 1.0, 2.3])) * dv)
    if image:
        n = int(rng.choice([1, 3, 5, 7, 9, 11, 15, 17]))
        img = rng.random((n, n)).astype(np.float32) + 0.05          # asymmetric: convolution, not correlation
        w = wl.config(4).scaled(psf_n=n, sigma0=float(rng.uniform(0.5, 3.0)) * dv, r0_lo=4.0, r0_hi=9.0,
                                mask_rule="m0_rel", **kw)
        psf = img.astype(np.float64) / img.astype(np.float64).sum()
    else:
        fw = float(rng.choice([0.0, 0.8, 1.7, 2.6, 3.9]))
        if np.ceil(4.0 * u * fw / 2.3548) > 16:          # the library's separable limit: R <= 16 fine pixels
            fw = 1.7
        w = wl.config(1).scaled(psf_fwhm=fw, sigma0=float(rng.uniform(0.5, 3.0)) * dv, **kw)
        psf = oracle.psf_gaussian_image(pu.f32(fw), u)
    lsf = oracle.gaussian_taps(pu.f32(w.lsf_sigma) / pu.f32(w.dv) if w.lsf_sigma > 0 else 0.0)
    g = oracle.Grid(nx=nx, ny=ny, nv=nv, u=u, v_center=0.0, dv=pu.f32(dv), rc_model=w.rc_model, psf=psf,
                    lsf=lsf)
    true = np.array([0.5 * nx + rng.uniform(-1, 1), 0.5 * ny + rng.uniform(-1, 1), rng.uniform(0, 360),
                     rng.uniform(20, 75), rng.uniform(-40, 40), rng.uniform(60, 280), rng.uniform(1, 6),
                     w.sigma0, rng.uniform(3, 8), rng.uniform(0.5, 3)], dtype=np.float32)
    m0, m1, m2 = oracle.model_maps(g, true.astype(np.float64))
    obs = wl.observe(w, m0[None], m1[None], m2[None], rng)
    K = int(rng.choice([1, 3, 17]))
    rows = _rows_near(w, true, rng, K)
    rows[:, wl.IX_SIG] = w.sigma0 * rng.uniform(0.7, 1.5, K)
    no_disp = bool(rng.random() < 0.25)
    ref = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], None if no_disp else obs.sobs[0],
                           None if no_disp else obs.serr[0], obs.mask[0], rows, want_maps=True)
    d = pu.gbk_desc(w, obs)
    if image:
        d["psf_image"] = img
    if no_disp:
        d["sobs"] = d["serr"] = None
    if rng.random() < 0.5:
        d["tile_w"], d["tile_h"] = int(rng.integers(1, nx + 1)), int(rng.integers(1, ny + 1))
    got = _gpu_eval(torch_cuda, gbk, d, rows)
    worst = pu.compare(ref, got, rows, True,
                       f"random case {seed}: {kw} image={image} tile={d.get('tile_w')},{d.get('tile_h')}")
    log = __import__("os").environ.get("GBK_FUZZ_LOG")      # one JSON line per case (profiles/: wide fuzz runs)
    if log:
        with open(log, "a") as f:
            f.write(__import__("json").dumps({"seed": seed, **worst}) + "\n")


def test_two_problems_with_different_tiles_coexist(oracle, torch_cuda, gbk):
    """The dynamic shared-memory opt-in is a property of the kernel: creating a second problem with
    a smaller tile must not break launches of the first, larger one."""
    torch = torch_cuda
    w_big, g_big, obs_big, true_big, rng = _tiny_case(oracle, nx=64, ny=64, nv=40)     # > 48 KB tile
    w_small, g_small, obs_small, true_small, _ = _tiny_case(oracle)
    rows_big = _rows_near(w_big, true_big, rng, 4)
    rows_small = _rows_near(w_small, true_small, rng, 4)
    with gbk.Problem(**pu.gbk_desc(w_big, obs_big, tile_w=64, tile_h=64)) as big:
        assert big.info.smem_bytes > 48 * 1024
        with gbk.Problem(**pu.gbk_desc(w_small, obs_small)) as small:
            a = small.eval(torch.from_numpy(rows_small).cuda())["chi2"].cpu().numpy()
            b = big.eval(torch.from_numpy(rows_big).cuda())["chi2"].cpu().numpy()      # after the small one
    ref_b = oracle.eval_rows(g_big, obs_big.vobs[0], obs_big.verr[0], obs_big.sobs[0], obs_big.serr[0],
                             obs_big.mask[0], rows_big)
    ref_a = oracle.eval_rows(g_small, obs_small.vobs[0], obs_small.verr[0], obs_small.sobs[0],
                             obs_small.serr[0], obs_small.mask[0], rows_small)
    pu.compare(ref_b, {"chi2": b}, rows_big, False, "big after small")
    pu.compare(ref_a, {"chi2": a}, rows_small, False, "small")


@pytest.mark.parametrize("nv,dv,sig", [(400, 5.0, 40.0), (333, 4.0, 4.5), (16, 120.0, 130.0), (9, 60.0, 20.0)])
def test_many_and_few_channels(oracle, torch_cuda, gbk, nv, dv, sig):
    """Bands of many fine channels (hundreds of blocks of the voxel loop, lines many channels wide),
    of very few coarse ones, and odd channel counts (padding of the last block)."""
    w, g, obs, true, rng = _tiny_case(oracle, nx=12, ny=10, nv=nv, dv=dv, sigma0=sig, lsf_sigma=0.7 * dv)
    true = true.copy()
    true[wl.IX_SIG] = sig
    g, obs = pu.single_galaxy_case(oracle, w, true, rng)
    rows = _rows_near(w, true, rng, 6)
    rows[:, wl.IX_SIG] = sig * np.array([1.0, 0.8, 1.3, 1.0, 2.0, 0.6], dtype=np.float32)
    rows[3, wl.IX_VSYS] += 0.4 * nv * dv          # most of the line outside the band
    ref = oracle.eval_rows(g, obs.vobs[0], obs.verr[0], obs.sobs[0], obs.serr[0], obs.mask[0], rows,
                           want_maps=True)
    got = _gpu_eval(torch_cuda, gbk, pu.gbk_desc(w, obs), rows)
    print("channels", nv, dv, sig, pu.compare(ref, got, rows, True, f"nv={nv} dv={dv} sigma0={sig}"))
