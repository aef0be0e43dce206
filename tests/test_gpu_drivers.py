"""The host drivers (gbk_fit_ng / gbk_fit_lm / gbk_fit_ns) on the GPU.

Several optimiser paths are correct, so what is compared is what is unique: the nested-grid path
is deterministic given the chi^2 values and must equal a replica of rule A19 driven by the same
chi^2 (gbk_eval_batch, itself parity-checked against the oracle elsewhere); LM and NS must recover
the parameters of noise-free synthetic data within the thresholds the paper uses for its own mock
data (Table 3: 1 px, 1 degree, 5 km/s).
"""
import numpy as np
import pytest

from paper_1510_01815_b200 import workloads as wl

import parity_util as pu

pytestmark = pytest.mark.gpu

FREE7 = [wl.IX_XO, wl.IX_YO, wl.IX_PA, wl.IX_INC, wl.IX_VSYS, wl.IX_VT, wl.IX_RT]
FREE4 = [wl.IX_PA, wl.IX_INC, wl.IX_VT, wl.IX_RT]
TABLE3 = {wl.IX_XO: 1.0, wl.IX_YO: 1.0, wl.IX_PA: 1.0, wl.IX_INC: 1.0, wl.IX_VSYS: 5.0, wl.IX_VT: 5.0,
          wl.IX_RT: 1.0}


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


def _case(oracle, cfg, true, **scale):
    w = wl.config(cfg).scaled(noise=0.0, **scale)
    rng = wl.rng_for(cfg, 7)
    g, obs = pu.single_galaxy_case(oracle, w, true, rng)
    return w, obs


def _true_row(w):
    t = np.array([0.5 * w.nx + 0.4, 0.5 * w.ny - 0.3, 123.0, 52.0, 8.0, 180.0, 3.5, w.sigma0,
                  w.r0_lo, 1.0], dtype=np.float32)
    return t


def _pa_diff(a, b):
    return abs((a - b + 180.0) % 360.0 - 180.0)


def test_nested_grids_follow_rule_a19_and_find_the_truth(oracle, torch_cuda, gbk):
    torch = torch_cuda
    w0 = wl.config(3).scaled(nx=32, ny=32, nv=48)
    true = _true_row(w0)
    w, obs = _case(oracle, 3, true, nx=32, ny=32, nv=48)
    b = wl.box(w)
    nodes, levels = 6, 4
    with gbk.Problem(**pu.gbk_desc(w, obs)) as prob:
        best, chi, st = gbk.gbk_fit_ng(prob.handle, true, 0, FREE4, b[FREE4, 0], b[FREE4, 1], nodes,
                                       levels)
        # replica of A19 in numpy, driven by the same chi^2
        centre = None
        for level in range(levels):
            rows = wl.nested_grid_rows(w, true, level=level, centre=centre, nodes=nodes)
            out = prob.eval(torch.from_numpy(rows).cuda())
            k = int(torch.argmin(out["chi2"]).item())
            centre = rows[k, FREE4].astype(np.float64)
            chi_rep = float(out["chi2"][k].item())
    assert st["launches"] == levels and st["evals"] == levels * nodes ** 4 and st["iterations"] == levels
    np.testing.assert_allclose(best[FREE4], centre, rtol=0, atol=1e-3)
    assert chi == pytest.approx(chi_rep, rel=1e-6)
    # the last level's spacing bounds the distance to the truth (noise-free data)
    h = (b[FREE4, 1] - b[FREE4, 0]) / (nodes * 2 ** (levels - 1))
    assert _pa_diff(best[wl.IX_PA], true[wl.IX_PA]) <= 1.5 * h[0]
    for a, j in enumerate(FREE4[1:], start=1):
        assert abs(best[j] - true[j]) <= 1.5 * h[a], (j, best[j], true[j])
    assert np.array_equal(np.delete(best, FREE4), np.delete(true, FREE4))


def test_nested_grids_per_axis_nodes_and_accuracy_thresholds(oracle, torch_cuda, gbk):
    """The paper's configuration: a node count per axis (7 for PA, 11 for r_t and V_t; i
    fixed) and accuracy thresholds (0.01 for r_t, 0.1 otherwise) that end the refinement."""
    w0 = wl.config(3).scaled(nx=32, ny=32, nv=48)
    true = _true_row(w0)
    w, obs = _case(oracle, 3, true, nx=32, ny=32, nv=48)
    b = wl.box(w)
    axes = [wl.IX_PA, wl.IX_RT, wl.IX_VT]
    nodes, acc = [7, 11, 11], [0.1, 0.01, 0.1]
    with gbk.Problem(**pu.gbk_desc(w, obs)) as prob:
        best, chi, st = gbk.gbk_fit_ng(prob.handle, true, 0, axes, b[axes, 0], b[axes, 1], nodes, 30, accuracy=acc)
        capped = gbk.gbk_fit_ng(prob.handle, true, 0, axes, b[axes, 0], b[axes, 1], nodes, 3, accuracy=acc)[2]
    width = b[axes, 1] - b[axes, 0]
    need = max(int(np.ceil(np.log2(width[a] / (nodes[a] * acc[a])))) for a in range(3)) + 1   # first level with h <= a on all axes
    assert st["iterations"] == need and st["evals"] == need * 7 * 11 * 11 and st["converged"] == 1
    assert capped["iterations"] == 3 and capped["converged"] == 0             # max_levels hit first
    assert _pa_diff(best[wl.IX_PA], true[wl.IX_PA]) <= 0.2
    assert abs(best[wl.IX_RT] - true[wl.IX_RT]) <= 0.02 and abs(best[wl.IX_VT] - true[wl.IX_VT]) <= 0.3


def test_levenberg_marquardt_recovers_noise_free_parameters(oracle, torch_cuda, gbk):
    w0 = wl.config(1)
    true = _true_row(w0)
    w, obs = _case(oracle, 1, true)
    b = wl.box(w)
    b[wl.IX_PA] = (true[wl.IX_PA] - 90.0, true[wl.IX_PA] + 90.0)    # PA does not wrap in LM
    rng = wl.rng_for(1, 11)
    starts = np.repeat(true[None], 4, axis=0).astype(np.float64)
    width = b[FREE7, 1] - b[FREE7, 0]
    starts[:, FREE7] += 0.1 * width * rng.uniform(-1, 1, (4, 7))
    starts[3, wl.IX_INC] = 90.0       # cos i = 0: out of domain, chi^2 = +INF at the start
    lo, hi = b[FREE7, 0].copy(), b[FREE7, 1].copy()
    hi[FREE7.index(wl.IX_INC)] = 90.0
    with gbk.Problem(**pu.gbk_desc(w, obs)) as prob:
        rows, chi, iters, st = gbk.gbk_fit_lm(prob.handle, starts, None, FREE7, lo, hi,
                                              rel_step=1e-3, max_iter=50, ftol=1e-6)
    assert np.isinf(chi[3]) and iters[3] == 0
    np.testing.assert_array_equal(rows[3], starts[3].astype(np.float32))
    for f in range(3):
        assert np.isfinite(chi[f]) and chi[f] < 1.0, (f, chi[f])     # noise-free: chi^2 -> 0
        for j in FREE7:
            d = _pa_diff(rows[f, j], true[j]) if j == wl.IX_PA else abs(rows[f, j] - true[j])
            assert d <= TABLE3[j], (f, j, rows[f, j], true[j])
        assert 1 <= iters[f] <= 50
    assert st["converged"] >= 3 and st["launches"] >= 2 and st["evals"] > 0


def test_levenberg_marquardt_mixed_galaxies(oracle, torch_cuda, gbk):
    """Config-5 style: several galaxies, each its own data set and PSF, fitted in one call."""
    w = wl.config(5).scaled(nx=24, ny=24, nv=64, n_gal=3)
    rng = wl.rng_for(5, 3)
    fw = np.array([1.6, 2.4, 3.3], np.float32)
    trues, maps = [], []
    for g in range(3):
        t = _true_row(w)
        t[[wl.IX_PA, wl.IX_INC, wl.IX_VT]] += (40.0 * g, 6.0 * g, -30.0 * g)
        t[wl.IX_R0] = 5.0 + g
        trues.append(t)
        grid = pu.oracle_grid(oracle, w, fwhm=float(fw[g]))
        maps.append(oracle.model_maps(grid, t.astype(np.float64)))
    m0, m1, m2 = (np.stack([m[i] for m in maps]) for i in range(3))
    obs = wl.observe(w, m0, m1, m2, rng)
    trues = np.stack(trues)
    b = wl.box(w)
    starts = trues.astype(np.float64)
    starts[:, FREE7] += 0.05 * (b[FREE7, 1] - b[FREE7, 0]) * rng.uniform(-1, 1, (3, 7))
    lo, hi = b[FREE7, 0].copy(), b[FREE7, 1].copy()
    lo[2], hi[2] = -360.0, 720.0
    with gbk.Problem(**pu.gbk_desc(w, obs, fwhms=fw)) as prob:
        rows, chi, iters, st = gbk.gbk_fit_lm(prob.handle, starts, np.arange(3), FREE7, lo, hi)
        gi = torch_cuda.arange(3, dtype=torch_cuda.int32, device="cuda")
        chi_true = prob.eval(torch_cuda.from_numpy(trues).cuda(), gi)["chi2"].cpu().numpy()
        chi_fit = prob.eval(torch_cuda.from_numpy(rows).cuda(), gi)["chi2"].cpu().numpy()
    # config 5 draws noise N(0, E) with per-spaxel errors: the fit must do at least as well as the
    # truth on the noisy data, report the chi^2 of the row it returns, and stay near the truth
    np.testing.assert_allclose(chi, chi_fit, rtol=1e-6)
    for f in range(3):
        assert chi[f] <= chi_true[f] * (1.0 + 1e-4), (f, chi[f], chi_true[f])
        for j in FREE7:
            d = _pa_diff(rows[f, j], trues[f, j]) if j == wl.IX_PA else abs(rows[f, j] - trues[f, j])
            assert d <= 3.0 * TABLE3[j], (f, j, rows[f, j], trues[f, j])


def test_nested_sampling_finds_the_mode(oracle, torch_cuda, gbk):
    w0 = wl.config(1)
    true = _true_row(w0)
    w, obs = _case(oracle, 1, true)
    b = wl.box(w)
    with gbk.Problem(**pu.gbk_desc(w, obs)) as prob:
        r = gbk.gbk_fit_ns(prob.handle, true, 0, FREE4, b[FREE4, 0], b[FREE4, 1], n_live=200,
                           batch=1024, max_batches=150, enlarge=0.3, tol=0.01, seed=20151001)
        r2 = gbk.gbk_fit_ns(prob.handle, true, 0, FREE4, b[FREE4, 0], b[FREE4, 1], n_live=200,
                            batch=1024, max_batches=150, enlarge=0.3, tol=0.01, seed=20151001)
    assert np.isfinite(r["log_evidence"]) and np.isfinite(r["best_chi2"])
    assert r["stats"]["evals"] >= 200 and r["stats"]["launches"] == r["stats"]["iterations"] + 1
    for row in (r["best_row"], r["mean_row"]):
        assert _pa_diff(row[wl.IX_PA], true[wl.IX_PA]) <= 2.0
        assert abs(row[wl.IX_INC] - true[wl.IX_INC]) <= 2.0
        assert abs(row[wl.IX_VT] - true[wl.IX_VT]) <= 10.0
        assert abs(row[wl.IX_RT] - true[wl.IX_RT]) <= 1.0
    # same seed, same path (the kernels are bit-reproducible)
    assert r2["log_evidence"] == r["log_evidence"] and np.array_equal(r2["best_row"], r["best_row"])


def test_driver_argument_errors(oracle, torch_cuda, gbk):
    w0 = wl.config(1)
    true = _true_row(w0)
    w, obs = _case(oracle, 1, true)
    with gbk.Problem(**pu.gbk_desc(w, obs)) as prob:
        for call in (
            lambda: gbk.gbk_fit_ng(prob.handle, true, 0, [2, 2], [0, 0], [1, 1], 4, 2),       # twice
            lambda: gbk.gbk_fit_ng(prob.handle, true, 0, [2], [0.0], [1.0], 1, 2),            # one node
            lambda: gbk.gbk_fit_ng(prob.handle, true, 0, [2], [0.0], [1.0], 4, 2, accuracy=[0.0]),   # threshold 0
            lambda: gbk.gbk_fit_ng(prob.handle, true, 0, [2], [1.0], [1.0], 4, 2),            # empty box
            lambda: gbk.gbk_fit_ng(prob.handle, true, 5, [2], [0.0], [1.0], 4, 2),            # gal
            lambda: gbk.gbk_fit_lm(prob.handle, true[None], None, [11], [0.0], [1.0]),        # index
            lambda: gbk.gbk_fit_ns(prob.handle, true, 0, [2], [0.0], [1.0], n_live=1),
        ):
            with pytest.raises(gbk.GbkError) as ei:
                call()
            assert ei.value.code == gbk.GBK_ERR_ARG


def test_lm_with_the_velocity_field_strategy_and_epinat_curve(oracle, torch_cuda, gbk):
    """The GHASP set-up of the paper: velocity-field strategy + Epinat curve, centre
    fixed, seven free parameters (PA, i, V_sys, V_t, r_t, a, g), fitted by the LM driver through
    gbk_set_strategy.  Noise-free data: the model velocity field must be reproduced (the four curve
    parameters are partly degenerate, so the check is on chi^2 and on the geometric parameters)."""
    w = wl.config(3).scaled(nx=48, ny=40, rc_model=wl.RC_EPINAT, noise=0.0)
    true = np.array([23.6, 19.7, 123.0, 52.0, 8.0, 180.0, 3.5, 40.0, 8.0, 1.0, 1.3, 0.9], dtype=np.float32)
    g = pu.oracle_grid(oracle, w)
    z = np.zeros((w.ny, w.nx), np.float32)
    v = oracle.vfield_rows(g, z, z + 1, None, true[None], want_maps=True)["vmap"][0]
    obs = wl.Observed(v[None].astype(np.float32), np.full((1, w.ny, w.nx), 5.0, np.float32),
                      np.zeros((1, w.ny, w.nx), np.float32), np.ones((1, w.ny, w.nx), np.float32),
                      np.ones((1, w.ny, w.nx), np.uint8))
    free = [wl.IX_PA, wl.IX_INC, wl.IX_VSYS, wl.IX_VT, wl.IX_RT, 10, 11]       # ..., a, g
    lo = np.array([30.0, 20.0, -50.0, 50.0, 1.0, 0.3, 0.3], np.float32)
    hi = np.array([210.0, 80.0, 50.0, 400.0, 10.0, 3.0, 3.0], np.float32)
    start = true.copy()
    start[free] = (110.0, 45.0, 0.0, 150.0, 3.0, 1.0, 1.0)          # a = g = 1 as in PAPER.md:154
    with gbk.Problem(**pu.gbk_desc(w, obs)) as prob:
        assert prob.info.strategy == gbk.GBK_STRATEGY_VFIELD          # Epinat problems start there
        rows, chi, iters, st = gbk.gbk_fit_lm(prob.handle, start, None, free, lo, hi, max_iter=100)
    npix = w.nx * w.ny
    assert chi[0] < 1e-3 * npix, chi          # rms residual < 0.03 sigma = 0.16 km/s
    assert _pa_diff(rows[0, wl.IX_PA], true[wl.IX_PA]) <= 1.0
    assert abs(rows[0, wl.IX_VSYS] - true[wl.IX_VSYS]) <= 1.0
    assert st["converged"] == 1


def test_nested_grids_with_the_velocity_field_strategy(oracle, torch_cuda, gbk):
    w0 = wl.config(3).scaled(nx=32, ny=32, nv=48)
    true = _true_row(w0)
    w, obs = _case(oracle, 3, true, nx=32, ny=32, nv=48)
    b = wl.box(w)
    with gbk.Problem(**pu.gbk_desc(w, obs)) as prob:
        gbk.gbk_set_strategy(prob.handle, gbk.GBK_STRATEGY_VFIELD)
        assert gbk.gbk_get_info(prob.handle).strategy == gbk.GBK_STRATEGY_VFIELD
        best, chi, st = gbk.gbk_fit_ng(prob.handle, true, 0, FREE4, b[FREE4, 0], b[FREE4, 1], 6, 3)
        rows = wl.nested_grid_rows(w, true, level=0, nodes=6)
        ref = prob.eval_vfield(torch_cuda.from_numpy(rows).cuda())["chi2"]
        k = int(torch_cuda.argmin(ref).item())
    assert st["evals"] == 3 * 6 ** 4 and np.isfinite(chi)
    assert chi <= float(ref[k].item()) * (1 + 1e-6)       # later levels can only improve on level 0


def test_monte_carlo_errors_are_consistent_table5(oracle, torch_cuda, gbk):
    """Monte-Carlo error estimation as the paper does for DYNAMO (refits of
    noise-perturbed data) as ONE batched LM call: G galaxies x R noise realisations are R*G data sets
    of one problem.  The scatter of the refits is the error bar; the standardised residuals of one
    realisation must then be distributed like Table 5 says (~68 % within 1 sigma,
    ~95 % within 2 sigma)."""
    G, R = 20, 48
    w = wl.config(5).scaled(nx=30, ny=30, nv=64, n_gal=G * R, err_lo=5.0, err_hi=5.0, noise=5.0,
                            psf_fwhm_hi=0.0, psf_fwhm=2.0)
    rng = wl.rng_for(5, 77)
    trues = wl.draw_rows(w, rng, G)
    trues[:, wl.IX_INC] = rng.uniform(35.0, 70.0, G)      # away from the V_t - i degeneracy's ends
    trues[:, wl.IX_VT] = rng.uniform(120.0, 300.0, G)
    g = pu.oracle_grid(oracle, w)
    clean = [oracle.model_maps(g, t.astype(np.float64)) for t in trues]
    m0, m1, m2 = (np.repeat(np.stack([c[i] for c in clean]), R, axis=0) for i in range(3))
    obs = wl.observe(w, m0, m1, m2, rng)                  # independent noise per data set
    b = wl.box(w)
    lo, hi = b[FREE7, 0].copy(), b[FREE7, 1].copy()
    lo[2], hi[2] = -360.0, 720.0
    lo[3], hi[3] = 5.0, 88.0
    hi[5] = 600.0
    starts = np.repeat(trues, R, axis=0).astype(np.float64)
    starts[:, FREE7] += 0.03 * (b[FREE7, 1] - b[FREE7, 0]) * rng.uniform(-1, 1, (G * R, 7))
    with gbk.Problem(**pu.gbk_desc(w, obs)) as prob:
        rows, chi, iters, st = gbk.gbk_fit_lm(prob.handle, starts, np.arange(G * R), FREE7, lo, hi,
                                              max_iter=60, ftol=1e-7)
    assert st["converged"] >= 0.98 * G * R and np.isfinite(chi).all()
    fit = rows[:, FREE7].astype(np.float64).reshape(G, R, 7)
    sigma = fit[:, 1:].std(axis=1, ddof=1)                 # error bars from realisations 1..R-1
    z = (fit[:, 0] - trues[:, FREE7]) / sigma              # realisation 0 plays "the observation"
    f1, f2 = float((np.abs(z) < 1).mean()), float((np.abs(z) < 2).mean())
    print("Table-5 fractions within 1 and 2 sigma:", f1, f2, "median sigma:", np.median(sigma, axis=0))
    assert 0.52 <= f1 <= 0.84 and f2 >= 0.86, (f1, f2)
    # the reduced chi^2 of the fits is ~1 (eq. 11 with the right error bars)
    ndof = 2 * obs.mask.reshape(G * R, -1).sum(axis=1) - 7
    assert 0.9 < float(np.median(chi / ndof)) < 1.1


def test_lm_failure_states_are_reported_not_counted_as_converged(oracle, torch_cuda, gbk):
    """A fit that cannot iterate ends as FAILED (gbk_fit_stats.failed), never as converged: a start row that
    is out of domain is returned unchanged with chi^2 = +INF; a finite-difference row that leaves the
    domain (sigma_0 free, stepping to sigma_0 <= 0) stops the fit; a step far below one ulp of the
    parameter is doubled until it moves the parameter, so no difference is ever divided by a zero step: the
    fit then either iterates or fails on a noise-dominated Jacobian, but never returns non-finite rows."""
    w0 = wl.config(1)
    true = _true_row(w0)
    w, obs = _case(oracle, 1, true)
    b = wl.box(w)
    lo, hi = b[FREE7, 0].copy(), b[FREE7, 1].copy()
    lo[2], hi[2] = -360.0, 720.0
    starts = np.repeat(true[None], 3, axis=0).astype(np.float32)
    starts[:, wl.IX_VT] += 15.0
    starts[1, wl.IX_R0] = -1.0                      # out of domain from the start
    with gbk.Problem(**pu.gbk_desc(w, obs)) as prob:
        chi_start = float(prob.eval(torch_cuda.from_numpy(starts[:1]).cuda())["chi2"].item())
        rows, chi, iters, st = gbk.gbk_fit_lm(prob.handle, starts, None, FREE7, lo, hi)
        assert st["failed"] == 1 and st["converged"] == 2
        assert np.isposinf(chi[1]) and iters[1] == 0 and np.array_equal(rows[1], starts[1])
        assert np.isfinite(chi[[0, 2]]).all() and abs(rows[0, wl.IX_VT] - true[wl.IX_VT]) <= 5.0
        # sigma_0 free with a backward difference that crosses zero: the difference row is out of domain
        s = true.copy()
        s[wl.IX_SIG] = 1e-3
        r2, c2, i2, st2 = gbk.gbk_fit_lm(prob.handle, s[None], None, [wl.IX_SIG], [1e-3], [2e-3 - 1e-9],
                                         rel_step=4.0)      # step 4 x the box width: forward leaves the box, backward crosses 0
        assert st2["failed"] == 1 and st2["converged"] == 0 and np.array_equal(r2[0], s)
        # a step of 1e-12 of the box is far below one ulp of V_t = 195: doubled until it moves the parameter
        r3, c3, i3, st3 = gbk.gbk_fit_lm(prob.handle, starts[:1], None, FREE7, lo, hi, rel_step=1e-12, max_iter=5)
        assert np.isfinite(r3).all() and np.isfinite(c3[0]) and c3[0] <= chi_start * (1 + 1e-6)
        assert st3["failed"] + st3["converged"] <= 1


def test_nested_grids_ghasp_setup_six_axes_on_the_velocity_field(oracle, torch_cuda, gbk):
    """The paper's GHASP configuration of the nested-grid optimiser: velocity-field
    strategy, Epinat curve, grid 7 x 11 x 11 x 5 x 5 over (PA, r_t, V_t, a, g) -- sigma is not part of a
    velocity field -- with V_sys, centre and inclination fixed; 21 175 rows per level, refined to the
    paper's accuracy thresholds.  Noise-free data: the velocity field must be reproduced."""
    w = wl.config(3).scaled(nx=40, ny=36, rc_model=wl.RC_EPINAT, noise=0.0)
    true = np.array([19.6, 17.7, 123.0, 52.0, 8.0, 180.0, 3.5, 40.0, 8.0, 1.0, 1.3, 0.9], dtype=np.float32)
    g = pu.oracle_grid(oracle, w)
    z = np.zeros((w.ny, w.nx), np.float32)
    v = oracle.vfield_rows(g, z, z + 1, None, true[None], want_maps=True)["vmap"][0]
    obs = wl.Observed(v[None].astype(np.float32), np.full((1, w.ny, w.nx), 5.0, np.float32),
                      np.zeros((1, w.ny, w.nx), np.float32), np.ones((1, w.ny, w.nx), np.float32),
                      np.ones((1, w.ny, w.nx), np.uint8))
    axes = [wl.IX_PA, wl.IX_RT, wl.IX_VT, 10, 11]
    lo = np.array([0.0, 1.0, 50.0, 0.3, 0.3], np.float32)
    hi = np.array([360.0, 8.0, 300.0, 3.0, 3.0], np.float32)
    with gbk.Problem(**pu.gbk_desc(w, obs)) as prob:
        assert prob.info.strategy == gbk.GBK_STRATEGY_VFIELD
        best, chi, st = gbk.gbk_fit_ng(prob.handle, true, 0, axes, lo, hi, [7, 11, 11, 5, 5], 30,
                                       accuracy=[0.1, 0.01, 0.1, 0.1, 0.1])
    assert st["converged"] == 1 and st["evals"] == st["iterations"] * 7 * 11 * 11 * 5 * 5
    npix = w.nx * w.ny
    assert chi < 0.05 * npix, chi                    # rms residual < 0.22 sigma = 1.1 km/s on a 5 km/s error map
    assert _pa_diff(best[wl.IX_PA], true[wl.IX_PA]) <= 1.0
