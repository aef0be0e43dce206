"""gbk_eval_batch_static (include/gbk.h): the eval call that allocates nothing, against gbk_eval_batch.

Collected last on purpose (the name): the run is `pytest -x`, and a failure here must not hide
the other tests.  Self-contained: its own seeded inputs, no oracle, passes alone in a fresh process and
after the rest of the suite (the static array then holds whatever earlier calls left in it).
"""
import numpy as np
import pytest

from paper_1510_01815_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL_CHI2_REL = 1e-4      # BASELINE.json's chi^2 tolerance, as in tests/parity_util.py
TOL_M0_REL = 1e-4
TOL_M12_ABS = 0.05       # km/s


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


def _desc(rng, nx=37, ny=29, nv=40, u=2, tile=(8, 6)):
    """A seeded problem of several ragged tiles: a plausible velocity map with noise, 10 % masked."""
    yy, xx = np.mgrid[0:ny, 0:nx]
    vobs = (120.0 * np.tanh((xx - nx / 2) / 6.0) + rng.normal(0, 5, (ny, nx))).astype(np.float32)
    sobs = (35.0 + 10.0 * rng.random((ny, nx))).astype(np.float32)
    mask = (rng.random((ny, nx)) > 0.1).astype(np.uint8)
    return dict(nx=nx, ny=ny, nv=nv, u=u, v_center=0.0, dv=20.0, rc_model=wl.RC_ARCTAN, n_gal=1,
                vobs=vobs[None], verr=np.full((1, ny, nx), 5.0, np.float32), sobs=sobs[None],
                serr=np.full((1, ny, nx), 5.0, np.float32), mask=mask[None], psf_kind=wl.PSF_GAUSSIAN,
                psf_fwhm=np.asarray([2.5], np.float32), lsf_sigma=25.0, tile_w=tile[0], tile_h=tile[1])


def _rows(rng, K, nx, ny):
    rows = np.empty((K, 10), np.float32)
    rows[:, 0] = nx / 2 + rng.uniform(-2, 2, K)
    rows[:, 1] = ny / 2 + rng.uniform(-2, 2, K)
    rows[:, 2] = rng.uniform(60, 120, K)      # PA
    rows[:, 3] = rng.uniform(25, 70, K)       # inclination
    rows[:, 4] = rng.uniform(-20, 20, K)      # V_sys
    rows[:, 5] = rng.uniform(100, 220, K)     # V_t
    rows[:, 6] = rng.uniform(2, 8, K)         # r_t
    rows[:, 7] = rng.uniform(25, 50, K)       # sigma_0
    rows[:, 8] = rng.uniform(4, 10, K)        # r_0
    rows[:, 9] = rng.uniform(0.5, 2, K)       # I_0
    return rows


def _outputs(torch, K, ny, nx):
    dev = "cuda:0"
    return dict(chi2=torch.full((K,), -1.0, dtype=torch.float32, device=dev),
                m0=torch.full((K, ny, nx), -1.0, dtype=torch.float32, device=dev),
                m1=torch.full((K, ny, nx), -1.0, dtype=torch.float32, device=dev),
                m2=torch.full((K, ny, nx), -1.0, dtype=torch.float32, device=dev),
                resid=torch.full((K, 2, ny, nx), -1.0, dtype=torch.float32, device=dev))


def _close(torch, got, ref, K):
    g = {k: v.cpu().numpy().astype(np.float64) for k, v in got.items()}
    r = {k: v.cpu().numpy().astype(np.float64) for k, v in ref.items()}
    assert np.all(np.isfinite(r["chi2"])) and np.all(r["chi2"] > 0), "the existing path must give real chi^2 here"
    assert np.all(np.abs(g["chi2"] - r["chi2"]) <= TOL_CHI2_REL * np.abs(r["chi2"]))
    assert np.all(np.abs(g["m0"] - r["m0"]) <= TOL_M0_REL * np.abs(r["m0"]))
    for k in ("m1", "m2"):
        assert np.array_equal(np.isnan(g[k]), np.isnan(r[k]))
        assert np.nanmax(np.abs(g[k] - r[k])) <= TOL_M12_ABS
    assert np.nanmax(np.abs(g["resid"] - r["resid"])) <= TOL_M12_ABS / 5.0 + 1e-6
    # same kernel, same fixed-order reduction: in fact the two agree to the bit
    for k in g:
        assert np.array_equal(g[k], r[k], equal_nan=True), k


def test_static_scratch_entry_matches_the_existing_path_on_two_calls_in_a_row(torch_cuda, gbk):
    torch = torch_cuda
    rng = np.random.default_rng(20261105)
    desc = _desc(rng)
    nx, ny = desc["nx"], desc["ny"]
    with gbk.Problem(**desc) as prob:
        info = prob.info
        assert info.tiles_x * info.tiles_y > 1, "the case must use the cross-tile scratch"
        st = torch.cuda.current_stream().cuda_stream
        # two calls in a row on the same stream: 24 rows, then 7 other rows (the array still holds the first
        # call's partials and whatever counters state it left)
        cases = []
        for K in (24, 7):
            p = torch.from_numpy(_rows(rng, K, nx, ny)).cuda()
            cases.append((K, p, _outputs(torch, K, ny, nx)))
        for K, p, out in cases:
            gbk.gbk_eval_batch_static(prob.handle, p, None, K, out["chi2"], out["m0"], out["m1"], out["m2"],
                                      out["resid"], st)
        torch.cuda.synchronize()
        for K, p, out in cases:
            ref = _outputs(torch, K, ny, nx)
            gbk.gbk_eval_batch(prob.handle, p, None, K, ref["chi2"], ref["m0"], ref["m1"], ref["m2"],
                               ref["resid"], st)
            torch.cuda.synchronize()
            _close(torch, out, ref, K)
        # chi^2 only (the other instantiation of the kernel), a third call
        K, p, out = cases[0]
        chi = torch.full((K,), -1.0, dtype=torch.float32, device="cuda:0")
        gbk.gbk_eval_batch_static(prob.handle, p, None, K, chi, stream=st)
        torch.cuda.synchronize()
        assert torch.equal(chi, out["chi2"])


def test_static_scratch_entry_rejects_what_does_not_fit(torch_cuda, gbk):
    torch = torch_cuda
    rng = np.random.default_rng(7)
    desc = _desc(rng, nx=12, ny=10, nv=24, u=1, tile=(4, 4))
    with gbk.Problem(**desc) as prob:
        tiles = prob.info.tiles_x * prob.info.tiles_y
        assert tiles == 9
        for K in (gbk.GBK_STATIC_MAX_ROWS + 1, gbk.GBK_STATIC_MAX_PARTIALS // tiles + 1):
            p = torch.from_numpy(np.repeat(_rows(rng, 1, 12, 10), K, axis=0)).cuda()
            chi = torch.zeros(K, dtype=torch.float32, device="cuda:0")
            with pytest.raises(gbk.GbkError) as e:
                gbk.gbk_eval_batch_static(prob.handle, p, None, K, chi)
            assert e.value.code == gbk.GBK_ERR_ARG and "GBK_STATIC_MAX" in str(e.value)
        # the largest batch that fits runs, and agrees with the existing path
        K = min(gbk.GBK_STATIC_MAX_ROWS, gbk.GBK_STATIC_MAX_PARTIALS // tiles)
        p = torch.from_numpy(_rows(rng, K, 12, 10)).cuda()
        chi = torch.zeros(K, dtype=torch.float32, device="cuda:0")
        ref = torch.zeros(K, dtype=torch.float32, device="cuda:0")
        gbk.gbk_eval_batch_static(prob.handle, p, None, K, chi)
        gbk.gbk_eval_batch(prob.handle, p, None, K, ref)
        torch.cuda.synchronize()
        assert torch.equal(chi, ref)
        prob.set_extraction(gbk.GBK_EXTRACT_GAUSSFIT)
        with pytest.raises(gbk.GbkError) as e:
            gbk.gbk_eval_batch_static(prob.handle, p[:4].contiguous(), None, 4, chi)
        assert e.value.code == gbk.GBK_ERR_UNSUPPORTED
