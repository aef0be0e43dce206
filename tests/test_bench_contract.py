"""bench.py's reference arm (this tier: the oracle timed on the host cores) runs without a GPU and prints
one JSON line with the keys the driver reads; and the per-config op counts of the roofline are the
SURVEY.md section 8(d) figures."""
import json
import os
import subprocess
import sys
import types

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_the_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0", "--ref-rows", "2"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "evals/s" and d["higher_is_better"] is True
    assert d["value"] > 0 and d["steps"] == 1 and d["dtype"] == "f64" and d["data"] == "synthetic"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": "evals/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert "workload" in d["config"] and d["vs_baseline"] is None


def test_algorithmic_op_count_is_the_survey_figure():
    """Config 3: 5 x 415 872 + 45 x 5 776 + 3 x 26 x 4 096 + 12 x 4 096 = 2 707 920 lane-ops per evaluation
    (SURVEY.md section 8(d)); config 4 with its 225-tap image: 68 715 732."""
    sys.path.insert(0, ROOT)
    import bench
    from paper_1510_01815_b200 import workloads as wl
    w = wl.config(3)
    info = types.SimpleNamespace(nv=64, r_v=4, tile_w=64, tile_h=64, tiles_x=1, tiles_y=1)
    n = bench.op_counts(info, w, np.full(4096, bench.psf_radius(w, w.psf_fwhm)))
    assert bench.psf_radius(w, w.psf_fwhm) == 6
    assert n["ext_voxels_per_eval"] == 415872 and n["ext_samples_per_eval"] == 5776
    assert n["ops_per_eval"] == 5 * 415872 + 45 * 5776 + 3 * 26 * 4096 + 12 * 4096 == 2707920
    w4 = wl.config(4)
    info4 = types.SimpleNamespace(nv=48, r_v=4, tile_w=64, tile_h=64, tiles_x=4, tiles_y=4)
    n4 = bench.op_counts(info4, w4, np.full(256, 7))
    # the algorithmic count extends the WHOLE FIELD by one PSF halo (SURVEY's 6.87e7 for config 4), whatever the
    # tiling; the halos the 16 tiles re-evaluate are reported apart
    assert n4["ext_samples_per_eval"] == 270 * 270 and n4["ext_samples_per_eval_tiled"] == 16 * 78 * 78
    assert n4["ops_per_eval"] == 5 * 270 * 270 * 56 + 45 * 270 * 270 + 3 * 225 * 65536 + 12 * 65536 == 68715732
    assert n4["ops_per_eval_tiled"] == 5 * 16 * 78 * 78 * 56 + 45 * 16 * 78 * 78 + 3 * 225 * 65536 + 12 * 65536
    assert n["ops_per_eval_tiled"] == n["ops_per_eval"]
