"""CPU-only checks of the boundary and the rank plumbing (no compute calls without a GPU):
  * libgbk.so loads and exports every function include/gbk.h declares, and the ctypes binding
    declares the same names;
  * the struct layouts of the binding match the header's field order;
  * compute calls fail loudly (an error code, never a CPU fallback) when there is no CUDA device;
  * rows shard without overlap, and the world-size-2 gloo path aggregates as bench.py expects.
"""
import ctypes as C
import os
import re
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "gbk.h")


def _header_text():
    with open(HEADER) as f:
        text = f.read()
    return re.sub(r"/\*.*?\*/", " ", text, flags=re.S)   # comments stripped


def _declared_functions():
    names = re.findall(r"\b(gbk_[a-z0-9_]+)\s*\(", _header_text())
    return sorted(set(names))


def _struct_fields(name):
    body = re.search(r"typedef struct \{([^{}]*)\}\s*" + name + r"\s*;", _header_text(), flags=re.S).group(1)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        decl = re.sub(r"^(const\s+)?(float|int32_t|int64_t|uint8_t|double)\b", "", decl)
        fields += [re.sub(r"[\s\*]", "", part) for part in decl.split(",")]
    return fields


@pytest.fixture(scope="module")
def libgbk():
    from paper_1510_01815_b200 import build, gbk
    build.build_lib()
    return gbk


def test_library_exports_every_declared_symbol(libgbk):
    names = _declared_functions()
    assert {"gbk_create_problem", "gbk_eval_batch", "gbk_destroy", "gbk_last_error",
            "gbk_eval_batch_unfused", "gbk_eval_batch_host", "gbk_get_info"} <= set(names)
    raw = C.CDLL(libgbk.LIB_PATH)
    for n in names:
        assert hasattr(raw, n), f"libgbk.so does not export {n}"
        assert hasattr(libgbk, n), f"the Python binding has no function named {n}"
    assert sorted(libgbk.EXPORTS) == names          # the binding's list is the header's, nothing less


def test_binding_struct_layout_follows_the_header(libgbk):
    for cname in ("gbk_problem_desc", "gbk_problem_info", "gbk_fit_stats"):
        want = _struct_fields(cname)
        got = [f[0] for f in getattr(libgbk, cname)._fields_]
        assert got == want, (cname, got, want)
    assert libgbk.GBK_P == 10 == int(re.search(r"#define GBK_P (\d+)", _header_text()).group(1))


def test_no_cpu_fallback_without_a_device(libgbk):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    z = np.zeros((1, 4, 4), np.float32)
    with pytest.raises(libgbk.GbkError) as ei:
        libgbk.Problem(nx=4, ny=4, nv=8, dv=10.0, vobs=z, verr=z + 1, sobs=z, serr=z + 1,
                       psf_fwhm=np.asarray([2.0], np.float32), lsf_sigma=10.0)
    assert ei.value.code == libgbk.GBK_ERR_CUDA
    assert libgbk.gbk_last_error() != ""


def test_argument_errors_need_no_device(libgbk):
    z = np.zeros((1, 4, 4), np.float32)
    for bad in (dict(u=0), dict(dv=0.0), dict(rc_model=7), dict(psf_kind=5), dict(nv=0)):
        kw = dict(nx=4, ny=4, nv=8, dv=10.0, vobs=z, verr=z + 1, sobs=z, serr=z + 1,
                  psf_fwhm=np.asarray([2.0], np.float32), lsf_sigma=10.0)
        kw.update(bad)
        with pytest.raises(libgbk.GbkError) as ei:
            libgbk.Problem(**kw)
        assert ei.value.code == libgbk.GBK_ERR_ARG, bad
    libgbk.gbk_destroy(None)   # NULL is a no-op


def test_shard_rows_partitions_exactly():
    from paper_1510_01815_b200 import workloads as wl
    for K in (0, 1, 7, 4096, 16385):
        for world in (1, 2, 3, 8):
            spans = [wl.shard_rows(K, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == K
            for (a0, a1), (b0, b1) in zip(spans, spans[1:]):
                assert a1 == b0 and a0 <= a1 and b0 <= b1
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _gloo_worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    from paper_1510_01815_b200 import dist, workloads as wl
    r = dist.init_from_env("gloo")
    try:
        assert (r.rank, r.world) == (rank, world)
        lo, hi = wl.shard_rows(4097, r.rank, r.world)
        dist.barrier(r)
        tmax = dist.max_over_ranks(r, 1.0 + rank)            # slowest rank
        total = dist.sum_over_ranks(r, hi - lo)
        value, sec = dist.aggregate_throughput(r, hi - lo, 0.5 * (1 + rank))
        out.put((rank, lo, hi, tmax, total, value, sec))
    finally:
        dist.finalize(r)


def test_world_size_2_gloo_aggregation():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_gloo_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, lo0, hi0, tmax0, tot0, v0, s0), (r1, lo1, hi1, tmax1, tot1, v1, s1) = got
    assert (lo0, hi0, lo1, hi1) == (0, 2049, 2049, 4097)
    assert tmax0 == tmax1 == 2.0                  # max over ranks, seen by both
    assert tot0 == tot1 == 4097.0                 # every row counted once
    assert s0 == s1 == 1.0 and v0 == v1 == 4097.0  # whole-job units / slowest rank's time
