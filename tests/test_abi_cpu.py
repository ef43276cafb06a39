"""CPU-side checks of the product: the C-ABI library loads and exports every symbol include/fg.h declares, host-only
entry points (graph validation, result merge) behave, compute entry points fail loudly without a GPU, and the
world_size-2 sharding logic works over gloo.  No kernel runs here."""
import ctypes as C
import os
import re
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def fg():
    from paper_1909_08015_b200 import build, fg as m
    build.build()
    return m


def test_library_exports_every_declared_symbol(fg):
    hdr = open(os.path.join(ROOT, "include", "fg.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(fg_[a-z_0-9]+)\s*\(", hdr))
    assert len(declared) >= 19
    L = fg.lib()
    for name in declared:
        assert hasattr(L, name), name
    assert declared == set(fg.EXPORTS)
    assert b"sm_100a" in L.fg_version()


def test_graph_validation_errors(fg):
    from paper_1909_08015_b200 import inputs
    ok = fg.Graph(inputs.edge_list(1, [(0, 2)]), 1)
    assert ok.h
    with pytest.raises(fg.FgError) as e:       # 2 lines: not 3n
        fg.Graph([(0, 1, 0), (1, 2, 0)], 1)
    assert e.value.code == -2
    with pytest.raises(fg.FgError) as e:       # electron lines close a loop
        fg.Graph([(0, 1, 0), (1, 0, 0), (0, 2, 1)], 1)
    assert e.value.code == -3
    with pytest.raises(fg.FgError) as e:       # vertex 1 carries the external photon and an internal one
        fg.Graph([(0, 1, 0), (1, 2, 0), (0, 1, 1)], 1)
    assert e.value.code == -4
    with pytest.raises(fg.FgError) as e:       # self-energy insertion on an external leg: e_4 not spanned
        fg.Graph(inputs.edge_list(0, [(1, 2), (3, 4)]), 0)
    assert e.value.code == -5
    with pytest.raises(fg.FgError) as e:       # 6 loops
        fg.Graph([(i, i + 1, 0) for i in range(12)] + [(i, 12 - i, 1) for i in range(6)], 6)
    assert e.value.code == -6
    # arbitrary vertex labels are accepted when the electron lines chain u -> v
    g = fg.Graph([(2, 0, 0), (0, 1, 0), (2, 1, 1)], 0)
    assert g.h


def test_compute_calls_fail_loudly_without_gpu(fg):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_1909_08015_b200 import inputs
    g = fg.Graph(inputs.edge_list(1, [(0, 2)]), 1)
    with pytest.raises(fg.FgError) as e:
        fg.Plan(g)
    assert e.value.code == -7 and "no CPU path" in str(e.value)
    with pytest.raises(fg.FgError):
        fg.dfma_peak()


def _res(fg, sy, sy2, n, fl=0, rej=0, big=0):
    r = fg.fg_result()
    r.sum_y[0], r.sum_y[1] = sy; r.sum_y2[0], r.sum_y2[1] = sy2
    r.n_samples, r.n_flagged, r.n_rejected, r.n_pdf_big_exp = n, fl, rej, big
    return r


def test_result_merge_is_exact(fg):
    a = _res(fg, (1.0, 2.0 ** -60), (3.0, 0.0), 100, 1, 2, 3)
    b = _res(fg, (2.0 ** -70, 0.0), (5.0, 2.0 ** -58), 50, 4, 5, 6)
    m = fg.result_merge(a, b)
    assert m.n_samples == 150 and m.n_flagged == 5 and m.n_rejected == 7 and m.n_pdf_big_exp == 9
    from fractions import Fraction as F
    want = F(1) + F(2) ** -60 + F(2) ** -70
    assert F(m.sum_y[0]) + F(m.sum_y[1]) == want          # double-double sums add without loss
    assert F(m.sum_y2[0]) + F(m.sum_y2[1]) == F(8) + F(2) ** -58
    assert abs(m.mean - float(want) / 150) < 1e-18
    var = 8.0 / 150 ** 2 - 1.0 / 150 ** 3                  # (17)
    assert abs(m.variance - var) < 1e-15


def test_shard_ranges_partition_the_sample_ids():
    from paper_1909_08015_b200.dist import shard_range
    for n, w in ((10, 3), (7, 8), (10 ** 10, 8), (5, 1)):
        pos = 0
        for r in range(w):
            f, c = shard_range(n, r, w)
            assert f == pos and c >= 0
            pos += c
        assert pos == n


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, q):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_1909_08015_b200 import fg
    from paper_1909_08015_b200.dist import gather_and_merge, shard_range
    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    f, c = shard_range(1001, rank, world)
    r = _res(fg, (float(rank + 1), 2.0 ** -60 * (rank + 1)), (float(10 * (rank + 1)), 0.0), c, rank, 2 * rank, 0)
    m = gather_and_merge(r)
    q.put((rank, m.sum_y[0], m.sum_y[1], m.sum_y2[0], int(m.n_samples), int(m.n_flagged), int(m.n_rejected), m.mean))
    dist.barrier(); dist.destroy_process_group()


def test_world_size_2_gather_and_merge_over_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn"); q = ctx.Queue(); port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    got = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    for rank, sy0, sy1, s20, n, fl, rej, mean in got:     # every rank holds the same exact merge
        assert sy0 == 3.0 and sy1 == 3 * 2.0 ** -60 and s20 == 30.0 and n == 1001 and fl == 1 and rej == 2
        assert abs(mean - 3.0 / 1001) < 1e-18
