"""Gauge-invariant classes (k, m, m') of PAPER.md:393 (class sums): the class of a graph is pinned to the
paper's own Table I (column N_diag: how many of the 3213 five-loop graphs fall into each of the nine
classes), for the oracle's plain definition and for the product's fg_graph_class separately; the class totals of a batch
(combination (19) restricted to a class, fg_batch_class_total) are checked on synthetic block results.  No GPU."""
import collections
import ctypes as C

import numpy as np
import pytest

from conftest import read_facts
from oracle import oracle as O
from paper_1909_08015_b200 import inputs

FACTS = read_facts()
TABLE_I = {tuple(int(t) for t in s.split(":")[0].split(",")): int(s.split(":")[1]) for s in FACTS["class_ndiag_5loop"]}


@pytest.fixture(scope="module")
def fg():
    from paper_1909_08015_b200 import build, fg as m
    build.build()
    return m


def undirected(graphs):
    """One representative of every pair (graph, mirror image): the paper counts graphs up to the direction of the electron line."""
    seen = set(); out = []
    for x, ph in graphs:
        key = (x, tuple(sorted(tuple(sorted(p)) for p in ph)))
        mx, mph = inputs.mirror(x, ph)
        mkey = (mx, tuple(sorted(tuple(sorted(p)) for p in mph)))
        if min(key, mkey) in seen:
            continue
        seen.add(min(key, mkey)); out.append((x, ph))
    return out


def test_table_one_counts_nine_classes_3213_graphs():
    assert len(TABLE_I) == 9 and sum(TABLE_I.values()) == int(FACTS["n_graphs_5loop_undirected"][0])
    assert all(k + m + mp == 5 and m >= mp and k >= 1 for k, m, mp in TABLE_I)


def test_oracle_classes_reproduce_table_one():
    und = undirected(O.enumerate_graphs(5))
    assert len(und) == 3213
    counts = collections.Counter(O.gauge_class(x, ph) for x, ph in und)
    assert dict(counts) == TABLE_I


def test_product_classes_reproduce_table_one_and_agree_with_the_oracle(fg):
    graphs = inputs.all_graphs(5)
    assert len(graphs) == 6354
    cls = {}
    for x, ph in graphs:
        c = fg.Graph(inputs.edge_list(x, ph), x).gauge_class()
        assert c == O.gauge_class(x, ph)
        mx, mph = inputs.mirror(x, ph)
        assert fg.Graph(inputs.edge_list(mx, mph), mx).gauge_class() == c          # a class does not depend on the direction
        cls[(x, tuple(ph))] = c
    counts = collections.Counter(cls[(x, tuple(ph))] for x, ph in undirected(graphs))
    assert dict(counts) == TABLE_I


def test_small_loop_counts(fg):
    # n = 1: the single graph is (1, 0, 0); n = 2: ladder and crossed graph are (2, 0, 0), the other four (1, 1, 0)
    assert [fg.Graph(inputs.edge_list(x, ph), x).gauge_class() for x, ph in inputs.all_graphs(1)] == [(1, 0, 0)]
    c2 = collections.Counter(fg.Graph(inputs.edge_list(x, ph), x).gauge_class() for x, ph in inputs.all_graphs(2))
    assert dict(c2) == {(2, 0, 0): 2, (1, 1, 0): 4}
    for n in (3, 4):
        for x, ph in inputs.all_graphs(n):
            k, m, mp = fg.Graph(inputs.edge_list(x, ph), x).gauge_class()
            assert (k, m, mp) == O.gauge_class(x, ph) and k + m + mp == n and k >= 1


class FakePlan:
    def __init__(self, k):
        self.h = C.c_void_p(0x2000 + 16 * k)


def test_class_totals_follow_combination_19(fg):
    from paper_1909_08015_b200 import sched
    rng = np.random.default_rng(11)
    classes = [(2, 0, 0), (1, 1, 0), (1, 1, 0), (2, 0, 0), (1, 1, 0), (1, 1, 0)]
    b = sched.Batch([FakePlan(k) for k in range(6)])
    b.set_classes(classes)
    mean = []; var = []
    for j in range(6):
        y = rng.normal(0.3 * j - 0.5, 1.0 + j, 5000)
        r = fg.fg_result(); sy = float(np.sum(y)); sy2 = float(np.sum(y * y)); n = len(y)
        r.sum_y[0] = sy; r.sum_y2[0] = sy2; r.n_samples = n; r.mean = sy / n; r.variance = sy2 / n ** 2 - sy ** 2 / n ** 3
        b.fold(j, r, 1e-3)
        mean.append(r.mean); var.append(r.variance)
    tot = b.total(); acc_v = 0.0; acc_s2 = 0.0
    for c in ((2, 0, 0), (1, 1, 0)):
        idx = [j for j in range(6) if classes[j] == c]
        t = b.class_total(c)
        assert t["n_graphs"] == len(idx)
        assert t["value"] == pytest.approx(sum(mean[j] for j in idx), rel=1e-14)
        assert t["sigma_down"] == pytest.approx(sum(var[j] for j in idx) ** 0.5, rel=1e-14)          # (19)
        acc_v += t["value"]; acc_s2 += t["sigma_down"] ** 2
    assert acc_v == pytest.approx(tot["value"], rel=1e-14) and acc_s2 ** 0.5 == pytest.approx(tot["sigma_down"], rel=1e-14)
    assert b.class_total((5, 0, 0)) == dict(value=0.0, sigma_down=0.0, n_graphs=0)
