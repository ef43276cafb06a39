"""Host logic of the product's planner (fg_host_plan: no device, no kernels) against the paper and the oracle:
subgraphs, forests and operator table, Deg/Z tables (bit-exact), and the number of
non-zero Dirac coefficients.  The host combinatorics of the two sides were written from the same reading, so
agreement here only shows that neither drifted; what pins them to the paper's definitions is tests/test_dirac_and_subgraphs.py
(brute-force subgraphs, explicit 4x4 matrices) and the oracle pins of tests/test_oracle_pins.py."""
import numpy as np
import pytest

from conftest import read_facts
from oracle import oracle as O
from paper_1909_08015_b200 import inputs

FACTS = read_facts()


@pytest.fixture(scope="module")
def fg():
    from paper_1909_08015_b200 import build, fg as m
    build.build()
    return m


def _key(subs, t):
    return (t["sign"], tuple(sorted(((subs[m]["a"], subs[m]["b"]), op) for m, op in t["members"])))


@pytest.mark.parametrize("n,step", [(1, 1), (2, 1), (3, 7), (4, 97)])
def test_structure_tables_and_coefficient_counts_match_the_oracle(fg, n, step):
    for x, ph in inputs.all_graphs(n)[::step]:
        for merge in (False, True):
            g = fg.Graph(inputs.edge_list(x, ph), x)
            stats, subs, terms, deg, z1 = fg.host_plan(g, merge_ext_lines=merge, tables=True)
            o = O.Oracle(x, ph, merge=merge, printed=False, structure_only=(n == 4))
            osubs = o.subs()
            assert sorted((s["a"], s["b"], s["type"], s["in_chain"]) for s in subs) == sorted((s["a"], s["b"], s["type"], s["in_chain"]) for s in osubs)
            assert set(_key(subs, t) for t in terms) == set(_key(osubs, t) for t in o.terms())
            assert (stats["M"], stats["n_forests"], stats["n_terms"]) == (o.M, o.n_forests, o.n_terms)
            if n < 4:
                do, zo = o.tables()
                assert np.array_equal(deg, do) and np.array_equal(z1, zo)
                assert stats["n_coefs_nonzero"] == o.n_patterns
                assert stats["n_geoms"] == o.n_geoms and stats["n_nums"] == o.n_nums


def test_expression_11_from_the_planner(fg):
    x = int(FACTS["eq11_x"][0]); ph = [tuple(int(t) for t in s.split("-")) for s in FACTS["eq11_photons"]]
    g = fg.Graph(inputs.edge_list(x, ph), x)
    stats, subs, terms = fg.host_plan(g, merge_ext_lines=True)
    want = sorted(tuple(int(t) for t in s.split("-")) for s in FACTS["eq11_subgraphs"])
    assert sorted((s["a"], s["b"]) for s in subs) == want
    assert stats["n_forests"] == int(FACTS["eq11_forests"][0]) and stats["n_terms"] == int(FACTS["eq11_terms"][0])
    assert stats["M"] == 14 and stats["n_loops"] == 5          # 13 integration dimensions
    types = {(s["a"], s["b"]): s["type"] for s in subs}
    assert types[(2, 3)] == "SE" and types[(5, 8)] == "SE" and types[(5, 7)] == "V" and types[(0, 10)] == "V"
    # every term has exactly one A; G carries A or L-U; members outside the chain carry U
    idx = {(s["a"], s["b"]): k for k, s in enumerate(subs)}
    for t in terms:
        ops = [op for _, op in t["members"]]
        assert ops.count("A") == 1
        gop = dict(t["members"])[idx[(0, 10)]]
        assert gop in ("A", "L-U")
        for m, op in t["members"]:
            if not subs[m]["in_chain"]:
                assert op == "U"
    assert stats["flops_per_sample"] > 1e5 and stats["n_coefs"] >= stats["n_coefs_nonzero"] > 1e5


def test_ladder_and_limits(fg):
    g = fg.Graph(inputs.edge_list(4, [(0, 8), (1, 7), (2, 6), (3, 5)]), 4)
    stats, subs, terms = fg.host_plan(g)
    assert (stats["n_subgraphs"], stats["n_forests"], stats["n_terms"]) == (4, 8, 20)
    table = np.array([bin(s).count("1") for s in range(1 << 12)], dtype=np.float64)          # Deg(s) = |s|: uniform density
    _, _, _, deg, z1 = fg.host_plan(g, deg_table=table, tables=True)
    assert np.all(z1[:-1] == 1.0) and z1[-1] == 12
