"""Pins of the host combinatorics of BOTH sides (the oracle and the product's planner) against definitions that neither
of them implements:

* UV-divergent subgraphs by the paper's own definition (PAPER.md:139 and fn.7 at 155): every set of vertices whose induced
  subgraph is connected, one-particle irreducible, and has N_e = 2 external electron lines and N_gamma = 0 or 1 external
  photon lines -- by brute force over all vertex subsets -- against the interval rule R-sub of DESIGN.md;
* Dirac coefficient tables at 4 and 5 loops against explicit 4x4 gamma matrices with explicit sums over every Lorentz
  index: the oracle's table engine AND the planner's (fg_host_dirac_table), pattern by pattern.
"""
import itertools
import random
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

from conftest import read_facts
from oracle import oracle as O
from paper_1909_08015_b200 import inputs

FACTS = read_facts()
EQ11 = (int(FACTS["eq11_x"][0]), [tuple(int(t) for t in s.split("-")) for s in FACTS["eq11_photons"]])
LADDER4 = (4, [(0, 8), (1, 7), (2, 6), (3, 5)])


@pytest.fixture(scope="module")
def fg():
    from paper_1909_08015_b200 import build, fg as m
    build.build()
    return m


# ------------------------------------------------------------------------------------------------ subgraphs
def brute_force_divergent_subgraphs(n, x, photons):
    """All UV-divergent subgraphs of the graph by the definition of PAPER.md:139 / fn.7, as (sorted vertex tuple, type).
    Lines: electron lines (i, i+1), i = 0..2n-1; photons; external lines: the incoming electron at v_0, the outgoing one at
    v_2n, the external photon at v_x.  A subgraph is the set of ALL lines that join a vertex set (fn.7)."""
    nv = 2 * n + 1
    lines = [("e", i, i + 1) for i in range(2 * n)] + [("p", min(a, b), max(a, b)) for a, b in photons]
    out = []
    for size in range(2, nv + 1):
        for vs in itertools.combinations(range(nv), size):
            vset = set(vs)
            inner = [l for l in lines if l[1] in vset and l[2] in vset]
            if not any(l[0] == "p" for l in inner):
                continue                                   # no loop, no divergence

            def connected(ls):
                adj = {v: set() for v in vset}
                for _, a, b in ls:
                    adj[a].add(b); adj[b].add(a)
                seen = {vs[0]}; stack = [vs[0]]
                while stack:
                    v = stack.pop()
                    for w in adj[v]:
                        if w not in seen:
                            seen.add(w); stack.append(w)
                return len(seen) == len(vset)
            if not connected(inner):
                continue
            if not all(connected(inner[:k] + inner[k + 1:]) for k in range(len(inner))):
                continue                                   # "strongly connected": stays connected when any one line is cut
            n_e = sum(1 for l in lines if l[0] == "e" and ((l[1] in vset) != (l[2] in vset)))
            n_e += (0 in vset) + (2 * n in vset)            # the external electron lines of G
            n_g = sum(1 for l in lines if l[0] == "p" and ((l[1] in vset) != (l[2] in vset))) + (x in vset)
            if n_e == 2 and n_g in (0, 1):
                out.append((vs, "V" if n_g == 1 else "SE"))
    return sorted(out)


def _interval_subs(subs):
    return sorted((tuple(range(s["a"], s["b"] + 1)), s["type"]) for s in subs)


@pytest.mark.parametrize("n,step", [(1, 1), (2, 1), (3, 1), (4, 7), (5, 211)])
def test_divergent_subgraphs_by_the_papers_definition(fg, n, step):
    graphs = inputs.all_graphs(n)[::step] if n < 5 else O.enumerate_graphs(5)[::step]
    if n == 5:
        graphs = graphs + [EQ11] + inputs.config(5)["graphs"][:4]
    for x, ph in graphs:
        want = brute_force_divergent_subgraphs(n, x, ph)
        o = O.Oracle(x, ph, structure_only=True)
        assert _interval_subs(o.subs()) == want, (x, ph)
        g = fg.Graph(inputs.edge_list(x, ph), x)
        _, subs, _ = fg.host_plan(g, structure_only=True)
        assert _interval_subs(subs) == want, (x, ph)
        assert sorted(tuple(range(s["a"], s["b"] + 1)) for s in subs if s["in_chain"]) == sorted(v for v, t in want if t == "V" and x in v)
        # chain I[G]: the vertexlike subgraphs that contain v_x
        assert sorted(tuple(range(s["a"], s["b"] + 1)) for s in o.subs() if s["in_chain"]) == sorted(v for v, t in want if t == "V" and x in v)


# ------------------------------------------------------------------------------------------------ Dirac tables
def _sample_patterns(rng, nslots, with_q, count):
    """Random (pairs, qslot, T) patterns of an element with nslots slots: all numbers of pairs, q-slot patterns included."""
    pats = []
    for k in range(count):
        npairs = rng.randrange(0, nslots // 2 + 1) if k % 3 else nslots // 2 - (k // 3) % 2
        npairs = max(0, min(npairs, nslots // 2))
        sl = list(range(nslots)); rng.shuffle(sl)
        pairs = sorted(tuple(sorted(sl[2 * i:2 * i + 2])) for i in range(npairs))
        un = sorted(sl[2 * npairs:])
        q = -1
        if with_q and un and k % 2:
            q = rng.choice(un)
        gaps = [s for s in un if s != q]
        T = rng.randrange(0, 1 << len(gaps)) if gaps else 0
        pats.append((pairs, q, gaps, T))
    return pats


def _dirac_cases():
    g17 = inputs.config(5)["graphs"][17]
    return [("4-loop ladder", LADDER4), ("expression (11) graph", EQ11), ("config-5 graph 17", g17)]


@pytest.mark.parametrize("name,graph", _dirac_cases(), ids=[c[0] for c in _dirac_cases()])
def test_dirac_tables_of_oracle_and_planner_vs_explicit_matrices(fg, name, graph):
    x, ph = graph
    o = O.Oracle(x, ph, printed=False, structure_only=2)
    g = fg.Graph(inputs.edge_list(x, ph), x)
    rng = random.Random(20190908)
    jobs = []
    for gi in range(o.n_geoms):
        d = o.geom_desc(gi)
        if d["type"] == 0:
            ops = [(1, 0), (1, 1)]                                   # self-energy element: U, components u and v
        else:
            ops = [(1, 0), (2, 0)]                                   # U, L
            if d["a"] <= x <= d["b"]:
                ops.append((0, 0))                                   # A on a member of the chain I[G]
            if d["a"] == 0 and d["b"] == 2 * len(ph):
                ops.append((3, 0))                                   # (L - U) on G
        for op, comp in ops:
            for pairs, q, gaps, T in _sample_patterns(rng, d["nslots"], op == 0, 20):
                jobs.append((gi, d, op, comp, pairs, q, gaps, T))
    assert len(jobs) >= 20 * 4

    def run(job):
        gi, d, op, comp, pairs, q, gaps, T = job
        tmask = sum(1 << gaps[k] for k in range(len(gaps)) if (T >> k) & 1)
        want = o.dirac_explicit(gi, op, comp, pairs, q, tmask)                       # explicit matrices
        ogaps, otab = o.dirac_table(gi, op, comp, pairs, q)                          # the oracle's table engine
        ns, pgaps, ptab = fg.host_dirac_table(g, d["a"], d["b"], d["children"], op, comp, pairs, q)    # the planner's
        assert ogaps == gaps and pgaps == gaps and ns == d["nslots"]
        return want, otab[T], ptab[T] / (-0.5) ** len(pairs)

    with ThreadPoolExecutor(8) as ex:
        res = list(ex.map(run, jobs))
    res = np.array(res)
    assert np.abs(res[:, 0]).max() > 1.0                              # the sample is not all zeros
    assert (res[:, 0] != 0).sum() > len(res) // 10
    assert np.abs(res[:, 1] - res[:, 0]).max() < 1e-9, "oracle table vs explicit matrices"
    assert np.abs(res[:, 2] - res[:, 0]).max() < 1e-9, "planner table vs explicit matrices"
