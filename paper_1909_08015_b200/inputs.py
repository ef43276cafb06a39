"""Seeded synthetic inputs for the five BASELINE.json configs.

This module holds NO arithmetic of the method: it only lists graphs (x, photons) as plain
integers.  It serves both the CUDA path's tests/bench and the oracle's tests, and imports neither.

A graph: electron path v_0..v_2n, external photon at v_x, n photons = perfect matching of the other
2n vertices.  A graph is admitted when every electron line e_i=(v_{i-1},v_i) is spanned by a photon
(a <= i-1, b >= i): one-particle irreducible, no leg corrections (fn.7 at 155).
"""
import random


def is_valid(n, x, photons):
    nv = 2 * n + 1
    seen = {x}
    for a, b in photons:
        if a == b or a in seen or b in seen or not (0 <= a < nv and 0 <= b < nv):
            return False
        seen.add(a); seen.add(b)
    if len(seen) != nv:
        return False
    for i in range(1, 2 * n + 1):
        if not any(min(a, b) <= i - 1 and max(a, b) >= i for a, b in photons):
            return False
    return True


def _matchings(vs):
    if not vs:
        yield []
        return
    a = vs[0]
    for k in range(1, len(vs)):
        rest = vs[1:k] + vs[k + 1:]
        for m in _matchings(rest):
            yield [(a, vs[k])] + m


def all_graphs(n):
    """All directed n-loop graphs, lexicographic in (x, sorted photons): 1, 6, 50, 518, 6354 for n=1..5."""
    out = []
    nv = 2 * n + 1
    for x in range(nv):
        vs = [v for v in range(nv) if v != x]
        for m in _matchings(vs):
            m = sorted(m)
            if is_valid(n, x, m):
                out.append((x, m))
    return out


def random_graph(n, rng):
    nv = 2 * n + 1
    while True:
        x = rng.randrange(nv)
        vs = [v for v in range(nv) if v != x]
        rng.shuffle(vs)
        m = sorted(tuple(sorted(vs[2 * k:2 * k + 2])) for k in range(n))
        if is_valid(n, x, m):
            return x, m


def config(i):
    """The i-th BASELINE.json config (1-based) as a list of graphs (x, photons) and option dict."""
    if i == 1:
        return dict(graphs=[(1, [(0, 2)])], merge=False, n_samples=10 ** 7, seed=1)
    if i == 2:
        return dict(graphs=all_graphs(2), merge=False, n_samples=10 ** 8, seed=1)
    if i == 3:
        return dict(graphs=all_graphs(3), merge=False, n_samples=10 ** 9, seed=1)
    if i == 4:
        return dict(graphs=[(4, [(0, 8), (1, 7), (2, 6), (3, 5)])], merge=False, n_samples=10 ** 10, seed=1)
    if i == 5:
        rng = random.Random(0x5EED)
        return dict(graphs=[random_graph(5, rng) for _ in range(32)], merge=True, n_samples=10 ** 10, seed=1)
    raise ValueError(i)


def edge_list(x, photons):
    """Canonical edge list for fg_graph_create: electron lines e_1..e_2n then photons sorted by lower end.
    Rows (u, v, kind) with kind 0 = electron, 1 = photon.  The Feynman parameters z follow this order."""
    n = len(photons)
    edges = [(i, i + 1, 0) for i in range(2 * n)]
    edges += [(min(a, b), max(a, b), 1) for a, b in sorted((min(a, b), max(a, b)) for a, b in photons)]
    return edges


def mirror(x, photons):
    n = len(photons)
    return 2 * n - x, sorted((2 * n - b, 2 * n - a) for a, b in ((min(p), max(p)) for p in photons))
