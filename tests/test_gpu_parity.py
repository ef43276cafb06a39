"""Parity of the CUDA path (through the C ABI) with the CPU oracle, element by element on the same seeded inputs.

Bars (BASELINE.json north_star): Philox integers and sector choices bit-exact; per-sample integrand values within
1e-12 relative; means within 1e-10 relative at equal sample sets.  z and pdf are compared to a few ulp (the device
log/pow differ from glibc's in the last bits), and the integrand is compared at the device's
own z so that this difference does not enter.
"""
import math
import os

import numpy as np
import pytest

from oracle import oracle as O
from paper_1909_08015_b200 import inputs

pytestmark = pytest.mark.gpu

G1 = (1, [(0, 2)])
G2 = inputs.all_graphs(2)
G3 = inputs.all_graphs(3)[::9]
G4 = (4, [(0, 8), (1, 7), (2, 6), (3, 5)])
EQ11 = (4, [(0, 10), (1, 9), (2, 3), (5, 7), (6, 8)])


@pytest.fixture(scope="module")
def fg():
    import torch
    assert torch.cuda.is_available()
    from paper_1909_08015_b200 import build, fg as m
    build.build()
    return m


_cache = {}


def pair(fg, x, ph, merge=False, **kw):
    key = (x, tuple(ph), merge, tuple(sorted(kw.items())))
    if key not in _cache:
        _cache[key] = (fg.plan_for(x, ph, merge_ext_lines=merge, **kw), O.Oracle(x, ph, merge=merge, printed=False))
    return _cache[key]


def test_philox_words_bit_exact(fg):
    plan, _ = pair(fg, *G2[1])
    for first, seed in ((0, 1), (2 ** 40 + 12345, 0xDEADBEEF12345678)):
        s = plan.sample_dump(first, 37, seed)
        for i in (0, 1, 17, 36):
            sid = first + i
            for call in range(plan.M):
                want = O.philox([sid & 0xFFFFFFFF, sid >> 32, call, 0], [seed & 0xFFFFFFFF, seed >> 32])
                assert [int(w) for w in s["words"][i, call]] == [int(w) for w in want]


@pytest.mark.parametrize("g,merge", [(G1, False), (G1, True)] + [(g, m) for g in G2 for m in (False, True)] + [(g, False) for g in G3[:3]] + [(G4, False)])
def test_sampler_parity(fg, g, merge):
    plan, orc = pair(fg, g[0], g[1], merge)
    n = 5000 + 37                       # several blocks and a ragged tail
    s = plan.sample_dump(11, n, 3); so = orc.sample(3, 11, n)
    assert np.array_equal(s["comp"], so["comp"])
    assert np.array_equal(s["order"], so["order"])                      # sector choices bit-exact
    assert np.array_equal(s["bad"], so["bad"])
    ok = so["bad"] == 0
    assert np.all(np.abs(s["z"][ok] - so["z"][ok]) <= 1e-13 * so["z"][ok])
    g_dev = s["pdf_mant"] * np.exp2(s["pdf_exp"].astype(np.float64)); g_orc = so["pdf_mant"] * np.exp2(so["pdf_exp"].astype(np.float64))
    assert np.all(np.abs(g_dev[ok] - g_orc[ok]) <= 1e-12 * g_orc[ok])
    assert np.all((s["pdf_mant"] >= 0.5) & (s["pdf_mant"] < 1.0))
    d, Z = plan.tables(); do, Zo = orc.tables()
    assert np.array_equal(d, do) and np.array_equal(Z, Zo)              # tables bit-exact


@pytest.mark.parametrize("g,merge", [(G1, False), (G1, True)] + [(g, m) for g in G2 for m in (False, True)] + [(g, False) for g in G3] + [(G3[1], True), (G4, False), (G4, True)])
def test_integrand_parity_per_sample(fg, g, merge):
    """flags: bit0 = re-evaluated in double-double, bit1 = non-finite / degenerate point, bit2 = not resolved by the
    last rung (contributes 0).  Unresolved points are the ones whose cancellation exceeds 106 bits; the
    oracle's own __float128 value is not reliable there either, so they are excluded and must be few."""
    plan, orc = pair(fg, g[0], g[1], merge)
    n = 3000 + 129
    z = plan.sample_dump(0, n, 1, words=False)["z"]
    Id, Iq, fl = orc.eval(z, rel_tol=1e-12)
    fin = np.isfinite(Iq) & (Iq != 0)
    # every point in double-double
    e2 = plan.eval_points(z, mode=2)
    ok2 = fin & ((e2["flags"] & 6) == 0)
    assert np.all(np.abs(e2["I"][ok2] - Iq[ok2]) <= 1e-12 * np.abs(Iq[ok2]))
    assert (~ok2 & fin).mean() < 0.08
    # as the integrator does it: double, conditioning check, flagged points redone in double-double
    e0 = plan.eval_points(z, mode=0)
    ok0 = fin & ((e0["flags"] & 6) == 0)
    assert np.array_equal(ok0, ok2)
    assert np.all(np.abs(e0["I"][ok0] - Iq[ok0]) <= 1e-12 * np.abs(Iq[ok0]))
    # the running error estimate bounds the actual error of the plain double pass ...
    e1 = plan.eval_points(z, mode=1)
    act = np.abs(e1["I_double"] - Iq)
    assert np.all(act[ok0] <= np.maximum(e0["err"][ok0], 1e-12 * np.abs(Iq[ok0])))
    # ... so the device flags a superset of what the oracle flags as unstable in double
    unstable = ok0 & ((fl & 1) == 1) & (act > 1e-12 * np.abs(Iq))
    assert np.all((e0["flags"][unstable] & 1) == 1)


def test_one_loop_closed_form(fg):
    plan, _ = pair(fg, *G1)
    z = np.random.default_rng(0).dirichlet(np.ones(3), 1000)
    e = plan.eval_points(z, mode=1)
    assert np.allclose(e["I"], z[:, 2] / (1 - z[:, 2]), rtol=1e-13)


@pytest.mark.parametrize("g,merge,n", [(G1, False, 200000), (G2[3], False, 100000), (G2[1], True, 100000), (G3[2], False, 20000), (G4, False, 4000)])
def test_means_at_equal_sample_sets(fg, g, merge, n):
    """Mean, variance and counters of fg_integrate against the oracle on the same samples.  The oracle's integrand is
    taken at the device's z (which differ from the oracle's own z in the last bits), its pdf from its own sampler; the
    sample set is the accepted one (the device's unresolved / degenerate samples contribute 0 on both sides)."""
    plan, orc = pair(fg, g[0], g[1], merge)
    first, seed = 5, 9
    r = plan.integrate_range(first, n, seed)
    d = plan.sample_eval_dump(first, n, seed); s = plan.sample_dump(first, n, seed, words=False); so = orc.sample(seed, first, n)
    Iq = orc.eval(s["z"])[1]
    gq = so["pdf_mant"] * np.exp2(so["pdf_exp"].astype(np.float64))
    acc = (d["flags"] & 6) == 0
    y_ref = np.where(acc, Iq / gq, 0.0)
    assert r["n_samples"] == n and r["n_rejected"] == int((~acc).sum()) and (~acc).mean() < 0.08
    assert r["n_pdf_big_exp"] == int(((so["pdf_exp"] > 1023) | (so["pdf_exp"] < -1021)).sum())
    assert r["n_flagged"] == int((d["flags"] & 1).sum())
    assert np.all(np.abs(d["y"] - y_ref) <= 2e-12 * np.abs(y_ref))
    sy = math.fsum(y_ref); sy2 = math.fsum(y_ref ** 2)
    assert abs(r["sum_y"][0] - sy) <= 1e-10 * abs(sy)
    assert abs(r["mean"] - sy / n) <= 1e-10 * abs(sy / n)
    var = sy2 / n ** 2 - sy ** 2 / n ** 3
    assert abs(r["variance"] - var) <= 1e-9 * var
    if acc.all():                       # then the oracle's own estimator (its own z) must agree too
        ro = orc.integrate(seed, first, n, quad=True)
        assert abs(r["mean"] - ro["mean"]) <= 1e-9 * abs(ro["mean"]) + 1e-10 * np.abs(y_ref).mean()


def test_one_loop_value_and_two_loop_sum(fg):
    plan, _ = pair(fg, *G1)
    r = plan.integrate(10 ** 7, 1)                  # config 1 at full size
    assert abs(r["mean"] - 0.5) < 4 * math.sqrt(r["variance"]) and math.sqrt(r["variance"]) < 5e-4
    tot = var = 0.0
    for x, ph in G2:
        r = pair(fg, x, ph)[0].integrate(4 * 10 ** 6, 1)
        tot += r["mean"]; var += r["variance"]
    target = -0.328478965579 - (119.0 / 36.0 - math.pi ** 2 / 3.0)
    assert abs(tot - target) < 4 * math.sqrt(var) and math.sqrt(var) < 0.01


def test_config2_full_size_two_loop_sum(fg):           # BASELINE.json config 2: 1e8 samples per graph
    """Sum of the six 2-loop graphs without lepton loops = A1^(4) - (119/36 - pi^2/3) (PAPER.md:28 and north_star)."""
    tot = var = 0.0; rej = 0
    for x, ph in G2:
        plan = fg.plan_for(x, ph, rel_tol=1e-9)
        r = plan.integrate(10 ** 8, 1)
        tot += r["mean"]; var += r["variance"]; rej += r["n_rejected"]
    target = -0.328478965579 - (119.0 / 36.0 - math.pi ** 2 / 3.0)
    assert math.sqrt(var) < 2.5e-3
    assert abs(tot - target) < 4 * math.sqrt(var), (tot, target, math.sqrt(var))
    assert rej < 6e8 * 1e-3


def test_ranges_shard_and_merge_exactly(fg):       # sharding by sample-id range
    plan, _ = pair(fg, *G2[2])
    whole = plan.integrate_range(100, 70001, 4, raw=True)
    a = plan.integrate_range(100, 30000, 4, raw=True); b = plan.integrate_range(30100, 40001, 4, raw=True)
    m = fg.result_merge(a, b)
    assert m.n_samples == whole.n_samples and m.n_flagged == whole.n_flagged
    assert abs(m.sum_y[0] - whole.sum_y[0]) <= 1e-25 * abs(whole.sum_y[0]) + abs(whole.sum_y[1]) * 1e-9
    assert abs(m.mean - whole.mean) <= 1e-15 * abs(whole.mean)
    again = plan.integrate_range(100, 70001, 4, raw=True)             # deterministic
    assert again.sum_y[0] == whole.sum_y[0] and again.sum_y2[0] == whole.sum_y2[0]


def test_more_than_one_slab(fg):                   # the integrator works in slabs of 2^24 samples
    plan, _ = pair(fg, *G1)
    n = (1 << 24) + 12345
    whole = plan.integrate_range(7, n, 3, raw=True)
    a = plan.integrate_range(7, 1 << 24, 3, raw=True); b = plan.integrate_range(7 + (1 << 24), 12345, 3, raw=True)
    m = fg.result_merge(a, b)
    assert whole.n_samples == n == m.n_samples and whole.n_flagged == m.n_flagged and whole.n_rejected == m.n_rejected
    assert abs(whole.sum_y[0] - m.sum_y[0]) <= 1e-14 * abs(m.sum_y[0]) and abs(whole.sum_y2[0] - m.sum_y2[0]) <= 1e-14 * m.sum_y2[0]
    assert abs(whole.mean - 0.5) < 5 * math.sqrt(whole.variance)


@pytest.mark.parametrize("n", [1, 2, 255, 256, 257, 4097])
def test_ragged_sizes(fg, n):
    plan, orc = pair(fg, *G2[0])
    r = plan.integrate_range(0, n, 2)
    d = plan.sample_eval_dump(0, n, 2); s = plan.sample_dump(0, n, 2, words=False); so = orc.sample(2, 0, n)
    acc = (d["flags"] & 6) == 0
    y_ref = np.where(acc, orc.eval(s["z"])[1] / (so["pdf_mant"] * np.exp2(so["pdf_exp"].astype(np.float64))), 0.0)
    assert r["n_samples"] == n
    assert abs(r["sum_y"][0] - math.fsum(y_ref)) <= 1e-10 * np.abs(y_ref).sum() + 1e-300


def test_empty_and_bad_arguments(fg):
    plan, _ = pair(fg, *G1)
    with pytest.raises(fg.FgError):
        plan.integrate(0, 1)
    assert plan.sample_dump(0, 0, 1, words=False)["z"].shape == (0, 3)
    with pytest.raises(fg.FgError):
        fg.plan_for(1, [(0, 2)], C4=[0.5, 0.5, 0.5, 0.5])


def test_structure_matches_expression_11(fg):
    x, ph = EQ11
    plan = fg.plan_for(x, ph, merge_ext_lines=True)
    subs, terms = plan.structure()
    assert sorted((s["a"], s["b"]) for s in subs) == [(0, 10), (1, 9), (2, 3), (5, 7), (5, 8), (6, 8)]
    assert plan.stats["n_forests"] == 24 and plan.stats["n_terms"] == 36 and plan.M == 14
    o = O.Oracle(x, ph, structure_only=True)
    osubs = o.subs()
    key = lambda ss, t: (t["sign"], tuple(sorted(((ss[m]["a"], ss[m]["b"]), op) for m, op in t["members"])))
    assert set(key(subs, t) for t in terms) == set(key(osubs, t) for t in o.terms())
    # degenerate density: uniform component only
    z = plan.sample_dump(0, 2000, 5, words=False)
    assert np.allclose(z["z"].sum(axis=1), 1.0, atol=1e-14) and not z["bad"].any()


def test_config3_all_fifty_three_loop_graphs(fg):       # BASELINE.json config 3: every graph, double-double fallback on
    worst = 0.0; unresolved = 0; total = 0
    for x, ph in inputs.all_graphs(3):
        plan = fg.plan_for(x, ph, rel_tol=1e-12); orc = O.Oracle(x, ph, printed=False)
        z = plan.sample_dump(0, 600, 3, words=False)["z"]
        Iq = orc.eval(z)[1]; e0 = plan.eval_points(z, mode=0)
        ok = np.isfinite(Iq) & (Iq != 0) & ((e0["flags"] & 6) == 0)
        worst = max(worst, float(np.max(np.abs(e0["I"][ok] - Iq[ok]) / np.abs(Iq[ok]))))
        unresolved += int((~ok).sum()); total += len(z)
    assert worst <= 1e-12 and unresolved < 0.03 * total


def test_config4_ladder_prefix_per_sample(fg):          # BASELINE.json config 4: per-sample agreement on a prefix
    plan, orc = pair(fg, *G4)
    n = 32768
    d = plan.sample_eval_dump(0, n, 1); s = plan.sample_dump(0, n, 1, words=False); so = orc.sample(1, 0, n)
    assert np.array_equal(s["order"], so["order"]) and np.array_equal(s["comp"], so["comp"])
    Iq = orc.eval(s["z"])[1]
    ok = np.isfinite(Iq) & (Iq != 0) & ((d["flags"] & 6) == 0)
    assert ok.mean() > 0.9
    assert np.all(np.abs(d["I"][ok] - Iq[ok]) <= 1e-12 * np.abs(Iq[ok]))
    gq = so["pdf_mant"] * np.exp2(so["pdf_exp"].astype(np.float64))
    assert np.all(np.abs(d["y"][ok] - Iq[ok] / gq[ok]) <= 2e-12 * np.abs(Iq[ok] / gq[ok]))


@pytest.mark.skipif((os.cpu_count() or 1) < 16 and not os.environ.get("FG_TEST_5LOOP"), reason="oracle tables of a 5-loop graph take ~5 min on 8 cores")
def test_five_loop_sampled_outputs(fg):            # config 5 in the launch configuration bench.py times
    cfg = inputs.config(5); x, ph = cfg["graphs"][0]
    plan = fg.plan_for(x, ph, merge_ext_lines=True)
    orc = O.Oracle(x, ph, merge=True, printed=False)
    z = plan.sample_dump(0, 4096, 1, words=False)["z"][::16]
    Id, Iq, fl = orc.eval(z)
    e0 = plan.eval_points(z, mode=0)
    ok = np.isfinite(Iq) & (Iq != 0) & ((e0["flags"] & 6) == 0)
    assert ok.mean() > 0.9
    assert np.all(np.abs(e0["I"][ok] - Iq[ok]) <= 1e-12 * np.abs(Iq[ok]))
    e1 = plan.eval_points(z, mode=1)
    assert np.all(np.abs(e1["I_double"] - Iq)[ok] <= np.maximum(e0["err"][ok], 1e-12 * np.abs(Iq[ok])))


@pytest.mark.gpu
def test_double_double_pass_same_values_at_every_queue_length(fg):
    """The double-double pass deals the records of a point out to groups of w = 2..32 lanes, w chosen from the queue
    length.  The value of a point must not depend on that choice: the same 300 points are evaluated in
    queues of growing length (w = 32 ... 2, then one point per thread, then several rounds) and compared with the
    oracle's __float128 and with each other."""
    g = G3[2]
    plan, orc = pair(fg, g[0], g[1], False)
    zb = plan.sample_dump(0, 300, 7, words=False)["z"]
    _, Iq, _ = orc.eval(zb, rel_tol=1e-12)
    ref = None
    for reps in (1, 10, 24, 47, 95, 200, 420):
        z = np.ascontiguousarray(np.tile(zb, (reps, 1)))
        e = plan.eval_points(z, mode=2)
        I = e["I"].reshape(reps, 300); fl = e["flags"].reshape(reps, 300)
        res = (fl & 6) == 0                       # resolved; a point at the edge of the tolerance may flip with the summation order
        assert (res != res[0]).mean() < 0.01
        ok = np.isfinite(Iq) & (Iq != 0) & res.all(axis=0)
        assert ok.mean() > 0.9
        assert np.all(np.abs(I[:, ok] - Iq[ok]) <= 1e-12 * np.abs(Iq[ok]))
        if ref is None:
            ref = (I[0], ok)
        both = ok & ref[1]
        assert np.all(np.abs(I[:, both] - ref[0][both]) <= 1e-14 * np.abs(ref[0][both]))
