"""Second random-number stream, MRG32k3a (Calc 1 of the paper).  CPU part: the oracle's generator
against the published self-check of the reference implementation, its jump against plain stepping, and the sampler's
normalisation under this stream.  GPU part: the CUDA stream (precomputed jump table, 64-bit constant-modulus arithmetic)
against the oracle's (matrix power per sample in 128-bit arithmetic): raw integers, sectors and components bit-exact,
coordinates, pdf and means to the tolerances of test_gpu_parity.py."""
import math

import numpy as np
import pytest

from conftest import golden
from oracle import oracle as O
from paper_1909_08015_b200 import inputs

G1 = (1, [(0, 2)])
G2 = inputs.all_graphs(2)
G4 = (4, [(0, 8), (1, 7), (2, 6), (3, 5)])


def kat():
    with open(golden("mrg32k3a_kat.txt")) as f:
        return {l.split()[0]: l.split()[1] for l in f if l.strip() and not l.startswith("#")}


def test_reference_implementation_self_check():
    u = O.mrg32k3a(0, 0, 10 ** 7)            # seed 0 = 12345 for all six components
    assert "%.2f" % float(np.sum(u)) == kat()["sum_first_1e7"]
    assert u.min() > 0.0 and u.max() < 1.0


def test_jump_equals_stepping():
    for seed, first in ((0, 0), (0, 977), (0x1234567812345678, 10 ** 12 + 5), (0xFFFFFFFFFFFFFFFF, 32 * (2 ** 40 + 12345))):
        a = O.mrg32k3a(seed, first, 300); b = O.mrg32k3a(seed, first, 300, by_jump=True)
        assert np.array_equal(a, b)
    long = O.mrg32k3a(7, 0, 5000)
    assert np.array_equal(long[4000:4100], O.mrg32k3a(7, 4000, 100))


def test_density_integrates_to_one_under_the_second_stream():      # E_g[(M-1)!/g] = 1
    x, ph = G2[1]
    o = O.Oracle(x, ph, structure_only=2); o.set_rng(1)
    s = o.sample(3, 0, 200000)
    g = s["pdf_mant"] * np.exp2(s["pdf_exp"].astype(np.float64))
    w = math.factorial(o.M - 1) / g
    assert abs(w.mean() - 1.0) < 5.0 * w.std() / math.sqrt(len(w))
    o0 = O.Oracle(x, ph, structure_only=2)
    assert not np.array_equal(o0.sample(3, 0, 64)["order"], s["order"][:64])      # really another stream


# ------------------------------------------------------------------------------------------------ GPU
@pytest.fixture(scope="module")
def fg():
    import torch
    assert torch.cuda.is_available()
    from paper_1909_08015_b200 import build, fg as m
    build.build()
    return m


@pytest.mark.gpu
def test_raw_integers_bit_exact(fg):
    plan = fg.plan_for(*G2[1], rng=1)
    M = plan.M; norm = 2.328306549295727688e-10
    for first, seed in ((0, 0), (5, 1), (2 ** 40 + 12345, 0xDEADBEEF12345678)):
        s = plan.sample_dump(first, 37, seed)
        for i in (0, 1, 17, 36):
            want = O.mrg32k3a(seed, 32 * (first + i), 4 * M)
            got = s["words"][i].reshape(-1).astype(np.float64) * norm
            assert np.array_equal(got, want)


@pytest.mark.gpu
@pytest.mark.parametrize("g,merge", [(G1, False), (G2[3], False), (G2[1], True), (G4, False), (inputs.config(5)["graphs"][0], True)])
def test_sampler_parity_under_the_second_stream(fg, g, merge):
    plan = fg.plan_for(g[0], g[1], merge_ext_lines=merge, rng=1)
    orc = O.Oracle(g[0], g[1], merge=merge, structure_only=2); orc.set_rng(1)
    n = 5000 + 37
    for first, seed in ((11, 3), (2 ** 33 + 7, 0xABCDEF0123456789)):
        s = plan.sample_dump(first, n, seed, words=False); so = orc.sample(seed, first, n)
        assert np.array_equal(s["comp"], so["comp"]) and np.array_equal(s["order"], so["order"]) and np.array_equal(s["bad"], so["bad"])
        ok = so["bad"] == 0
        assert np.all(np.abs(s["z"][ok] - so["z"][ok]) <= 1e-13 * so["z"][ok])
        g_dev = s["pdf_mant"] * np.exp2(s["pdf_exp"].astype(np.float64)); g_orc = so["pdf_mant"] * np.exp2(so["pdf_exp"].astype(np.float64))
        assert np.all(np.abs(g_dev[ok] - g_orc[ok]) <= 1e-12 * g_orc[ok])


@pytest.mark.gpu
def test_values_under_the_second_stream(fg):
    p1 = fg.plan_for(*G1, rng=1)
    r = p1.integrate(10 ** 6, 1)
    assert abs(r["mean"] - 0.5) < 4.0 * math.sqrt(r["variance"])                     # A1^(2) = 1/2
    r0 = fg.plan_for(*G1).integrate(10 ** 6, 1)
    assert r0["mean"] != r["mean"]
    # means at equal sample sets against the oracle's own estimator (2-loop ladder)
    x, ph = G2[3]
    plan = fg.plan_for(x, ph, rng=1, rel_tol=1e-12); orc = O.Oracle(x, ph, printed=False); orc.set_rng(1)
    n = 50000
    r = plan.integrate_range(5, n, 9)
    ro = orc.integrate(9, 5, n, wide=True)
    assert r["n_rejected"] == 0 and ro["n_rejected"] == 0
    assert abs(r["mean"] - ro["mean"]) <= 1e-9 * abs(ro["mean"])
    assert abs(r["variance"] - ro["variance"]) <= 1e-8 * ro["variance"]
