"""GPU tests of what sits on top of the single-graph path: sharding by sample-id range and the
multi-graph scheduler with its initialisation stage, acceptance rule (18) and combination (19)."""
import math
from fractions import Fraction as F

import numpy as np
import pytest

from paper_1909_08015_b200 import inputs

pytestmark = pytest.mark.gpu
G2 = inputs.all_graphs(2)
TARGET_2LOOP = -0.328478965579 - (119.0 / 36.0 - math.pi ** 2 / 3.0)      # PAPER.md:28 minus the closed-form VP-insertion graph


@pytest.fixture(scope="module")
def fg():
    import torch
    assert torch.cuda.is_available()
    from paper_1909_08015_b200 import build, fg as m
    build.build()
    return m


def _exact(r, field):
    v = getattr(r, field)
    return F(v[0]) + F(v[1])


@pytest.mark.parametrize("world", [2, 3, 8])
def test_shards_merge_to_the_single_range_result(fg, world):
    """dist.integrate_sharded's split and merge, the shards run one after another on this device: counters identical, sums
    identical to the last bits of the double-double (the grouping of the additions differs, nothing else)."""
    from paper_1909_08015_b200 import dist
    x, ph = G2[2]
    plan = fg.plan_for(x, ph)
    n, first, seed = 70001, 100, 4
    whole = plan.integrate_range(first, n, seed, raw=True)
    m = dist.integrate_shards_on_one_device(plan, n, seed, world, first_sample=first)
    assert (m.n_samples, m.n_flagged, m.n_flagged2, m.n_rejected, m.n_pdf_big_exp) == (whole.n_samples, whole.n_flagged, whole.n_flagged2, whole.n_rejected, whole.n_pdf_big_exp)
    for field in ("sum_y", "sum_y2"):
        a, b = _exact(m, field), _exact(whole, field)
        assert abs(a - b) <= abs(b) * F(1, 10 ** 27)
    assert m.sum_y[0] == whole.sum_y[0] and m.sum_y2[0] == whole.sum_y2[0]
    assert abs(m.mean - whole.mean) <= 1e-15 * abs(whole.mean) and abs(m.variance - whole.variance) <= 1e-14 * whole.variance
    # the blocking multi-rank entry point with world = 1 is the plain call
    one = dist.integrate_sharded(plan, n, seed, 0, 1, first_sample=first)
    assert one.sum_y[0] == whole.sum_y[0] and one.sum_y[1] == whole.sum_y[1]


def test_scheduler_reaches_the_two_loop_value_with_fewer_samples(fg):
    """The six 2-loop graphs as one batch: pilot stage, then blocks drawn with p_j ~ C_j / sqrt(t_j).  The combined error (19)
    falls below what the uniform split of test_config2_full_size_two_loop_sum reaches with 6e8 samples (2.5e-3 asserted
    there) on fewer samples, and the sum is A1^(4) minus the VP-insertion graph within 4 sigma."""
    from paper_1909_08015_b200 import sched
    plans = [fg.plan_for(x, ph, rel_tol=1e-9) for x, ph in G2]
    b = sched.Batch(plans)
    b.pilot(1 << 20, 1, first_sample=0, target_samples=0.0, rel_tol=1e-9)
    p0 = b.probabilities()
    assert abs(p0.sum() - 1.0) < 1e-12 and p0.min() > 0
    tols = b.abs_tol
    assert all(t > 0 for t in tols)
    # (18): the tolerances are proportional to the sigmas of the graphs
    sig = np.array([math.sqrt(b.result(j)["variance"]) for j in range(6)])
    assert np.allclose(np.array(tols) / sig, 0.25 * math.sqrt((sig ** 2).sum()) / sig.sum(), rtol=1e-9)
    uniform_total = 6 * 10 ** 8
    while b.total()["sigma_down"] >= 2.5e-3 and b.total()["n_samples"] < uniform_total:
        b.run(8, 1 << 22, 1, 77)
    tot = b.total()
    print("scheduler: value %.6f +- %.6f (target %.6f) after %.3e samples; per graph N = %s" % (
        tot["value"], tot["sigma_down"], TARGET_2LOOP, tot["n_samples"], [b.result(j)["n_samples"] for j in range(6)]))
    assert tot["sigma_down"] < 2.5e-3 and tot["n_samples"] < 0.9 * uniform_total
    assert abs(tot["value"] - TARGET_2LOOP) < 4 * tot["sigma_down"]
    assert sum(b.result(j)["n_rejected"] for j in range(6)) < 1e-5 * tot["n_samples"]
    # sample ranges of a graph are handed out once: its running n_samples equals pilot + blocks * block size
    for j in range(6):
        assert (b.result(j)["n_samples"] - (1 << 20)) % (1 << 22) == 0
