"""Host logic of the multi-graph scheduler (fg_batch_*: PAPER.md:286, 290-294, 328-359) without a GPU: synthetic block
results are folded in, and the schedule, the acceptance tolerances (18) and the combination (19) are compared with the plain
restatement in oracle/sched_oracle.py; then two ranks run one schedule over gloo and must end in the same state."""
import ctypes as C
import math
import os
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


class FakePlan:
    """A batch only stores its plan handles; next / fold / probabilities never touch them."""
    def __init__(self, k):
        self.h = C.c_void_p(0x1000 + 16 * k)


def block_result(fg, rng, mean, sd, n):
    y = rng.normal(mean, sd, n)
    r = fg.fg_result(); sy = float(np.sum(y)); sy2 = float(np.sum(y * y))
    r.sum_y[0] = sy; r.sum_y2[0] = sy2; r.n_samples = n
    r.mean = sy / n; r.variance = sy2 / n ** 2 - sy ** 2 / n ** 3
    return r


def test_schedule_tolerances_and_combination_follow_the_paper(fg):
    from oracle import sched_oracle as SO
    from paper_1909_08015_b200 import sched
    rng = np.random.default_rng(7)
    means = [0.8, -0.5, 0.03, -0.3, 1.7]; sds = [3.0, 0.4, 9.0, 1.0, 0.05]; times = [1e-6, 4e-6, 2e-7, 1e-6, 3e-5]
    b = sched.Batch([FakePlan(k) for k in range(5)])
    assert np.allclose(b.probabilities(), 0.2)                 # nothing known: uniform
    sy = [0.0] * 5; sy2 = [0.0] * 5; nn = [0] * 5
    for j in range(5):                                         # "initialisation stage": one block per graph
        r = block_result(fg, rng, means[j], sds[j], 4000)
        b.fold(j, r, times[j] * 4000)
        sy[j] += r.sum_y[0]; sy2[j] += r.sum_y2[0]; nn[j] += 4000
    b.set_times(times)
    seed = 0xC0FFEE; counts = [0] * 5; firsts = [0] * 5
    for k in range(400):
        p = SO.probabilities(sy, sy2, nn, times)
        assert np.allclose(b.probabilities(), p, rtol=1e-12)
        j, first = b.next(seed, 1000)
        assert j == SO.pick(p, seed, k) and first == firsts[j]
        firsts[j] += 1000; counts[j] += 1
        r = block_result(fg, rng, means[j], sds[j], 1000)
        b.fold(j, r, 0.0)
        sy[j] += r.sum_y[0]; sy2[j] += r.sum_y2[0]; nn[j] += 1000
        if k % 50 == 0:
            tol = SO.abs_tol_18(sy, sy2, nn)
            assert np.allclose(b.abs_tol, tol, rtol=1e-9)
    # graphs with large C_j / sqrt(t_j) get the blocks: sd 9 at 2e-7 s dominates, sd 0.05 at 3e-5 s gets (almost) none
    assert counts[2] > 250 and counts[4] <= 2 and sum(counts) == 400
    tot = b.total()
    assert tot["n_samples"] == sum(nn)
    assert abs(tot["value"] - sum(a / m for a, m in zip(sy, nn))) < 1e-12
    assert abs(tot["sigma_down"] - SO.combine_19([SO.sigma_down(a, c, m) ** 2 for a, c, m in zip(sy, sy2, nn)])) < 1e-12 * tot["sigma_down"]


def test_optimal_allocation_beats_uniform(fg):
    """The rule minimises sigma^2 t: with the p_j of the paper the predicted variance at equal total time
    is not larger than with a uniform split."""
    from oracle import sched_oracle as SO
    C_ = np.array([3.0, 0.4, 9.0, 1.0, 0.05]); t = np.array([1e-6, 4e-6, 2e-7, 1e-6, 3e-5])
    p = np.array(SO.probabilities([0] * 5, list(C_ ** 2 * 100), [100] * 5, list(t)))      # sum_y = 0, sum_y2 = C^2 N
    cost = lambda q: (C_ ** 2 / q).sum() * (q * t).sum()
    assert cost(p) <= cost(np.full(5, 0.2)) * (1 + 1e-12)
    for _ in range(100):
        q = np.random.default_rng(_).dirichlet(np.ones(5))
        assert cost(p) <= cost(q) * (1 + 1e-12)


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, q):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_1909_08015_b200 import fg, sched
    from paper_1909_08015_b200.dist import run_batch_rounds
    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    means = [0.8, -0.5, 0.03]; sds = [3.0, 0.4, 9.0]
    b = sched.Batch([FakePlan(k) for k in range(3)])
    for j in range(3):
        b.fold(j, block_result(fg, np.random.default_rng(100 + j), means[j], sds[j], 2000), 0.0)
    b.set_times([1e-6, 2e-6, 5e-7])

    def integrate(j, first, n):          # stands in for plan.integrate_range on this rank's GPU: depends on (graph, range) only
        return block_result(fg, np.random.default_rng(first * 7 + j), means[j], sds[j], n), 0.0
    log = run_batch_rounds(b, 25, 500, 11, rank, world, integrate)
    tot = b.total()
    q.put((rank, tuple(log), tot["value"], tot["sigma_down"], tot["n_samples"], tuple(b.probabilities())))
    dist.barrier(); dist.destroy_process_group()


def test_two_ranks_run_one_schedule_over_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn"); q = ctx.Queue(); port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    got = sorted(q.get(timeout=180) for _ in ps)
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    a, b = got
    assert a[1:] == b[1:]                                   # same schedule, same sums, same probabilities on both ranks
    assert len(a[1]) == 50 and a[4] == 3 * 2000 + 50 * 500   # 25 rounds x 2 ranks
    # ranges of one graph never overlap
    seen = {}
    for j, first in a[1]:
        assert first == seen.get(j, 0); seen[j] = first + 500
