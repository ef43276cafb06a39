"""Plain restatement of the paper's block-scheduling and acceptance rules, TEST INFRASTRUCTURE
ONLY (imported by tests/; the product's scheduler is paper_1909_08015_b200/csrc/fg_batch.cpp and shares nothing with this).

  C_j = sigma_j sqrt(N_j)                       (the paper's sigma_up is not available: sigma_down of (17) stands in)
  p_j = (C_j / sqrt t_j) / sum_l (C_l / sqrt t_l)
  (18): width_j <= (1/4) sigma_down,j sqrt(sum_l sigma_down,l^2) / sum_l sigma_down,l
  (19): sigma^2 = sum_j sigma_j^2
The uniform that picks the graph of block k is the oracle's Philox4x32-10 with key = scheduler seed, counter = (k, 0, 0, 0),
words 0 and 1 (DESIGN.md R-rng)."""
import math

from . import oracle as O


def sigma_down(sum_y, sum_y2, n):
    """(17)"""
    return math.sqrt(max(sum_y2 / n ** 2 - sum_y ** 2 / n ** 3, 0.0))


def probabilities(sum_y, sum_y2, n, t):
    c = [sigma_down(a, b, m) * math.sqrt(m) / math.sqrt(tt) for a, b, m, tt in zip(sum_y, sum_y2, n, t)]
    tot = 0.0
    for v in c:
        tot = tot + v
    return [v / tot for v in c] if tot > 0 else [1.0 / len(c)] * len(c)


def pick(p, sched_seed, block):
    w = O.philox([block & 0xFFFFFFFF, block >> 32, 0, 0], [sched_seed & 0xFFFFFFFF, sched_seed >> 32])
    u = O.u01(int(w[0]), int(w[1]))
    cum = 0.0
    for j, v in enumerate(p):
        cum = cum + v
        if u < cum:
            return j
    return len(p) - 1


def abs_tol_18(sum_y, sum_y2, n, target=0.0):
    """(18) with sigma_l at N = target samples per graph (target > 0) or at the samples seen so far."""
    sig = []
    for a, b, m in zip(sum_y, sum_y2, n):
        s = sigma_down(a, b, m) * math.sqrt(m)                 # per-sample standard deviation
        sig.append(s / math.sqrt(target if target > 0 else m))
    s1 = sum(sig); s2 = sum(v * v for v in sig)
    return [0.25 * v * math.sqrt(s2) / s1 for v in sig]


def combine_19(variances):
    return math.sqrt(sum(variances))
