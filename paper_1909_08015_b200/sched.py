"""Thin binding of the fg_batch_* calls of include/fg.h: several graphs integrated together -- initialisation stage,
acceptance rule (18), block scheduling p_j ~ C_j / sqrt(t_j), combination (19).
Argument marshalling only; the logic lives in csrc/fg_batch.cpp."""
import ctypes as C

import numpy as np

from . import fg


class Batch:
    def __init__(self, plans):
        self.plans = list(plans)
        arr = (C.c_void_p * len(self.plans))(*[p.h for p in self.plans])
        h = C.c_void_p()
        fg._check(fg.lib().fg_batch_create(arr, len(self.plans), C.byref(h)))
        self.h = h

    def __del__(self):
        try:
            if getattr(self, "h", None):
                fg.lib().fg_batch_destroy(self.h); self.h = None
        except Exception:
            pass

    def pilot(self, n_pilot, seed, first_sample=0, target_samples=0.0, rel_tol=0.0, stream=None):
        fg._check(fg.lib().fg_batch_pilot(self.h, int(n_pilot), int(seed), int(first_sample), float(target_samples), float(rel_tol), fg._stream(stream)))

    def set_times(self, seconds_per_sample):
        t = np.ascontiguousarray(seconds_per_sample, dtype=np.float64)
        fg._check(fg.lib().fg_batch_set_times(self.h, fg._p(t)))

    def probabilities(self):
        p = np.zeros(len(self.plans))
        fg._check(fg.lib().fg_batch_probabilities(self.h, fg._p(p)))
        return p

    def next(self, sched_seed, block_samples):
        j = C.c_int32(); first = C.c_uint64()
        fg._check(fg.lib().fg_batch_next(self.h, int(sched_seed), int(block_samples), C.byref(j), C.byref(first)))
        return j.value, first.value

    def fold(self, graph, result, seconds=0.0):
        fg._check(fg.lib().fg_batch_fold(self.h, int(graph), C.byref(result), float(seconds)))

    def run(self, n_blocks, block_samples, seed, sched_seed, stream=None):
        fg._check(fg.lib().fg_batch_run(self.h, int(n_blocks), int(block_samples), int(seed), int(sched_seed), fg._stream(stream)))

    def result(self, graph, raw=False):
        r = fg.fg_result(); tol = C.c_double(); t = C.c_double()
        fg._check(fg.lib().fg_batch_result(self.h, int(graph), C.byref(r), C.byref(tol), C.byref(t)))
        if raw:
            return r
        d = r.as_dict(); d["abs_tol"] = tol.value; d["seconds_per_sample"] = t.value
        return d

    @property
    def abs_tol(self):
        return [self.result(j)["abs_tol"] for j in range(len(self.plans))]

    def total(self):
        v = C.c_double(); s = C.c_double(); n = C.c_uint64()
        fg._check(fg.lib().fg_batch_total(self.h, C.byref(v), C.byref(s), C.byref(n)))
        return dict(value=v.value, sigma_down=s.value, n_samples=int(n.value))

    def set_classes(self, classes):
        """fg_batch_set_classes: one (k, m, m') per graph, e.g. [fg.Graph(...).gauge_class() ...]."""
        a = np.ascontiguousarray(classes, dtype=np.int32).reshape(len(self.plans), 3)
        fg._check(fg.lib().fg_batch_set_classes(self.h, fg._p(a)))

    def class_total(self, kmm):
        """fg_batch_class_total: value, sigma_down by (19) and number of graphs of one class."""
        a = np.ascontiguousarray(kmm, dtype=np.int32).reshape(3)
        v = C.c_double(); s = C.c_double(); n = C.c_int32()
        fg._check(fg.lib().fg_batch_class_total(self.h, fg._p(a), C.byref(v), C.byref(s), C.byref(n)))
        return dict(value=v.value, sigma_down=s.value, n_graphs=int(n.value))
