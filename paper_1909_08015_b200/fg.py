"""Thin ctypes binding of the C ABI in include/fg.h (argument marshalling only; every step runs in the CUDA
kernels of libfg.so).  Names follow the C calls: fg_graph_create -> Graph, fg_plan_create -> Plan,
fg_integrate -> Plan.integrate, ...  There is no CPU fallback: without libfg.so or without a CUDA device the
calls raise.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("FG_LIB") or os.path.join(_HERE, "libfg.so")     # FG_LIB: a variant build (profiling counters)

EXPORTS = ["fg_graph_create", "fg_graph_destroy", "fg_plan_opts_default", "fg_plan_create", "fg_plan_destroy",
           "fg_plan_info", "fg_plan_phase_cycles", "fg_host_plan", "fg_host_dirac_table", "fg_plan_set_tol", "fg_plan_profile", "fg_plan_timing", "fg_plan_structure", "fg_plan_tables", "fg_integrate", "fg_integrate_range",
           "fg_integrate_async", "fg_result_merge", "fg_sample_dump", "fg_eval_points", "fg_sample_eval_dump",
           "fg_dfma_peak", "fg_dmma_peak", "fg_strerror", "fg_last_error_message", "fg_version",
           "fg_batch_create", "fg_batch_destroy", "fg_batch_pilot", "fg_batch_set_times", "fg_batch_probabilities", "fg_batch_next",
           "fg_batch_fold", "fg_batch_run", "fg_batch_result", "fg_batch_total", "fg_batch_set_classes", "fg_batch_class_total", "fg_graph_class",
           "fg_noalloc_setup", "fg_noalloc_limits", "fg_eval_points_dd_noalloc"]


class FgError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("fg error %d: %s" % (code, msg))
        self.code = code


class fg_edge(C.Structure):
    _fields_ = [("u", C.c_int32), ("v", C.c_int32), ("kind", C.c_int32)]


class fg_plan_opts(C.Structure):
    _fields_ = [("C", C.c_double * 4), ("D", C.c_double), ("merge_ext_lines", C.c_int32), ("deg_rule", C.c_int32),
                ("deg_table", C.c_void_p), ("rel_tol", C.c_double), ("abs_tol", C.c_double), ("err_factor", C.c_double),
                ("deg_consts", C.c_double * 6), ("structure_only", C.c_int32), ("rng", C.c_int32)]


class fg_plan_stats(C.Structure):
    _fields_ = [("n_loops", C.c_int32), ("M", C.c_int32), ("n_subgraphs", C.c_int32), ("n_forests", C.c_int32),
                ("n_terms", C.c_int32), ("n_geoms", C.c_int32), ("n_nums", C.c_int32), ("n_nodes", C.c_int32),
                ("n_records", C.c_int64), ("n_coefs", C.c_int64), ("n_coefs_nonzero", C.c_int64),
                ("table_bytes", C.c_int64), ("stream_bytes", C.c_int64), ("flops_per_sample", C.c_double),
                ("exec_flops_per_sample", C.c_double), ("plan_seconds", C.c_double), ("wave_samples", C.c_int64)]


class fg_result(C.Structure):
    _fields_ = [("mean", C.c_double), ("variance", C.c_double), ("sum_y", C.c_double * 2), ("sum_y2", C.c_double * 2),
                ("n_samples", C.c_uint64), ("n_flagged", C.c_uint64), ("n_flagged2", C.c_uint64), ("n_rejected", C.c_uint64),
                ("n_pdf_big_exp", C.c_uint64)]

    def as_dict(self):
        return dict(mean=self.mean, variance=self.variance, sum_y=(self.sum_y[0], self.sum_y[1]),
                    sum_y2=(self.sum_y2[0], self.sum_y2[1]), n_samples=int(self.n_samples),
                    n_flagged=int(self.n_flagged), n_flagged2=int(self.n_flagged2), n_rejected=int(self.n_rejected),
                    n_pdf_big_exp=int(self.n_pdf_big_exp))


_lib = None


def lib():
    """Loads libfg.so (built by paper_1909_08015_b200.build).  Raises if it is missing: no fallback."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FgError(-7, "libfg.so is not built (run `python -m paper_1909_08015_b200.build`); there is no CPU path")
        L = C.CDLL(LIB_PATH)
        vp = C.c_void_p
        L.fg_graph_create.argtypes = [vp, C.c_int32, C.c_int32, C.POINTER(vp)]
        L.fg_graph_destroy.argtypes = [vp]
        L.fg_plan_opts_default.argtypes = [C.POINTER(fg_plan_opts)]
        L.fg_plan_create.argtypes = [vp, C.POINTER(fg_plan_opts), C.c_int32, C.POINTER(vp)]
        L.fg_plan_destroy.argtypes = [vp]
        L.fg_host_plan.argtypes = [vp, C.POINTER(fg_plan_opts), C.POINTER(fg_plan_stats), vp, C.c_int32, vp, C.c_int32, vp, vp]
        L.fg_host_dirac_table.argtypes = [vp, C.c_int32, C.c_int32, vp, C.c_int32, C.c_int32, C.c_int32, vp, C.c_int32, C.c_int32, vp, C.c_int32, vp, vp]
        L.fg_plan_set_tol.argtypes = [vp, C.c_double, C.c_double]
        L.fg_plan_profile.argtypes = [vp, C.c_int32]
        L.fg_plan_timing.argtypes = [vp, vp, vp]
        L.fg_plan_info.argtypes = [vp, C.POINTER(fg_plan_stats)]
        L.fg_plan_phase_cycles.argtypes = [vp, vp, C.c_int32]
        L.fg_plan_structure.argtypes = [vp, vp, vp, C.c_int32]
        L.fg_plan_tables.argtypes = [vp, vp, vp]
        L.fg_integrate.argtypes = [vp, C.c_uint64, C.c_uint64, vp, C.POINTER(fg_result)]
        L.fg_integrate_range.argtypes = [vp, C.c_uint64, C.c_uint64, C.c_uint64, vp, C.POINTER(fg_result)]
        L.fg_integrate_async.argtypes = [vp, C.c_uint64, C.c_uint64, C.c_uint64, vp, vp]
        L.fg_result_merge.argtypes = [C.POINTER(fg_result), C.POINTER(fg_result), C.POINTER(fg_result)]
        L.fg_sample_dump.argtypes = [vp, C.c_uint64, C.c_uint64, C.c_uint64, vp] + [vp] * 7
        L.fg_eval_points.argtypes = [vp, vp, C.c_uint64, C.c_int32, vp] + [vp] * 4
        L.fg_sample_eval_dump.argtypes = [vp, C.c_uint64, C.c_uint64, C.c_uint64, vp] + [vp] * 3
        L.fg_dfma_peak.argtypes = [C.c_int32, C.c_int32, vp, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.fg_dmma_peak.argtypes = [C.c_int32, C.c_int32, vp, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.fg_graph_class.argtypes = [vp, vp]
        L.fg_batch_set_classes.argtypes = [vp, vp]
        L.fg_batch_class_total.argtypes = [vp, vp, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_int32)]
        L.fg_batch_create.argtypes = [vp, C.c_int32, C.POINTER(vp)]
        L.fg_batch_destroy.argtypes = [vp]
        L.fg_batch_pilot.argtypes = [vp, C.c_uint64, C.c_uint64, C.c_uint64, C.c_double, C.c_double, vp]
        L.fg_batch_set_times.argtypes = [vp, vp]
        L.fg_batch_probabilities.argtypes = [vp, vp]
        L.fg_batch_next.argtypes = [vp, C.c_uint64, C.c_uint64, C.POINTER(C.c_int32), C.POINTER(C.c_uint64)]
        L.fg_batch_fold.argtypes = [vp, C.c_int32, C.POINTER(fg_result), C.c_double]
        L.fg_batch_run.argtypes = [vp, C.c_uint64, C.c_uint64, C.c_uint64, C.c_uint64, vp]
        L.fg_batch_result.argtypes = [vp, C.c_int32, C.POINTER(fg_result), C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.fg_batch_total.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_uint64)]
        L.fg_noalloc_setup.argtypes = [C.c_int32]
        L.fg_noalloc_limits.argtypes = [C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
        L.fg_eval_points_dd_noalloc.argtypes = [vp, vp, C.c_uint64, vp, vp, vp, vp]
        for f in ("fg_strerror", "fg_last_error_message", "fg_version"):
            getattr(L, f).restype = C.c_char_p
        L.fg_strerror.argtypes = [C.c_int]
        _lib = L
    return _lib


def _check(rc):
    if rc < 0:
        raise FgError(rc, "%s: %s" % (lib().fg_strerror(rc).decode(), lib().fg_last_error_message().decode()))
    return rc


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _stream(stream):
    if stream is None:
        return None
    return C.c_void_p(int(getattr(stream, "cuda_stream", stream)))


def version():
    return lib().fg_version().decode()


class Graph:
    """fg_graph_create: edge list (u, v, kind) with kind 0 = electron, 1 = photon; vertex of the external photon."""

    def __init__(self, edges, ext_photon_vertex):
        arr = (fg_edge * len(edges))(*[fg_edge(int(u), int(v), int(k)) for u, v, k in edges])
        h = C.c_void_p()
        _check(lib().fg_graph_create(arr, len(edges), int(ext_photon_vertex), C.byref(h)))
        self.h = h

    def __del__(self):
        try:
            if getattr(self, "h", None):
                lib().fg_graph_destroy(self.h); self.h = None
        except Exception:
            pass

    def gauge_class(self):
        """fg_graph_class: (k, m, m') of PAPER.md:393."""
        kmm = np.zeros(3, dtype=np.int32)
        _check(lib().fg_graph_class(self.h, _p(kmm)))
        return tuple(int(v) for v in kmm)


class Plan:
    """fg_plan_create (+ fg_plan_info, fg_integrate, ... on the plan)."""

    def __init__(self, graph, merge_ext_lines=False, C4=None, D=None, deg_table=None, rel_tol=1e-12, abs_tol=0.0,
                 err_factor=0.0, device=0, deg_rule=0, deg_consts=None, rng=0):
        o = fg_plan_opts(); lib().fg_plan_opts_default(C.byref(o)); o.rng = int(rng)
        if C4 is not None:
            for k in range(4):
                o.C[k] = float(C4[k])
        if D is not None:
            o.D = float(D)
        o.merge_ext_lines = int(bool(merge_ext_lines)); o.rel_tol = float(rel_tol); o.abs_tol = float(abs_tol)
        o.err_factor = float(err_factor); o.deg_rule = int(deg_rule)
        if deg_consts is not None:
            for k in range(6):
                o.deg_consts[k] = float(deg_consts[k])
        self._deg = None
        if deg_table is not None:
            self._deg = np.ascontiguousarray(deg_table, dtype=np.float64); o.deg_table = self._deg.ctypes.data
        h = C.c_void_p()
        _check(lib().fg_plan_create(graph.h, C.byref(o), int(device), C.byref(h)))
        self.h = h
        self.stats = self.info()
        self.M = self.stats["M"]

    def __del__(self):
        try:
            if getattr(self, "h", None):
                lib().fg_plan_destroy(self.h); self.h = None
        except Exception:
            pass

    def info(self):
        s = fg_plan_stats(); _check(lib().fg_plan_info(self.h, C.byref(s)))
        return {k: getattr(s, k) for k, _ in fg_plan_stats._fields_}

    def set_tol(self, rel_tol, abs_tol):
        _check(lib().fg_plan_set_tol(self.h, float(rel_tol), float(abs_tol)))

    def profile(self, enable=True):
        _check(lib().fg_plan_profile(self.h, int(bool(enable))))

    def timing(self):
        ms = np.zeros(3); n = np.zeros(1, dtype=np.int64)
        _check(lib().fg_plan_timing(self.h, _p(ms), _p(n)))
        return dict(ms_double=ms[0], ms_dd=ms[1], ms_reduce=ms[2], launches=int(n[0]))

    def phase_cycles(self, reset=True):
        """fg_plan_phase_cycles: (built_with_counters, warp-cycles per phase) of a -DFG_PHASE_PROF build."""
        c = np.zeros(16, dtype=np.uint64)
        rc = _check(lib().fg_plan_phase_cycles(self.h, _p(c), int(bool(reset))))
        return bool(rc), c

    def wave_samples(self):
        """Samples of one wave of the double-precision pass (one fg_geom_kernel + one fg_stream_kernel launch)."""
        return int(self.stats["wave_samples"])

    def structure(self):
        ns = self.stats["n_subgraphs"]
        subs = np.zeros((ns, 4), dtype=np.int32); buf = np.zeros(1 << 16, dtype=np.int32)
        w = _check(lib().fg_plan_structure(self.h, _p(subs), _p(buf), len(buf)))
        ops = {0: "A", 1: "U", 2: "L", 3: "L-U"}
        terms, i = [], 0
        while i < w:
            sign, gp, nm = int(buf[i]), int(buf[i + 1]), int(buf[i + 2]); i += 3
            terms.append(dict(sign=sign, gprime=gp, members=[(int(buf[i + 2 * k]), ops[int(buf[i + 2 * k + 1])]) for k in range(nm)]))
            i += 2 * nm
        return [dict(a=int(r[0]), b=int(r[1]), type="V" if r[2] else "SE", in_chain=bool(r[3])) for r in subs], terms

    def tables(self):
        d = np.zeros(1 << self.M); z = np.zeros(1 << self.M)
        _check(lib().fg_plan_tables(self.h, _p(d), _p(z)))
        return d, z

    def integrate(self, n_samples, seed, stream=None):
        r = fg_result(); _check(lib().fg_integrate(self.h, int(n_samples), int(seed), _stream(stream), C.byref(r)))
        return r.as_dict()

    def integrate_range(self, first_sample, n_samples, seed, stream=None, raw=False):
        r = fg_result()
        _check(lib().fg_integrate_range(self.h, int(first_sample), int(n_samples), int(seed), _stream(stream), C.byref(r)))
        return r if raw else r.as_dict()

    def integrate_async(self, first_sample, n_samples, seed, out_dev_ptr, stream=None):
        """Result (sizeof(fg_result) = 80 bytes) is left at device address out_dev_ptr; no synchronisation."""
        _check(lib().fg_integrate_async(self.h, int(first_sample), int(n_samples), int(seed), _stream(stream),
                                        C.c_void_p(int(out_dev_ptr))))

    def sample_dump(self, first, n, seed, stream=None, words=True):
        M = self.M
        w = np.zeros((n, M, 4), dtype=np.uint32) if words else None
        comp = np.zeros(n, dtype=np.int32); order = np.zeros((n, M), dtype=np.uint8); z = np.zeros((n, M))
        pm = np.zeros(n); pe = np.zeros(n, dtype=np.int32); bad = np.zeros(n, dtype=np.uint8)
        _check(lib().fg_sample_dump(self.h, int(first), int(n), int(seed), _stream(stream), _p(w), _p(comp), _p(order),
                                    _p(z), _p(pm), _p(pe), _p(bad)))
        return dict(words=w, comp=comp, order=order, z=z, pdf_mant=pm, pdf_exp=pe, bad=bad)

    def eval_points(self, z, mode=0, stream=None):
        z = np.ascontiguousarray(z, dtype=np.float64).reshape(-1, self.M); n = len(z)
        I = np.zeros(n); Id = np.zeros(n); err = np.zeros(n); fl = np.zeros(n, dtype=np.uint8)
        _check(lib().fg_eval_points(self.h, _p(z), n, int(mode), _stream(stream), _p(I), _p(Id), _p(err), _p(fl)))
        return dict(I=I, I_double=Id, err=err, flags=fl)

    def eval_points_dd_noalloc(self, z_dev_ptr, n, I_dev_ptr, err_dev_ptr, flags_dev_ptr, stream=None):
        """fg_eval_points_dd_noalloc: every argument is a DEVICE address (int) owned by the caller; allocates nothing."""
        _check(lib().fg_eval_points_dd_noalloc(self.h, C.c_void_p(int(z_dev_ptr)), int(n), _stream(stream), C.c_void_p(int(I_dev_ptr)),
                                               C.c_void_p(int(err_dev_ptr)) if err_dev_ptr else None, C.c_void_p(int(flags_dev_ptr))))

    def sample_eval_dump(self, first, n, seed, stream=None):
        I = np.zeros(n); y = np.zeros(n); fl = np.zeros(n, dtype=np.uint8)
        _check(lib().fg_sample_eval_dump(self.h, int(first), int(n), int(seed), _stream(stream), _p(I), _p(y), _p(fl)))
        return dict(I=I, y=y, flags=fl)


_OPS = {0: "A", 1: "U", 2: "L", 3: "L-U"}


def host_plan(graph, merge_ext_lines=False, deg_table=None, tables=False, structure_only=False):
    """fg_host_plan: the planner alone (host, no device): (stats, subgraphs, terms[, Deg, Z_1])."""
    o = fg_plan_opts(); lib().fg_plan_opts_default(C.byref(o)); o.merge_ext_lines = int(bool(merge_ext_lines))
    o.structure_only = int(bool(structure_only))
    keep = None
    if deg_table is not None:
        keep = np.ascontiguousarray(deg_table, dtype=np.float64); o.deg_table = keep.ctypes.data
    st = fg_plan_stats(); subs = np.zeros((64, 4), dtype=np.int32); buf = np.zeros(1 << 16, dtype=np.int32)
    deg = z1 = None
    if tables:
        deg = np.zeros(1 << 15); z1 = np.zeros(1 << 15)
    w = _check(lib().fg_host_plan(graph.h, C.byref(o), C.byref(st), _p(subs), 64, _p(buf), len(buf), _p(deg), _p(z1)))
    stats = {k: getattr(st, k) for k, _ in fg_plan_stats._fields_}
    terms, i = [], 0
    while i < w:
        sign, gp, nm = int(buf[i]), int(buf[i + 1]), int(buf[i + 2]); i += 3
        terms.append(dict(sign=sign, gprime=gp, members=[(int(buf[i + 2 * k]), _OPS[int(buf[i + 2 * k + 1])]) for k in range(nm)]))
        i += 2 * nm
    ss = [dict(a=int(r[0]), b=int(r[1]), type="V" if r[2] else "SE", in_chain=bool(r[3])) for r in subs[:stats["n_subgraphs"]]]
    if tables:
        n = 1 << stats["M"]
        return stats, ss, terms, deg[:n], z1[:n]
    return stats, ss, terms


def host_dirac_table(graph, a, b, kids, op, comp, pairs, qslot=-1):
    """fg_host_dirac_table: (n_slots, gaps, table over the subsets of the gaps) of one matching of one element."""
    kd = np.asarray(kids, dtype=np.int32).reshape(-1); pr = np.asarray(pairs, dtype=np.int32).reshape(-1)
    tab = np.zeros(1 << 12); gaps = np.zeros(16, dtype=np.int32); ng = np.zeros(1, dtype=np.int32)
    ns = _check(lib().fg_host_dirac_table(graph.h, int(a), int(b), _p(kd), len(kd) // 2, int(op), int(comp), _p(pr), len(pr) // 2,
                                          int(qslot), _p(tab), len(tab), _p(gaps), _p(ng)))
    n = int(ng[0])
    return ns, [int(v) for v in gaps[:n]], tab[:1 << n].copy()


def result_merge(a, b):
    """fg_result_merge on two raw fg_result structs."""
    out = fg_result(); _check(lib().fg_result_merge(C.byref(a), C.byref(b), C.byref(out)))
    return out


def noalloc_setup(device=0):
    _check(lib().fg_noalloc_setup(int(device)))


def noalloc_limits():
    a = C.c_uint64(); b = C.c_uint64()
    _check(lib().fg_noalloc_limits(C.byref(a), C.byref(b)))
    return int(a.value), int(b.value)


def dfma_peak(device=0, iters=200000, stream=None):
    """fg_dfma_peak: measured FP64-FMA throughput (TFLOP/s, FMA = 2) and kernel time in ms."""
    t = C.c_double(); ms = C.c_double()
    _check(lib().fg_dfma_peak(int(device), int(iters), _stream(stream), C.byref(t), C.byref(ms)))
    return t.value, ms.value


def dmma_peak(device=0, iters=20000, stream=None):
    """fg_dmma_peak: measured FP64 tensor-core (DMMA m8n8k4) throughput (TFLOP/s) and kernel time in ms."""
    t = C.c_double(); ms = C.c_double()
    _check(lib().fg_dmma_peak(int(device), int(iters), _stream(stream), C.byref(t), C.byref(ms)))
    return t.value, ms.value


def plan_for(x, photons, **kw):
    """Convenience: (x, photons) in the notation of paper_1909_08015_b200.inputs -> Plan."""
    from . import inputs
    g = Graph(inputs.edge_list(x, photons), x)
    return Plan(g, **kw)
