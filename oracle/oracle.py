"""ctypes binding of the CPU oracle (oracle/fg_oracle.cpp).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs.  The product package never imports this module.
"""
import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libfg_oracle.so")
_SRC = os.path.join(_HERE, "fg_oracle.cpp")


def build(force=False):
    """Compile the oracle (g++, OpenMP, no FMA contraction)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC",
                               "-o", _SO, _SRC])
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        L.fgo_create.restype = C.c_void_p
        L.fgo_create.argtypes = [C.c_int, C.c_int, C.c_void_p, C.c_int, C.c_void_p, C.c_double, C.c_void_p, C.c_int, C.c_int]
        L.fgo_destroy.argtypes = [C.c_void_p]
        L.fgo_set_rng.argtypes = [C.c_void_p, C.c_int]
        L.fgo_mrg32k3a.argtypes = [C.c_uint64, C.c_uint64, C.c_long, C.c_int, C.c_void_p]
        L.fgo_info.argtypes = [C.c_void_p, C.c_void_p]
        L.fgo_subs.argtypes = [C.c_void_p, C.c_void_p]
        L.fgo_terms.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        L.fgo_tables.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.fgo_eval.argtypes = [C.c_void_p, C.c_void_p, C.c_long, C.c_double, C.c_double, C.c_int, C.c_void_p,
                               C.c_void_p, C.c_void_p, C.c_void_p]
        L.fgo_sample.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.c_long] + [C.c_void_p] * 6
        L.fgo_integrate.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.c_long, C.c_int, C.c_double, C.c_double,
                                    C.c_void_p]
        L.fgo_eval_wide.argtypes = [C.c_void_p, C.c_void_p, C.c_long, C.c_void_p, C.c_void_p, C.c_void_p]
        L.fgo_bf_op.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
        L.fgo_eval_abs.argtypes = [C.c_void_p, C.c_void_p, C.c_long, C.c_void_p]
        L.fgo_geom_eval.restype = C.c_int
        L.fgo_geom_eval.argtypes = [C.c_void_p, C.c_int] + [C.c_void_p] * 10
        L.fgo_dirac_selfcheck.restype = C.c_double
        L.fgo_dirac_selfcheck.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.fgo_geom_desc.restype = C.c_int
        L.fgo_geom_desc.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.fgo_dirac_table.restype = C.c_int
        L.fgo_dirac_table.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        L.fgo_dirac_explicit.restype = C.c_double
        L.fgo_dirac_explicit.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_int, C.c_uint]
        L.fgo_u01.restype = C.c_double
        L.fgo_u01.argtypes = [C.c_uint32, C.c_uint32]
        L.fgo_enumerate.argtypes = [C.c_int, C.c_void_p, C.c_int]
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def philox(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32); k = np.asarray(key, dtype=np.uint32); o = np.zeros(4, dtype=np.uint32)
    lib().fgo_philox(_p(c), _p(k), _p(o))
    return o


def u01(w0, w1):
    return lib().fgo_u01(int(w0), int(w1))


def enumerate_graphs(n):
    """All directed n-loop vertex graphs without lepton loops: list of (x, [(a,b),...])."""
    cap = 8000
    out = np.zeros(cap * (1 + 2 * n), dtype=np.int32)
    cnt = lib().fgo_enumerate(n, _p(out), cap)
    out = out.reshape(cap, 1 + 2 * n)[:cnt]
    return [(int(r[0]), [(int(r[1 + 2 * k]), int(r[2 + 2 * k])) for k in range(n)]) for r in out]


def count_undirected(n):
    return lib().fgo_count_undirected(n)


def mrg32k3a(seed, first, n, by_jump=False):
    """Raw MRG32k3a outputs first .. first+n-1 of the sequence of `seed` (seed 0 = L'Ecuyer's 12345 x 6)."""
    out = np.zeros(n)
    lib().fgo_mrg32k3a(int(seed), int(first), int(n), int(bool(by_jump)), _p(out))
    return out


def gauge_class(x, photons):
    """Class (k, m, m') of PAPER.md:393 (Table I): m, m' = internal photons to the left / right of the external photon
    (the larger first), k = photons whose ends lie on opposite sides of it.  Plain definition."""
    left = sum(1 for a, b in photons if max(a, b) < x)
    right = sum(1 for a, b in photons if min(a, b) > x)
    k = sum(1 for a, b in photons if min(a, b) < x < max(a, b))
    assert left + right + k == len(photons)
    return k, max(left, right), min(left, right)


OPS = {0: "A", 1: "U", 2: "L", 3: "L-U"}


class Oracle:
    def __init__(self, x, photons, merge=False, C4=(0.9, 0.03, 0.01, 0.06), D=0.75, deg_table=None, printed=None, structure_only=False):
        n = len(photons)
        self.n, self.x, self.photons = n, x, [tuple(p) for p in photons]
        ph = np.asarray(photons, dtype=np.int32).reshape(-1)
        c4 = np.asarray(C4, dtype=np.float64)
        if printed is None:
            printed = n <= 3          # the projector exactly as stated; its reduced form (pinned equal) above 3 loops
        dt = None if deg_table is None else np.ascontiguousarray(deg_table, dtype=np.float64)
        # structure_only: True / 1 = subgraphs, forests and terms only; 2 = also the element geometries (no numerator tables)
        self.h = lib().fgo_create(n, x, _p(ph), int(bool(merge)), _p(c4), float(D), _p(dt), int(bool(printed)), int(structure_only))
        if not self.h:
            raise ValueError("invalid graph")
        self.rng = 0
        info = np.zeros(8, dtype=np.int64)
        lib().fgo_info(self.h, _p(info))
        self.M, self.n_subs, self.n_forests, self.n_terms, self.n_geoms, self.n_nums, self.n_patterns = map(int, info[:7])

    def __del__(self):
        try:
            if self.h:
                lib().fgo_destroy(self.h)
                self.h = None
        except Exception:
            pass

    def subs(self):
        out = np.zeros((self.n_subs, 4), dtype=np.int32)
        lib().fgo_subs(self.h, _p(out))
        return [dict(a=int(r[0]), b=int(r[1]), type="V" if r[2] else "SE", in_chain=bool(r[3])) for r in out]

    def terms(self):
        buf = np.zeros(200000, dtype=np.int32)
        w = lib().fgo_terms(self.h, _p(buf), len(buf))
        assert w >= 0
        res, i = [], 0
        while i < w:
            sign, gp, nm = int(buf[i]), int(buf[i + 1]), int(buf[i + 2]); i += 3
            mem = [(int(buf[i + 2 * k]), OPS[int(buf[i + 2 * k + 1])]) for k in range(nm)]; i += 2 * nm
            res.append(dict(sign=sign, gprime=gp, members=mem))
        return res

    def tables(self):
        d = np.zeros(1 << self.M); z = np.zeros(1 << self.M)
        lib().fgo_tables(self.h, _p(d), _p(z))
        return d, z

    def eval(self, z, rel_tol=1e-12, abs_tol=0.0, quad=True, terms=False):
        z = np.ascontiguousarray(z, dtype=np.float64).reshape(-1, self.M)
        n = len(z)
        Id = np.zeros(n); Iq = np.zeros(n); fl = np.zeros(n, dtype=np.uint8)
        td = np.zeros((n, self.n_terms + 1)) if terms else None
        lib().fgo_eval(self.h, _p(z), n, rel_tol, abs_tol, int(quad), _p(Id), _p(Iq), _p(fl), _p(td))
        return (Id, Iq, fl, td) if terms else (Id, Iq, fl)

    def eval_wide(self, z):
        """(I_w, I_q, dist): integrand in 256-bit arithmetic and in __float128 (both rounded to double) and the relative
        distance |I_q - I_w| / |I_w| of the two."""
        z = np.ascontiguousarray(z, dtype=np.float64).reshape(-1, self.M)
        n = len(z)
        Iw = np.zeros(n); Iq = np.zeros(n); dist = np.zeros(n)
        lib().fgo_eval_wide(self.h, _p(z), n, _p(Iw), _p(Iq), _p(dist))
        return Iw, Iq, dist

    def eval_abs(self, z):
        """Upper bound of the sum of |terms| of the oracle's own evaluation (diagnostic of cancellation)."""
        z = np.ascontiguousarray(z, dtype=np.float64).reshape(-1, self.M); out = np.zeros(len(z))
        lib().fgo_eval_abs(self.h, _p(z), len(z), _p(out))
        return out

    def set_rng(self, rng):
        """0: Philox4x32-10 (Calc 2); 1: MRG32k3a (Calc 1)."""
        self.rng = int(rng); lib().fgo_set_rng(self.h, int(rng))

    def sample(self, seed, first, n):
        M = self.M
        comp = np.zeros(n, dtype=np.int32); order = np.zeros((n, M), dtype=np.uint8); z = np.zeros((n, M))
        pm = np.zeros(n); pe = np.zeros(n, dtype=np.int32); bad = np.zeros(n, dtype=np.uint8)
        lib().fgo_sample(self.h, seed, first, n, _p(comp), _p(order), _p(z), _p(pm), _p(pe), _p(bad))
        return dict(comp=comp, order=order, z=z, pdf_mant=pm, pdf_exp=pe, bad=bad)

    def integrate(self, seed, first, n, quad=False, rel_tol=1e-12, abs_tol=0.0, wide=False):
        """quad: y from the __float128 integrand; wide: from the 256-bit one (the reference at ill-conditioned points)."""
        out = np.zeros(8)
        lib().fgo_integrate(self.h, seed, first, n, 2 if wide else int(quad), rel_tol, abs_tol, _p(out))
        return dict(sum_y=out[0], sum_y2=out[1], n_flagged=int(out[2]), n_rejected=int(out[3]), n_pdf_big_exp=int(out[4]),
                    mean=out[5], variance=out[6], n_samples=n)

    def geom_eval(self, gi, zlines):
        zl = np.ascontiguousarray(zlines, dtype=np.float64)
        U = np.zeros(1); W = np.zeros(1); beta = np.zeros(400); A = np.zeros(20); Aq = np.zeros(20)
        own = np.zeros(40, dtype=np.int32); nl = np.zeros(1, dtype=np.int32); ends = np.zeros(80, dtype=np.int32)
        xiq = np.zeros(20, dtype=np.int32)
        ne = lib().fgo_geom_eval(self.h, gi, _p(zl), _p(U), _p(W), _p(beta), _p(A), _p(Aq), _p(own), _p(nl), _p(ends), _p(xiq))
        nlines = int(nl[0])
        return dict(ne=ne, U=U[0], W=W[0], beta=beta[:ne * ne].reshape(ne, ne).copy(), A=A[:ne].copy(), Aq=Aq[:ne].copy(), xiq=xiq[:ne].copy(),
                    own=own[:nlines].copy(), ends=ends[:2 * nlines].reshape(nlines, 2).copy())

    def geom_desc(self, gi):
        buf = np.zeros(64, dtype=np.int32)
        w = lib().fgo_geom_desc(self.h, gi, _p(buf))
        return dict(a=int(buf[0]), b=int(buf[1]), type=int(buf[2]), nslots=int(buf[3]), l=int(buf[4]),
                    children=[(int(buf[6 + 2 * k]), int(buf[7 + 2 * k])) for k in range(int(buf[5]))])

    def dirac_table(self, gi, op, comp, pairs, qslot):
        """(gaps, table over the subsets of the gaps) of one matching of element gi from the oracle's fast engine."""
        pr = np.asarray(pairs, dtype=np.int32).reshape(-1); tab = np.zeros(1 << 12); gaps = np.zeros(16, dtype=np.int32)
        ng = lib().fgo_dirac_table(self.h, gi, int(op), int(comp), len(pr) // 2, _p(pr), int(qslot), _p(tab), _p(gaps))
        return [int(v) for v in gaps[:ng]], tab[:1 << ng].copy()

    def dirac_explicit(self, gi, op, comp, pairs, qslot, tmask):
        """Coefficient of one pattern of element gi from explicit 4x4 matrices (without (-1/2)^pairs)."""
        pr = np.asarray(pairs, dtype=np.int32).reshape(-1)
        return lib().fgo_dirac_explicit(self.h, gi, int(op), int(comp), len(pr) // 2, _p(pr), int(qslot), int(tmask))

    def dirac_selfcheck(self, maxpat=50):
        cnt = np.zeros(1, dtype=np.int64)
        w = lib().fgo_dirac_selfcheck(self.h, maxpat, _p(cnt))
        return w, int(cnt[0])


def bf_op(op, a3, b3):
    """The oracle's 256-bit arithmetic on a = sum(a3), b = sum(b3): op 0 +, 1 -, 2 *, 3 /; result as five doubles."""
    a = np.asarray(a3, dtype=np.float64); b = np.asarray(b3, dtype=np.float64); r = np.zeros(5)
    lib().fgo_bf_op(int(op), _p(a), _p(b), _p(r))
    return r


def threads():
    return lib().fgo_threads()
