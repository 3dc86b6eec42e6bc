"""ctypes loader for the CPU oracle (oracle/lst_oracle.cpp) -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from the CUDA package.
"""
import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lst_oracle.cpp")
_LIB = os.path.join(_HERE, "liblst_oracle.so")
CXXFLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC"]

CUTS = ["M2", "M3", "L1", "L2", "L3", "T1", "T2", "T3", "Q1", "Q2", "P5", "P3"]
STAGE = {"sort": 0, "md": 1, "ls": 2, "t3": 3, "t5": 4, "tc": 5, "clean": 6}


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", *CXXFLAGS, "-o", _LIB, _SRC])
    return _LIB


_lib = None


def _bind(path):
    """dlopen an oracle library and declare its signatures."""
    L = C.CDLL(path)
    L.lst_oracle_run.restype = C.c_void_p
    L.lst_oracle_run.argtypes = [C.c_int32] + [C.c_void_p] * 5 + [C.c_int32] + [C.c_void_p] * 4 + \
        [C.c_int32] + [C.c_void_p] * 5 + [C.c_void_p, C.c_int32, C.c_void_p, C.c_int32, C.c_int32] + [C.c_int32, C.c_int32, C.c_void_p]
    L.lst_oracle_count.restype = C.c_int64
    L.lst_oracle_count.argtypes = [C.c_void_p, C.c_int32]
    L.lst_oracle_copy_int.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
    L.lst_oracle_copy_real.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
    L.lst_oracle_free.argtypes = [C.c_void_p]
    L.lst_oracle_md_eval.restype = C.c_int32
    L.lst_oracle_md_eval.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p]
    L.lst_oracle_ls_eval.restype = C.c_int32
    L.lst_oracle_ls_eval.argtypes = [C.c_void_p] * 3
    L.lst_oracle_t3_eval.restype = C.c_int32
    L.lst_oracle_t3_eval.argtypes = [C.c_void_p] * 3 + [C.c_float, C.c_float, C.c_void_p]
    L.lst_oracle_bridge_eval.restype = C.c_int32
    L.lst_oracle_bridge_eval.argtypes = [C.c_void_p] * 4
    L.lst_oracle_pls_match.restype = C.c_int32
    L.lst_oracle_pls_match.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_int32, C.c_void_p]
    L.lst_oracle_pls_residual.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]
    L.lst_oracle_tc_clean.argtypes = [C.c_int32] + [C.c_void_p] * 5
    L.lst_oracle_arcfac.restype = C.c_float
    L.lst_oracle_arcfac.argtypes = [C.c_float]
    L.lst_oracle_arcfac_f64.restype = C.c_double
    L.lst_oracle_arcfac_f64.argtypes = [C.c_double]
    L.lst_oracle_features.argtypes = [C.c_void_p] * 4 + [C.c_float] * 3 + [C.c_void_p]
    L.lst_oracle_mlp.restype = C.c_float
    L.lst_oracle_mlp.argtypes = [C.c_void_p, C.c_void_p]
    L.lst_oracle_mlp_n.restype = C.c_float
    L.lst_oracle_mlp_n.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32]
    L.lst_oracle_features38.argtypes = [C.c_void_p] * 5 + [C.c_float] * 3 + [C.c_void_p]
    return L


def lib():
    global _lib
    if _lib is None:
        _lib = _bind(build())
    return _lib


class use_library:
    """Context manager for tests/test_oracle_mutants.py: route every call of this module through another
    build of the oracle (a deliberately broken copy) so that the pins can be shown to notice the breakage."""

    def __init__(self, path):
        self.path = path

    def __enter__(self):
        global _lib
        self.saved = _lib
        _lib = _bind(self.path)
        return self

    def __exit__(self, *exc):
        global _lib
        _lib = self.saved
        return False


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class OracleResult:
    """Outputs of one oracle run.  Index tables are in the oracle's build order (SPEC.md 5):
    md_hits[n,2] original hit indices (lower, upper); ls[n,2] MD indices; t3[n,5] = MD a,b,c + LS i,j;
    t5c[n,8] = MD[5], T3 in, T3 out, pass; t5[n] candidate indices; tc[n,3] = type, pLS, object."""

    def __init__(self, h, L, n_feat=23):
        cnt = lambda w: int(L.lst_oracle_count(h, w))

        def ints(w, k, nw=None):
            n = cnt((w if w < 7 else 5) if nw is None else nw)
            o = np.zeros((n, k), dtype=np.int32)
            if n:
                L.lst_oracle_copy_int(h, w, _p(o))
            return o

        def reals(w, k, nw=None):
            n = cnt(w if nw is None else nw)
            o = np.zeros((n, k), dtype=np.float64)
            if n:
                L.lst_oracle_copy_real(h, w, _p(o))
            return o

        self.flags = cnt(20)
        self.hit_orig = ints(0, 1)[:, 0]
        ss = np.zeros(cnt(21), dtype=np.int32)
        L.lst_oracle_copy_int(h, 21, _p(ss))
        self.sensor_start = ss
        md = ints(1, 3)
        self.md_hits, self.md_mod = md[:, :2].copy(), md[:, 2].copy()
        self.md_real = reals(1, 6)          # c, w, x, y, z, r
        self.ls = ints(2, 2)
        self.ls_c = reals(2, 1)[:, 0]
        self.t3 = ints(3, 5)
        self.t3_k = reals(3, 1)[:, 0]
        self.t5c = ints(4, 8)
        r5 = reals(4, 42)
        self.t5c_curv, self.t5c_score, self.t5c_feat = r5[:, :3].copy(), r5[:, 3].copy(), r5[:, 4:4 + n_feat].copy()
        self.t5 = ints(5, 1)[:, 0]
        self.tc = ints(6, 3)
        self.best5_pls = ints(7, 1)[:, 0]
        self.chi5 = reals(7, 1, nw=5)[:, 0]
        self.chi3 = reals(9, 1, nw=3)[:, 0]
        self.tcc = ints(8, 3, nw=8)                 # cleaned TC list (SPEC.md 4.7)
        self.tc_keep = ints(9, 1, nw=6)[:, 0]
        has_clean = len(self.tc_keep) == len(self.tc)
        self.tc_hits = ints(10, 10, nw=6) if has_clean else np.zeros((0, 10), np.int32)     # hit tuple of every TC row
        self.tc_q = ints(11, 1, nw=6)[:, 0].view(np.uint32) if has_clean else np.zeros(0, np.uint32)
        # f4 (SPEC.md 4.8): the MD / LS graph -- nodes = MDs, CSR edges = LSs by inner MD
        self.graph = dict(rowptr=ints(12, 1, nw=22)[:, 0], col=self.ls[:, 1].copy(), node_hits=self.md_hits, node_feat=reals(12, 8, nw=1),
                          edge_c=self.ls_c)
        self.counts = dict(hits=cnt(0), md=cnt(1), ls=cnt(2), t3=cnt(3), t5c=cnt(4), t5=cnt(5), tc=cnt(6),
                           md_pairs=cnt(10), ls_pairs=cnt(11), t3_pairs=cnt(12), t5_pairs=cnt(13),
                           match5=cnt(14), match3=cnt(15))


def run(geo, weights, ev, *, t5_override=None, loosen=None, use_double=False, last_stage="clean",
        counts_only=False, dnn=(23, 2)):
    """Run the whole chain on one event.  `geo` needs n_modules, subdet, mtype, conn_rowptr, conn_col (and `layer` for the
    38-input DNN variant).  `dnn` = (n_feat, n_hidden) of SPEC.md 4.9."""
    L = lib()
    w = np.ascontiguousarray(weights, dtype=np.float32)
    ov = None if t5_override is None else np.ascontiguousarray(t5_override, dtype=np.int8)
    lo = None
    if loosen is not None:
        lo = np.ones(len(CUTS), dtype=np.float32)
        for k, v in loosen.items():
            lo[CUTS.index(k)] = v
    h = L.lst_oracle_run(int(geo.n_modules), _p(geo.subdet), _p(geo.mtype), _p(geo.conn_rowptr), _p(geo.conn_col),
                         _p(w), ev.n_hits, _p(ev.x), _p(ev.y), _p(ev.z), _p(ev.key), ev.n_pls, _p(ev.pls_px),
                         _p(ev.pls_py), _p(ev.pls_pz), _p(ev.pls_z0), _p(ev.pls_q), _p(ov),
                         0 if ov is None else int(ov.size), _p(lo), int(bool(use_double)), STAGE[last_stage],
                         int(dnn[0]), int(dnn[1]), _p(np.ascontiguousarray(geo.layer, dtype=np.uint8)) if dnn[0] == 38 else None)
    try:
        if counts_only:
            names = dict(hits=0, md=1, ls=2, t3=3, t5c=4, t5=5, tc=6, md_pairs=10, ls_pairs=11, t3_pairs=12,
                         t5_pairs=13, match5=14, match3=15)
            return {k: int(L.lst_oracle_count(h, v)) for k, v in names.items()}
        return OracleResult(h, L, int(dnn[0]))
    finally:
        L.lst_oracle_free(h)


# ---- single predicates (for the brute-force / closed-form pins) ----
def md_eval(h1, h2, subdet, mtype):
    a = np.ascontiguousarray(h1, dtype=np.float32); b = np.ascontiguousarray(h2, dtype=np.float32)
    out = np.zeros(6, dtype=np.float32)
    ok = lib().lst_oracle_md_eval(_p(a), _p(b), int(subdet), int(mtype), _p(out))
    return bool(ok), out


def ls_eval(a9, b9):
    a = np.ascontiguousarray(a9, dtype=np.float32); b = np.ascontiguousarray(b9, dtype=np.float32)
    c = np.zeros(1, dtype=np.float32)
    return bool(lib().lst_oracle_ls_eval(_p(a), _p(b), _p(c))), float(c[0])


def t3_eval(a9, b9, c9, c_ab, c_bc):
    a, b, c = (np.ascontiguousarray(v, dtype=np.float32) for v in (a9, b9, c9))
    k = np.zeros(1, dtype=np.float32)
    return bool(lib().lst_oracle_t3_eval(_p(a), _p(b), _p(c), float(c_ab), float(c_bc), _p(k))), float(k[0])


def bridge_eval(a9, b9, c9):
    a, b, c = (np.ascontiguousarray(v, dtype=np.float32) for v in (a9, b9, c9))
    k = np.zeros(1, dtype=np.float32)
    return bool(lib().lst_oracle_bridge_eval(_p(a), _p(b), _p(c), _p(k))), float(k[0])


def pls_match(pls5, q, anchors9):
    p = np.ascontiguousarray(pls5, dtype=np.float32)
    a = np.ascontiguousarray(anchors9, dtype=np.float32).reshape(-1, 9)
    chi = np.zeros(1, dtype=np.float32)
    return bool(lib().lst_oracle_pls_match(_p(p), int(q), _p(a), int(a.shape[0]), _p(chi))), float(chi[0])


def pls_residual(pls5, q, xyz):
    p = np.ascontiguousarray(pls5, dtype=np.float64); a = np.ascontiguousarray(xyz, dtype=np.float64)
    out = np.zeros(3, dtype=np.float64)
    lib().lst_oracle_pls_residual(_p(p), int(q), _p(a), _p(out))
    return out


def tc_clean(types, chi2, hits, nh):
    """SPEC.md 4.7 on hand-made candidates: types[n], chi2[n] (fp32), hits[n][10] (-1 padded), nh[n] -> keep[n]"""
    t = np.ascontiguousarray(types, dtype=np.int32); n = t.size
    q = np.ascontiguousarray(chi2, dtype=np.float32).view(np.uint32)
    h = np.ascontiguousarray(hits, dtype=np.int32).reshape(n, 10); k = np.ascontiguousarray(nh, dtype=np.int32)
    keep = np.zeros(n, dtype=np.int32)
    lib().lst_oracle_tc_clean(n, _p(t), _p(q), _p(h), _p(k), _p(keep))
    return keep


def arcfac(u, f64=False):
    return lib().lst_oracle_arcfac_f64(float(u)) if f64 else lib().lst_oracle_arcfac(float(u))


def features(ax, ay, az, ar, cin, cbr, cout):
    a = [np.ascontiguousarray(v, dtype=np.float32) for v in (ax, ay, az, ar)]
    out = np.zeros(23, dtype=np.float32)
    lib().lst_oracle_features(_p(a[0]), _p(a[1]), _p(a[2]), _p(a[3]), float(cin), float(cbr), float(cout), _p(out))
    return out


def mlp(weights, x23):
    w = np.ascontiguousarray(weights, dtype=np.float32); x = np.ascontiguousarray(x23, dtype=np.float32)
    return float(lib().lst_oracle_mlp(_p(w), _p(x)))


def mlp_n(weights, x, n_hidden):
    w = np.ascontiguousarray(weights, dtype=np.float32); x = np.ascontiguousarray(x, dtype=np.float32)
    return float(lib().lst_oracle_mlp_n(_p(w), _p(x), int(x.size), int(n_hidden)))


def features38(ax, ay, az, ar, layer, cin, cbr, cout):
    a = [np.ascontiguousarray(v, dtype=np.float32) for v in (ax, ay, az, ar)]
    lay = np.ascontiguousarray(layer, dtype=np.int32)
    out = np.zeros(38, dtype=np.float32)
    lib().lst_oracle_features38(_p(a[0]), _p(a[1]), _p(a[2]), _p(a[3]), _p(lay), float(cin), float(cbr), float(cout), _p(out))
    return out
