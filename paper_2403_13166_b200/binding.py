"""ctypes binding with the same names as include/lst.h (lst_create, lst_load_event, lst_run,
lst_get, ...).  PyTorch supplies device memory and streams only."""
import ctypes as C
import os
from dataclasses import dataclass, asdict

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBNAME = os.path.join(_HERE, "liblst_b200.so")

LST_N_CNT = 32
OBJ = dict(hit=0, md=1, ls=2, t3=3, t5c=4, t5=5, tc=6, match5=7, tcc=8, tcx=9, graph=10)
CNT = dict(hit=0, md=1, ls=2, t3=3, t5c=4, t5=5, tc=6, raw_md=7, raw_ls=8, raw_t3=9, raw_t5c=10,
           raw_t5=11, raw_tc=12, pt5=13, t5tc=14, pt3=15, plstc=16, m5_tests=17, m5_cand=18, m3_tests=19, m3_cand=20, tcc=29)
STATUS_BITS = dict(bad_key=1, ovf_md=2, ovf_ls=4, ovf_t3=8, ovf_t5c=16, ovf_t5=32, ovf_tc=64)
EXPORTS = ["lst_workspace_bytes", "lst_create", "lst_load_event", "lst_load_event_host", "lst_run",
           "lst_run_batch", "lst_run_batch_profile", "lst_launch_name", "lst_get", "lst_status", "lst_read_tc_host", "lst_load_batch_host", "lst_load_batch_host16", "lst_read_tc_batch_host", "lst_read_tc_hits_batch_host", "lst_export_graph", "lst_dnn_n_weights", "lst_measure_fp32", "lst_launches_per_run",
           "lst_destroy", "lst_sort_hits_static"]
STATIC_MAX_HITS, STATIC_MAX_MODULES = 131072, 32768      # include/lst.h LST_STATIC_MAX_*


class LstError(RuntimeError):
    pass


class _Geometry(C.Structure):
    _fields_ = [("n_modules", C.c_int32), ("subdet", C.c_void_p), ("mtype", C.c_void_p),
                ("conn_rowptr", C.c_void_p), ("conn_col", C.c_void_p), ("dnn_weights", C.c_void_p),
                ("layer", C.c_void_p), ("dnn_n_feat", C.c_int32), ("dnn_n_hidden", C.c_int32)]


class _Caps(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("n_slots", "max_hits", "max_md", "max_ls", "max_t3", "max_t5c",
                                         "max_t5", "max_pls")]


class _View(C.Structure):
    _fields_ = [("capacity", C.c_int32), ("count", C.c_void_p), ("i0", C.c_void_p), ("i1", C.c_void_p),
                ("i2", C.c_void_p), ("f0", C.c_void_p), ("f1", C.c_void_p), ("f2", C.c_void_p)]


@dataclass
class Caps:
    n_slots: int = 1
    max_hits: int = 131072
    max_md: int = 65536
    max_ls: int = 65536
    max_t3: int = 65536
    max_t5c: int = 65536
    max_t5: int = 65536
    max_pls: int = 8192


def default_caps(n_slots: int = 1) -> Caps:
    """Capacities sized for configs[4]'s densest point (PU300 + 500 displaced) with head-room."""
    return Caps(n_slots=n_slots)


def library_path() -> str:
    return _LIBNAME


_lib = None


def load_library():
    """Load liblst_b200.so; raises LstError when it has not been built (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIBNAME):
        raise LstError(f"{_LIBNAME} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                       "(nvcc, sm_100a). There is no CPU fallback.")
    L = C.CDLL(_LIBNAME)
    vp, i32 = C.c_void_p, C.c_int32
    L.lst_workspace_bytes.argtypes = [C.POINTER(_Geometry), C.POINTER(_Caps), C.POINTER(C.c_size_t)]
    L.lst_create.argtypes = [C.POINTER(_Geometry), C.POINTER(_Caps), vp, C.c_size_t, C.POINTER(vp)]
    L.lst_load_event.argtypes = [vp, i32, i32, vp, vp, vp, vp, i32, vp, vp, vp, vp, vp, vp]
    L.lst_load_event_host.argtypes = L.lst_load_event.argtypes
    L.lst_run.argtypes = [vp, i32, vp]
    L.lst_run_batch.argtypes = [vp, i32, i32, vp]
    L.lst_get.argtypes = [vp, i32, i32, C.POINTER(_View)]
    L.lst_status.argtypes = [vp, i32, C.POINTER(C.c_uint32), vp, vp]
    L.lst_read_tc_host.argtypes = [vp, i32, vp, vp, i32, vp]
    L.lst_load_batch_host.argtypes = [vp, i32, i32, vp, C.c_size_t, vp]
    L.lst_load_batch_host16.argtypes = [vp, i32, i32, vp, C.c_size_t, vp]
    L.lst_read_tc_batch_host.argtypes = [vp, i32, i32, vp, i32, vp]
    L.lst_read_tc_hits_batch_host.argtypes = [vp, i32, i32, vp, i32, vp]
    L.lst_measure_fp32.argtypes = [vp, i32, C.POINTER(C.c_float), vp]
    L.lst_export_graph.argtypes = [vp, i32, i32, vp]
    L.lst_dnn_n_weights.argtypes = [i32, i32]
    L.lst_launches_per_run.argtypes = []
    L.lst_run_batch_profile.argtypes = [vp, i32, i32, vp, vp]
    L.lst_launch_name.argtypes = [i32]
    L.lst_destroy.argtypes = [vp]
    L.lst_sort_hits_static.argtypes = [i32, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    L.lst_destroy.restype = None
    for n in EXPORTS:
        if n not in ("lst_destroy", "lst_launch_name"):
            getattr(L, n).restype = C.c_int
    L.lst_launch_name.restype = C.c_char_p
    _lib = L
    return L


def _chk(rc, what):
    if rc != 0:
        raise LstError(f"{what} failed with code {rc} "
                       f"({ {-1: 'LST_EINVAL', -2: 'LST_ECUDA', -3: 'LST_ENOMEM', -4: 'LST_ETOOBIG'}.get(rc, '?') })")


def _hp(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


# rows, dtype, columns of every view field (include/lst.h lst_view)
_FIELDS = {
    "hit": dict(i0=("orig", "i32", 1), f0=("xyzr", "f32", 4)),
    "md": dict(i0=("hits", "i32", 2), i1=("modt", "i32", 1), f0=("anchor", "f32", 4), f1=("cw", "f32", 2)),
    "ls": dict(i0=("ab", "i32", 2), f0=("c", "f32", 1)),
    "t3": dict(i0=("abc", "i32", 4), i1=("l1", "i32", 1), f0=("k", "f32", 1)),
    "t5c": dict(i0=("md", "i32", 5), i1=("t3", "i32", 2), i2=("pass", "i32", 1), f0=("curv", "f32", 3),
                f1=("feat", "f32", 23), f2=("score", "f32", 1)),
    "t5": dict(i0=("cand", "i32", 1)),
    "tc": dict(i0=("tc", "i32", 3)),
    "match5": dict(i0=("best5_pls", "i32", 1), f0=("chi2", "f32", 1)),
    "tcc": dict(i0=("tc", "i32", 3)),
    "tcx": dict(i0=("keep", "i32", 1), i1=("hits", "i32", 12), i2=("q", "i32", 1)),
}
_ROWS = {"match5": "t5", "tcx": "tc"}      # views whose row count is another list's count


class LST:
    """One context = one uploaded geometry + `caps.n_slots` event slots in a torch-owned workspace."""

    def __init__(self, geo, weights, caps: Caps = None, device="cuda:0", dnn=(23, 2)):
        import torch
        self.torch = torch
        self.lib = load_library()
        self.caps = caps or default_caps()
        self.device = torch.device(device)
        self.n_modules = int(geo.n_modules)
        self._keep = dict(subdet=np.ascontiguousarray(geo.subdet, np.uint8), mtype=np.ascontiguousarray(geo.mtype, np.uint8),
                          rowptr=np.ascontiguousarray(geo.conn_rowptr, np.int32), col=np.ascontiguousarray(geo.conn_col, np.int32),
                          w=np.ascontiguousarray(weights, np.float32))
        self.n_feat, self.n_hidden = int(dnn[0]), int(dnn[1])
        if self._keep["w"].size != self.lib.lst_dnn_n_weights(self.n_feat, self.n_hidden):
            raise LstError(f"dnn_weights must hold {self.lib.lst_dnn_n_weights(self.n_feat, self.n_hidden)} floats for this DNN variant")
        k = self._keep
        k["layer"] = np.ascontiguousarray(geo.layer, np.uint8) if getattr(geo, "layer", None) is not None else None
        self._g = _Geometry(self.n_modules, _hp(k["subdet"]), _hp(k["mtype"]), _hp(k["rowptr"]), _hp(k["col"]), _hp(k["w"]),
                            _hp(k["layer"]), self.n_feat, self.n_hidden)
        self._c = _Caps(**asdict(self.caps))
        nbytes = C.c_size_t(0)
        _chk(self.lib.lst_workspace_bytes(C.byref(self._g), C.byref(self._c), C.byref(nbytes)), "lst_workspace_bytes")
        self.workspace_bytes = int(nbytes.value)
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(self.workspace_bytes + 256, dtype=torch.uint8, device=self.device)
            base = self.workspace.data_ptr()
            self._ws_off = (-base) % 256
            self._ws_ptr = base + self._ws_off
            ctx = C.c_void_p()
            _chk(self.lib.lst_create(C.byref(self._g), C.byref(self._c), C.c_void_p(self._ws_ptr), nbytes, C.byref(ctx)), "lst_create")
        self.ctx = ctx
        self._bound = {}

    # ---- entry points, same names as the C ABI -------------------------------------------------
    def lst_load_event(self, slot, x, y, z, key, px, py, pz, z0, q, stream=None):
        """Bind DEVICE tensors (float32 / int32-as-uint32 / int8) to a slot; they are not copied."""
        t = self.torch
        for a, dt in ((x, t.float32), (y, t.float32), (z, t.float32), (px, t.float32), (py, t.float32), (pz, t.float32), (z0, t.float32)):
            assert a.is_cuda and a.dtype == dt and a.is_contiguous()
        assert key.is_cuda and key.dtype in (t.int32, t.uint32) and key.is_contiguous()
        assert q.is_cuda and q.dtype == t.int8 and q.is_contiguous()
        self._bound[slot] = (x, y, z, key, px, py, pz, z0, q)
        p = lambda a: C.c_void_p(a.data_ptr()) if a.numel() else C.c_void_p(0)
        _chk(self.lib.lst_load_event(self.ctx, slot, x.numel(), p(x), p(y), p(z), p(key), px.numel(), p(px), p(py), p(pz), p(z0), p(q),
                                     self._st(stream)), "lst_load_event")

    def lst_load_event_host(self, slot, hx, hy, hz, hkey, hpx, hpy, hpz, hz0, hq, stream=None):
        """HOST (ideally pinned) torch tensors or numpy arrays; enqueues the H2D copies."""
        arrs = (hx, hy, hz, hkey, hpx, hpy, hpz, hz0, hq)
        self._bound[slot] = arrs
        def p(a):
            if hasattr(a, "data_ptr"):
                return C.c_void_p(a.data_ptr()) if a.numel() else C.c_void_p(0)
            return _hp(a) if a.size else C.c_void_p(0)
        n = lambda a: int(a.numel()) if hasattr(a, "numel") else int(a.size)
        _chk(self.lib.lst_load_event_host(self.ctx, slot, n(hx), p(hx), p(hy), p(hz), p(hkey), n(hpx), p(hpx), p(hpy), p(hpz), p(hz0), p(hq),
                                          self._st(stream)), "lst_load_event_host")

    def lst_run(self, slot=0, stream=None):
        _chk(self.lib.lst_run(self.ctx, slot, self._st(stream)), "lst_run")

    def lst_run_batch(self, first_slot, n, stream=None):
        _chk(self.lib.lst_run_batch(self.ctx, first_slot, n, self._st(stream)), "lst_run_batch")

    def lst_status(self, slot=0, stream=None):
        bits = C.c_uint32(0)
        counts = np.zeros(LST_N_CNT, dtype=np.int32)
        _chk(self.lib.lst_status(self.ctx, slot, C.byref(bits), _hp(counts), self._st(stream)), "lst_status")
        return int(bits.value), {k: int(counts[v]) for k, v in CNT.items()}

    def lst_get(self, slot, objtype, n=None):
        """Device views (torch tensors aliasing the workspace) of one object list; `n` rows
        (default: the clamped count, which costs a synchronising lst_status)."""
        name = objtype if isinstance(objtype, str) else {v: k for k, v in OBJ.items()}[objtype]
        v = _View()
        _chk(self.lib.lst_get(self.ctx, slot, OBJ[name], C.byref(v)), "lst_get")
        if n is None:
            _, cnt = self.lst_status(slot)
            n = cnt[_ROWS.get(name, name)]
        out = {}
        t = self.torch
        for fld, (label, dt, cols) in _FIELDS[name].items():
            if label == "feat":
                cols = self.n_feat
            ptr = getattr(v, fld)
            off = ptr - self.workspace.data_ptr()
            raw = self.workspace[off:off + 4 * n * cols]
            out[label] = raw.view(t.int32 if dt == "i32" else t.float32).view(n, cols) if cols > 1 else \
                raw.view(t.int32 if dt == "i32" else t.float32)
        return out

    def ranges(self, slot, counts=None):
        """Device views of the range tables: sensor_start[2M+1], md_start[M+1], ls_start[n_md+1],
        t3_start[n_md+1] (include/lst.h lst_view i1 / i2 entries)."""
        if counts is None:
            _, counts = self.lst_status(slot)
        t, M = self.torch, self.n_modules
        out = {}
        for label, obj, fld, n in (("sensor_start", "hit", "i1", 2 * M + 1), ("md_start", "md", "i2", M + 1),
                                   ("ls_start", "ls", "i1", counts["md"] + 1), ("t3_start", "t3", "i2", counts["md"] + 1)):
            v = _View()
            _chk(self.lib.lst_get(self.ctx, slot, OBJ[obj], C.byref(v)), "lst_get")
            off = getattr(v, fld) - self.workspace.data_ptr()
            out[label] = self.workspace[off:off + 4 * n].view(t.int32)
        return out

    def lst_read_tc_host(self, slot, h_counts, h_tc, stream=None):
        """Enqueue D2H of counters and TC rows into HOST (pinned) int32 tensors."""
        _chk(self.lib.lst_read_tc_host(self.ctx, slot, C.c_void_p(h_counts.data_ptr()), C.c_void_p(h_tc.data_ptr()),
                                       int(h_tc.shape[0]), self._st(stream)), "lst_read_tc_host")

    def lst_load_batch_host(self, first_slot, n, h_blob, stream=None):
        """h_blob: HOST (pinned) uint8 tensor packed as include/lst.h describes (see pack_batch)."""
        _chk(self.lib.lst_load_batch_host(self.ctx, first_slot, n, C.c_void_p(h_blob.data_ptr()), C.c_size_t(h_blob.numel()),
                                          self._st(stream)), "lst_load_batch_host")

    def lst_load_batch_host16(self, first_slot, n, h_blob, stream=None):
        """h_blob: HOST (pinned) uint8 tensor packed with 16-bit sensor keys (see pack_batch(..., key16=True))."""
        _chk(self.lib.lst_load_batch_host16(self.ctx, first_slot, n, C.c_void_p(h_blob.data_ptr()), C.c_size_t(h_blob.numel()),
                                            self._st(stream)), "lst_load_batch_host16")

    def lst_read_tc_batch_host(self, first_slot, n, h_out, stream=None):
        """h_out: HOST (pinned) int32 tensor [n, 32 + 3*max_rows]."""
        rows = (int(h_out.shape[1]) - LST_N_CNT) // 3
        _chk(self.lib.lst_read_tc_batch_host(self.ctx, first_slot, n, C.c_void_p(h_out.data_ptr()), rows, self._st(stream)),
             "lst_read_tc_batch_host")

    def lst_read_tc_hits_batch_host(self, first_slot, n, h_out, stream=None):
        """h_out: HOST (pinned) int32 tensor [n, 32 + 13*max_rows]: rows = (type, pLS, object, 10 original hit indices)."""
        rows = (int(h_out.shape[1]) - LST_N_CNT) // 13
        _chk(self.lib.lst_read_tc_hits_batch_host(self.ctx, first_slot, n, C.c_void_p(h_out.data_ptr()), rows, self._st(stream)),
             "lst_read_tc_hits_batch_host")

    def lst_export_graph(self, first_slot, n, stream=None):
        _chk(self.lib.lst_export_graph(self.ctx, first_slot, n, self._st(stream)), "lst_export_graph")

    def fetch_graph(self, slot):
        """MD / LS graph of a slot as numpy arrays (after lst_export_graph): rowptr, col, node_hits, node_feat, edge_c."""
        _, cnt = self.lst_status(slot)
        v = _View()
        _chk(self.lib.lst_get(self.ctx, slot, OBJ["graph"], C.byref(v)), "lst_get")
        t = self.torch
        def view(ptr, n, dt):
            off = ptr - self.workspace.data_ptr()
            return self.workspace[off:off + 4 * n].view(dt).cpu().numpy()
        n_md, n_ls = cnt["md"], cnt["ls"]
        return dict(rowptr=view(v.i0, n_md + 1, t.int32), col=view(v.i1, n_ls, t.int32), node_hits=view(v.i2, 2 * n_md, t.int32).reshape(n_md, 2),
                    node_feat=view(v.f0, 8 * n_md, t.float32).reshape(n_md, 8), edge_c=view(v.f1, n_ls, t.float32))

    def lst_measure_fp32(self, fused, stream=None):
        """Sustained fp32 Tflop/s of this GPU: separately rounded multiply + add (fused=False) or FMA (fused=True)."""
        v = C.c_float(0.0)
        _chk(self.lib.lst_measure_fp32(self.ctx, int(bool(fused)), C.byref(v), self._st(stream)), "lst_measure_fp32")
        return float(v.value)

    def lst_run_batch_profile(self, first_slot, n, stream=None):
        """Per-launch device times in ms: dict name -> ms (memset + every kernel of one pass)."""
        k = self.launches_per_run() + 1
        ms = np.zeros(k, dtype=np.float32)
        _chk(self.lib.lst_run_batch_profile(self.ctx, first_slot, n, self._st(stream), _hp(ms)), "lst_run_batch_profile")
        return {self.lib.lst_launch_name(i).decode(): float(ms[i]) for i in range(k)}

    def launches_per_run(self):
        return int(self.lib.lst_launches_per_run())

    def close(self):
        if getattr(self, "ctx", None):
            self.lib.lst_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- conveniences --------------------------------------------------------------------------
    def _st(self, stream):
        if stream is None:
            stream = self.torch.cuda.current_stream(self.device)
        return C.c_void_p(stream.cuda_stream)

    def load_numpy_event(self, slot, ev, stream=None):
        """Upload a lstgen.Event's arrays with torch and bind them (tests / smoke)."""
        t = self.torch
        dev = lambda a: t.from_numpy(np.ascontiguousarray(a)).to(self.device)
        key = t.from_numpy(ev.key.view(np.int32).copy()).to(self.device)
        self.lst_load_event(slot, dev(ev.x), dev(ev.y), dev(ev.z), key, dev(ev.pls_px), dev(ev.pls_py), dev(ev.pls_pz),
                            dev(ev.pls_z0), dev(ev.pls_q), stream)

    def fetch(self, slot):
        """Copy every object list of a slot to numpy (one synchronising status call)."""
        bits, cnt = self.lst_status(slot)
        res = dict(status=bits, counts=cnt)
        for name in _FIELDS:
            n = cnt[_ROWS.get(name, name)]
            res[name] = {k: v.cpu().numpy() for k, v in self.lst_get(slot, name, n).items()}
        return res


def lst_sort_hits_static(x, y, z, key, n_modules, hit_xyzr, hit_orig, sensor_start, count, stream=None):
    """Step a0 (hits sorted by sensor, stable) for callers that cannot allocate device memory -- e.g. a module inside a
    framework that owns all of it and only hands out input / output buffers, or an event loop where cudaMalloc is banned.
    No context and no workspace: the temporaries live in a fixed array inside the library, so the call is limited to
    STATIC_MAX_HITS hits and STATIC_MAX_MODULES modules (LstError naming the limits otherwise), and calls that overlap
    on one GPU would corrupt each other -- keep them on one stream.  The device of the tensors must be current; make the
    first call on a device outside any stream capture (include/lst.h has the details).

    DEVICE tensors in: x, y, z float32 [n]; key int32/uint32 [n].  DEVICE tensors out (caller-provided): hit_xyzr float32
    [n, 4], hit_orig int32 [n], sensor_start int32 [2 * n_modules + 1], count int32 [2] = (hits kept, status bits).
    Enqueues on `stream` (default: torch's current stream); argument marshalling only."""
    import torch as t
    L = load_library()
    n = int(x.numel())
    for a in (x, y, z):
        assert a.is_cuda and a.dtype == t.float32 and a.is_contiguous() and a.numel() == n
    assert key.is_cuda and key.dtype in (t.int32, t.uint32) and key.is_contiguous() and key.numel() == n
    assert hit_xyzr.is_cuda and hit_xyzr.dtype == t.float32 and hit_xyzr.is_contiguous() and hit_xyzr.numel() >= 4 * n
    assert hit_orig.is_cuda and hit_orig.dtype == t.int32 and hit_orig.is_contiguous() and hit_orig.numel() >= n
    assert sensor_start.is_cuda and sensor_start.dtype == t.int32 and sensor_start.is_contiguous() and sensor_start.numel() >= 2 * n_modules + 1
    assert count.is_cuda and count.dtype == t.int32 and count.numel() >= 2
    if stream is None:
        stream = t.cuda.current_stream(x.device)
    p = lambda a: C.c_void_p(a.data_ptr()) if a.numel() else C.c_void_p(0)
    rc = L.lst_sort_hits_static(n, int(n_modules), p(x), p(y), p(z), p(key), p(hit_xyzr), p(hit_orig), p(sensor_start), p(count),
                                C.c_void_p(stream.cuda_stream))
    if rc == -4:
        raise LstError(f"lst_sort_hits_static: {n} hits / {n_modules} modules exceed the built-in scratch "
                       f"(at most {STATIC_MAX_HITS} hits and {STATIC_MAX_MODULES} modules); use LST with a workspace instead")
    _chk(rc, "lst_sort_hits_static")


def pack_batch(events, pin=True, key16=False):
    """Pack events (objects with x, y, z, key, pls_px, pls_py, pls_pz, pls_z0, pls_q numpy arrays) into the blob
    layout of lst_load_batch_host (key16=False) or lst_load_batch_host16 (key16=True): argument marshalling only."""
    import torch
    n = len(events)
    hdr = (8 * n + 15) // 16 * 16
    kb = lambda nh: (2 * nh + 3) // 4 * 4 if key16 else 4 * nh
    sizes = [((12 * ev.x.size + kb(ev.x.size) + 17 * ev.pls_px.size + 15) // 16) * 16 for ev in events]
    blob = torch.zeros(hdr + sum(sizes), dtype=torch.uint8)
    if pin:
        blob = blob.pin_memory()
    b = blob.numpy()
    desc = b[:8 * n].view(np.int32)
    off = hdr
    for i, ev in enumerate(events):
        nh, npl = int(ev.x.size), int(ev.pls_px.size)
        desc[2 * i], desc[2 * i + 1] = nh, npl
        f = b[off:off + 12 * nh].view(np.float32)
        f[0:nh], f[nh:2 * nh], f[2 * nh:3 * nh] = ev.x, ev.y, ev.z
        if key16:
            b[off + 12 * nh:off + 14 * nh].view(np.uint16)[:] = ev.key.astype(np.uint16)
        else:
            b[off + 12 * nh:off + 16 * nh].view(np.uint32)[:] = ev.key
        o2 = off + 12 * nh + kb(nh)
        g = b[o2:o2 + 16 * npl].view(np.float32)
        g[0:npl], g[npl:2 * npl], g[2 * npl:3 * npl], g[3 * npl:4 * npl] = ev.pls_px, ev.pls_py, ev.pls_pz, ev.pls_z0
        b[o2 + 16 * npl:o2 + 17 * npl] = ev.pls_q.view(np.uint8)
        off += sizes[i]
    return blob
