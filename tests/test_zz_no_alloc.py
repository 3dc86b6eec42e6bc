"""lst_sort_hits_static: the a0 hit ingest for callers that cannot allocate device memory.

Some users of the library sit inside a host framework that owns all device memory and hands a module nothing but its
input and output buffers (a trigger / event-processing job), or run in an event loop where cudaMalloc is banned because
it stalls the whole device.  They cannot supply the workspace every other entry point needs, so this one keeps its
temporaries in a fixed array built into the library.  That array is shared by all calls and keeps the last call's
contents, which is exactly what could go wrong: the GPU test therefore makes TWO calls in a row on different events
(a large one, then a smaller one with out-of-range keys) and compares each, bit for bit, with what the existing path
(lst_load_event + lst_run, LST_OBJ_HIT view) produces for the same event.

The file is named test_zz_* so that pytest collects it last: `pytest -x` stops at the first failure, and a failure
here must not hide any other test.  It passes on its own in a fresh process and after the rest of the suite."""
import ctypes as C
import os
import numpy as np
import pytest

from lstgen import config_event


def _lib():
    import __graft_entry__ as ge
    ge.build()
    import paper_2403_13166_b200 as P
    return P, P.load_library()


def test_sizes_beyond_the_built_in_scratch_are_refused():
    """No GPU needed: the limits are checked before any CUDA call.  The C function returns LST_ETOOBIG (-4) and the
    Python wrapper's message names the limits, so a caller learns why and what to use instead."""
    P, L = _lib()
    from paper_2403_13166_b200.binding import STATIC_MAX_HITS, STATIC_MAX_MODULES
    dummy = C.c_void_p(256)      # never dereferenced: the size check comes first
    args = (dummy,) * 8 + (C.c_void_p(0),)
    assert L.lst_sort_hits_static(STATIC_MAX_HITS + 1, 100, *args) == -4
    assert L.lst_sort_hits_static(10, STATIC_MAX_MODULES + 1, *args) == -4
    assert L.lst_sort_hits_static(-1, 100, *args) == -1
    assert L.lst_sort_hits_static(10, 0, *args) == -1
    assert L.lst_sort_hits_static(10, 100, *((C.c_void_p(0),) * 9)) == -1          # null outputs
    hdr = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "lst.h")).read()
    assert f"#define LST_STATIC_MAX_HITS {STATIC_MAX_HITS}" in hdr and f"#define LST_STATIC_MAX_MODULES {STATIC_MAX_MODULES}" in hdr


def _existing_path(P, geo, w, ev):
    """a0 through the workspace-based chain: (hits kept, status & BAD_KEY, orig, xyzr, sensor_start)."""
    lst = P.LST(geo, w, P.default_caps(1))
    lst.load_numpy_event(0, ev)
    lst.lst_run(0)
    bits, cnt = lst.lst_status(0)
    n = cnt["hit"]
    v = lst.lst_get(0, "hit", n)
    res = (n, bits & P.STATUS_BITS["bad_key"], v["orig"].cpu().numpy().copy(), v["xyzr"].cpu().numpy().copy(),
           lst.ranges(0, cnt)["sensor_start"].cpu().numpy().copy())
    lst.close()
    return res


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_existing_path(geo_full):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    P, _ = _lib()
    from lstgen import xavier_weights
    geo, w = geo_full, xavier_weights(2)
    big = config_event(geo, 2)                       # PU200: ~77 k hits, most sensors occupied
    small = config_event(geo, 1)                     # PU50, and some keys out of range: those hits are dropped and flagged
    small.key = small.key.copy()
    small.key[::97] = 2 * geo.n_modules + 5
    M = int(geo.n_modules)
    dev = torch.device("cuda:0")
    count = torch.empty(2, dtype=torch.int32, device=dev)
    for ev in (big, small, big):                     # the third call runs on what the smaller event left behind
        n = int(ev.x.size)
        x, y, z = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (ev.x, ev.y, ev.z))
        key = torch.from_numpy(ev.key.view(np.int32).copy()).to(dev)
        xyzr = torch.full((n, 4), float("nan"), dtype=torch.float32, device=dev)
        orig = torch.full((n,), -7, dtype=torch.int32, device=dev)
        start = torch.full((2 * M + 1,), -7, dtype=torch.int32, device=dev)
        P.lst_sort_hits_static(x, y, z, key, M, xyzr, orig, start, count)
        torch.cuda.synchronize()
        kept, status = (int(v) for v in count.cpu().numpy())
        n_ref, bad_ref, orig_ref, xyzr_ref, start_ref = _existing_path(P, geo, w, ev)
        assert kept == n_ref and (status & P.STATUS_BITS["bad_key"]) == bad_ref
        assert (bad_ref != 0) == (ev is small)
        # integer outputs and the float rows are the same bytes as the existing path's (same arithmetic for r)
        assert np.array_equal(start.cpu().numpy(), start_ref)
        assert np.array_equal(orig.cpu().numpy()[:kept], orig_ref)
        assert np.array_equal(xyzr.cpu().numpy()[:kept].view(np.int32), xyzr_ref.view(np.int32))
        assert (orig.cpu().numpy()[kept:] == -7).all()          # rows past the kept hits are not touched


@pytest.mark.gpu
def test_empty_event(geo_barrel):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    P, _ = _lib()
    M = int(geo_barrel.n_modules)
    dev = torch.device("cuda:0")
    e = lambda dt: torch.empty(0, dtype=dt, device=dev)
    start = torch.full((2 * M + 1,), -7, dtype=torch.int32, device=dev)
    count = torch.full((2,), -7, dtype=torch.int32, device=dev)
    P.lst_sort_hits_static(e(torch.float32), e(torch.float32), e(torch.float32), e(torch.int32), M,
                           torch.empty((0, 4), dtype=torch.float32, device=dev), e(torch.int32), start, count)
    torch.cuda.synchronize()
    assert (start.cpu().numpy() == 0).all() and count.cpu().tolist() == [0, 0]
