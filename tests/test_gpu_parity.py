"""Parity of the CUDA path (through the C ABI) against the CPU oracle.  `-m gpu` only."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from lstgen import build_geometry, make_event, config_event, xavier_weights
import parity


@pytest.fixture(scope="module")
def P():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2403_13166_b200 as P
    P.load_library()      # fails loudly if the extension is missing
    return P


def _run_one(P, geo, w, ev, caps=None):
    lst = P.LST(geo, w, caps or P.default_caps(1))
    lst.load_numpy_event(0, ev)
    lst.lst_run(0)
    out = lst.fetch(0)
    lst.close()
    return out


def test_config0_barrel_toy(P, geo_barrel):
    w = xavier_weights(1)
    ev = config_event(geo_barrel, 0)
    c = parity.compare(geo_barrel, w, ev, _run_one(P, geo_barrel, w, ev))
    assert c["md"] == 60 and c["t5c"] == 20


def test_config1_pu50(P, geo_full):
    w = xavier_weights(2)
    ev = config_event(geo_full, 1)
    c = parity.compare(geo_full, w, ev, _run_one(P, geo_full, w, ev))
    assert c["t5c"] > 500


def test_config2_pu200_headline(P, geo_full):
    w = xavier_weights(3)
    ev = config_event(geo_full, 2)
    c = parity.compare(geo_full, w, ev, _run_one(P, geo_full, w, ev))
    assert c["md"] > 10000 and c["tc"] > 2000


@pytest.mark.parametrize("pileup", [0, 100, 200, 300])
def test_config4_displaced_stress(P, geo_full, pileup):
    w = xavier_weights(3)
    ev = config_event(geo_full, 4, seed=200 + pileup // 100, pileup=pileup)
    out = _run_one(P, geo_full, w, ev)
    assert out["status"] == 0
    parity.compare(geo_full, w, ev, out)


def test_biased_weights_balanced_decisions(P, geo_full):
    """Weights with biases put many scores on both sides of 0.5, so the decision comparison bites."""
    w = xavier_weights(5, bias_scale=0.5)
    w[-1] = -0.6
    ev = config_event(geo_full, 2, seed=77)
    out = _run_one(P, geo_full, w, ev)
    frac = out["t5c"]["pass"].mean()
    assert 0.05 < frac < 0.95
    parity.compare(geo_full, w, ev, out)


def test_empty_and_degenerate_events(P, geo_full):
    w = xavier_weights(3)
    ev = make_event(geo_full, 9)                                  # no hits, no pLS
    out = _run_one(P, geo_full, w, ev)
    assert out["status"] == 0 and all(out["counts"][k] == 0 for k in ("hit", "md", "ls", "t3", "t5c", "t5", "tc"))
    ev = make_event(geo_full, 9, n_noise=500)                     # hits but nothing to build, no pLS
    parity.compare(geo_full, w, ev, _run_one(P, geo_full, w, ev))
    ev = config_event(geo_full, 1, seed=12)                       # pLS only: every seed becomes a pLS candidate
    ev.x = ev.x[:0]; ev.y = ev.y[:0]; ev.z = ev.z[:0]; ev.key = ev.key[:0]
    out = _run_one(P, geo_full, w, ev)
    assert out["counts"]["plstc"] == ev.n_pls == out["counts"]["tc"]
    parity.compare(geo_full, w, ev, out)


def test_bad_key_is_flagged(P, geo_full):
    w = xavier_weights(3)
    ev = config_event(geo_full, 1, seed=13)
    ev.key[5] = 2 * geo_full.n_modules
    ev.key[9] = 0xFFFFFFFF
    out = _run_one(P, geo_full, w, ev)
    assert out["status"] & P.STATUS_BITS["bad_key"]
    assert out["counts"]["hit"] == ev.n_hits - 2
    parity.compare(geo_full, w, ev, out)


def test_every_overflow_flag(P, geo_full):
    """configs[4]: shrink each capacity in turn; the stage keeps the first `cap` objects in build
    order, flags the overflow and reports the unclamped total."""
    from oracle import lst_oracle as O
    w = xavier_weights(3)
    ev = config_event(geo_full, 1)
    ref = O.run(geo_full, w, ev)
    full = dict(max_md=ref.counts["md"], max_ls=ref.counts["ls"], max_t3=ref.counts["t3"], max_t5c=ref.counts["t5c"], max_t5=ref.counts["t5"])
    for name, bit, cnt in [("max_md", "ovf_md", "md"), ("max_ls", "ovf_ls", "ls"), ("max_t3", "ovf_t3", "t3"),
                           ("max_t5c", "ovf_t5c", "t5c"), ("max_t5", "ovf_t5", "t5")]:
        kw = dict(n_slots=1, max_hits=32768, max_pls=2048, max_md=16384, max_ls=16384, max_t3=16384, max_t5c=16384, max_t5=16384)
        kw[name] = full[name] // 2
        out = _run_one(P, geo_full, w, ev, P.Caps(**kw))
        assert out["status"] & P.STATUS_BITS[bit], name
        assert out["counts"][cnt] == kw[name] and out["counts"]["raw_" + cnt] == full[name]
        if name == "max_md":
            assert np.array_equal(out["md"]["hits"], ref.md_hits[:kw[name]])
        if name == "max_ls":
            assert np.array_equal(out["ls"]["ab"], ref.ls[:kw[name]])
        if name == "max_t3":          # the first cap objects in build order, as include/lst.h promises
            assert np.array_equal(out["t3"]["abc"][:, :3], ref.t3[:kw[name], :3]) and np.array_equal(out["t3"]["l1"], ref.t3[:kw[name], 4])
        if name == "max_t5c":
            assert np.array_equal(out["t5c"]["md"], ref.t5c[:kw[name], :5])
        if name == "max_t5":
            assert np.array_equal(out["t5"]["cand"], ref.t5[:kw[name]])
        # LST_ST_OVF_TC cannot occur: the TC capacity is max_pls + max_t5 and the list holds at most one row per pLS and T5
        assert not out["status"] & P.STATUS_BITS["ovf_tc"]
    # exact fit: no flag
    kw = dict(n_slots=1, max_hits=ev.n_hits, max_pls=ev.n_pls, **full)
    out = _run_one(P, geo_full, w, ev, P.Caps(**kw))
    assert out["status"] == 0
    parity.compare(geo_full, w, ev, out)


def test_batch_equals_single_and_is_deterministic(P, geo_full):
    """configs[3] in small: a batched launch over several slots = each event alone; repeated runs
    give identical bytes."""
    import torch
    w = xavier_weights(3)
    evs = [config_event(geo_full, 2, seed=100 + i) for i in range(4)] + [make_event(geo_full, 1), config_event(geo_full, 1, seed=5)]
    lst = P.LST(geo_full, w, P.default_caps(len(evs)))
    for i, ev in enumerate(evs):
        lst.load_numpy_event(i, ev)
    lst.lst_run_batch(0, len(evs))
    first = [lst.fetch(i) for i in range(len(evs))]
    for i, ev in enumerate(evs):
        parity.compare(geo_full, w, ev, first[i])
    for _ in range(3):
        lst.lst_run_batch(0, len(evs))
        again = [lst.fetch(i) for i in range(len(evs))]
        for a, b in zip(first, again):
            for obj in ("md", "ls", "t3", "t5c", "t5", "tc", "match5"):
                for k in a[obj]:
                    assert np.array_equal(a[obj][k].view(np.int32) if a[obj][k].dtype == np.float32 else a[obj][k],
                                          b[obj][k].view(np.int32) if b[obj][k].dtype == np.float32 else b[obj][k]), (obj, k)
    # streams: two halves on two streams
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    lst.lst_run_batch(0, 3, s1); lst.lst_run_batch(3, 3, s2)
    torch.cuda.synchronize()
    for i, ev in enumerate(evs):
        parity.compare(geo_full, w, ev, lst.fetch(i))
    lst.close()


def test_host_load_path(P, geo_full):
    import torch
    w = xavier_weights(2)
    ev = config_event(geo_full, 1, seed=21)
    lst = P.LST(geo_full, w, P.default_caps(1))
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    args = [pin(ev.x), pin(ev.y), pin(ev.z), pin(ev.key.view(np.int32)), pin(ev.pls_px), pin(ev.pls_py), pin(ev.pls_pz), pin(ev.pls_z0), pin(ev.pls_q)]
    lst.lst_load_event_host(0, *args)
    lst.lst_run(0)
    h_cnt = torch.zeros(32, dtype=torch.int32).pin_memory()
    h_tc = torch.zeros((lst.caps.max_pls + lst.caps.max_t5, 3), dtype=torch.int32).pin_memory()
    lst.lst_read_tc_host(0, h_cnt, h_tc)
    torch.cuda.synchronize()
    out = lst.fetch(0)
    parity.compare(geo_full, w, ev, out)
    n = int(h_cnt[P.CNT["tc"]])
    assert n == out["counts"]["tc"] and np.array_equal(h_tc[:n].numpy(), out["tc"]["tc"].reshape(-1, 3))
    lst.close()


def test_packed_host_buffers_single_copies(P, geo_full):
    """lst_load_event_host / lst_read_tc_host with adjacent host arrays ([x|y|z|key], [px|py|pz|z0|q], counters +
    TC rows in one buffer) take the single-transfer path (include/lst.h); the result is the same event."""
    import torch
    w = xavier_weights(3)
    ev = config_event(geo_full, 1)
    lst = P.LST(geo_full, w, P.default_caps(1), device="cuda:0")
    n, m = ev.n_hits, ev.n_pls
    hb = torch.empty(4 * n, dtype=torch.float32).pin_memory()
    hn = hb.numpy()
    hn[0:n], hn[n:2 * n], hn[2 * n:3 * n] = ev.x, ev.y, ev.z
    hn[3 * n:4 * n] = ev.key.view(np.float32)
    pb = torch.empty(17 * m, dtype=torch.uint8).pin_memory()
    pf = pb[:16 * m].view(torch.float32).numpy()
    pf[0:m], pf[m:2 * m], pf[2 * m:3 * m], pf[3 * m:4 * m] = ev.pls_px, ev.pls_py, ev.pls_pz, ev.pls_z0
    pb[16 * m:].numpy()[:] = ev.pls_q.view(np.uint8)
    lst.lst_load_event_host(0, hb[0:n], hb[n:2 * n], hb[2 * n:3 * n], hb[3 * n:4 * n].view(torch.int32),
                            pb[0:4 * m].view(torch.float32), pb[4 * m:8 * m].view(torch.float32), pb[8 * m:12 * m].view(torch.float32),
                            pb[12 * m:16 * m].view(torch.float32), pb[16 * m:].view(torch.int8))
    lst.lst_run(0)
    rows = 4096
    h = torch.zeros(32 + 3 * rows, dtype=torch.int32).pin_memory()
    lst.lst_read_tc_host(0, h[:32], h[32:].view(rows, 3))
    torch.cuda.synchronize()
    out = lst.fetch(0)
    parity.compare(geo_full, w, ev, out)
    assert int(h[31]) == 0 and int(h[P.CNT["tc"]]) == out["counts"]["tc"]
    ntc = out["counts"]["tc"]
    assert np.array_equal(h[32:32 + 3 * ntc].numpy().reshape(ntc, 3), out["tc"]["tc"].reshape(ntc, 3))
    lst.close()


def test_bench_launch_configuration_sampled(P, geo_full):
    """The configuration bench.py times (configs[3]): 64 PU200 events, seeds 100-163, 4 streams x 16-event batched
    launches, bench capacities.  ALL 64 events are compared with the oracle in full; every event must be
    overflow-free and satisfy the TC partition identity n_pLS = pT5 + pT3 + pLS-TC."""
    import torch
    w = xavier_weights(3)
    E, S = 64, 4
    evs = [config_event(geo_full, 2, seed=100 + i) for i in range(E)]
    caps = P.Caps(n_slots=E, max_hits=114688, max_md=49152, max_ls=49152, max_t3=32768, max_t5c=16384, max_t5=16384, max_pls=4096)
    lst = P.LST(geo_full, w, caps)
    for i, ev in enumerate(evs):
        lst.load_numpy_event(i, ev)
    streams = [torch.cuda.Stream() for _ in range(S)]
    torch.cuda.synchronize()
    for _ in range(2):                                    # second pass runs on warm state, as in the timed region
        for si, st in enumerate(streams):
            lst.lst_run_batch(si * (E // S), E // S, st)
    torch.cuda.synchronize()
    for i, ev in enumerate(evs):
        bits, c = lst.lst_status(i)
        assert bits == 0, (i, bits)
        assert c["pt5"] + c["pt3"] + c["plstc"] == ev.n_pls and c["pt5"] + c["t5tc"] + c["pt3"] + c["plstc"] == c["tc"], (i, c)
    for i in range(E):                                    # every event of the timed configuration, in full
        parity.compare(geo_full, w, evs[i], lst.fetch(i))
    lst.close()


def test_batched_host_load_and_read(P, geo_full):
    """lst_load_batch_host (one blob, one H2D copy) + lst_read_tc_batch_host (one D2H copy) give the same events
    and TC rows as the per-event path; malformed blobs are rejected."""
    import torch
    w = xavier_weights(3)
    evs = [config_event(geo_full, 1, seed=7), make_event(geo_full, 3), config_event(geo_full, 2, seed=101)]
    lst = P.LST(geo_full, w, P.default_caps(4))
    blob = P.pack_batch(evs)
    lst.lst_load_batch_host(1, 3, blob)                  # slots 1..3
    lst.lst_run_batch(1, 3)
    rows = 4096
    h = torch.zeros((3, 32 + 3 * rows), dtype=torch.int32).pin_memory()
    lst.lst_read_tc_batch_host(1, 3, h)
    torch.cuda.synchronize()
    for i, ev in enumerate(evs):
        out = lst.fetch(1 + i)
        parity.compare(geo_full, w, ev, out)
        ntc = out["counts"]["tc"]
        assert int(h[i, 31]) == 0 and int(h[i, P.CNT["tc"]]) == ntc
        assert np.array_equal(h[i, 32:32 + 3 * ntc].numpy().reshape(ntc, 3), out["tc"]["tc"].reshape(ntc, 3))
    # the 16-bit-key wire format gives the same events
    lst.lst_load_batch_host16(1, 3, P.pack_batch(evs, key16=True))
    lst.lst_run_batch(1, 3)
    h2 = torch.zeros((3, 32 + 13 * rows), dtype=torch.int32).pin_memory()
    lst.lst_read_tc_hits_batch_host(1, 3, h2)
    torch.cuda.synchronize()
    for i, ev in enumerate(evs):
        out = lst.fetch(1 + i)
        parity.compare(geo_full, w, ev, out)
        ntc = out["counts"]["tc"]
        got = h2[i, 32:32 + 13 * ntc].numpy().reshape(ntc, 13)
        assert np.array_equal(got[:, :3], out["tc"]["tc"].reshape(ntc, 3)) and np.array_equal(got[:, 3:], out["tcx"]["hits"].reshape(ntc, 12)[:, :10])
    with pytest.raises(P.LstError):                      # short buffer
        lst.lst_load_batch_host(0, 3, blob[:1000])
    bad = blob.clone()
    bad.numpy()[:4].view(np.int32)[0] = 10 ** 8          # n_hits above the capacity
    with pytest.raises(P.LstError):
        lst.lst_load_batch_host(0, 3, bad)
    lst.close()


def test_graph_export(P, geo_full):
    """f4 (SPEC.md 4.8): nodes = MDs, CSR edges = LSs, original hit numbering, for a batch of events."""
    w = xavier_weights(3)
    evs = [config_event(geo_full, 2, seed=100), config_event(geo_full, 1), make_event(geo_full, 9)]
    lst = P.LST(geo_full, w, P.default_caps(len(evs)))
    for i, ev in enumerate(evs):
        lst.load_numpy_event(i, ev)
    lst.lst_run_batch(0, len(evs))
    lst.lst_export_graph(0, len(evs))
    n_edges = [parity.compare_graph(geo_full, w, ev, lst.fetch_graph(i)) for i, ev in enumerate(evs)]
    assert n_edges[0] > 10000 and n_edges[2] == 0
    lst.close()


@pytest.mark.parametrize("n_feat,n_hidden", [(23, 1), (23, 3), (23, 4), (38, 1), (38, 2), (38, 3), (38, 4)])
def test_dnn_variants(P, geo_full, n_feat, n_hidden):
    """f3 (SPEC.md 4.9): the paper's 38 inputs and the 1 / 3 / 4 hidden-layer networks of its depth scan, end to end."""
    w = xavier_weights(11, bias_scale=0.3, n_feat=n_feat, n_hidden=n_hidden)
    ev = config_event(geo_full, 1, seed=31)
    lst = P.LST(geo_full, w, P.default_caps(1), dnn=(n_feat, n_hidden))
    lst.load_numpy_event(0, ev)
    lst.lst_run(0)
    out = lst.fetch(0)
    lst.close()
    assert out["t5c"]["feat"].shape[1] == n_feat
    c = parity.compare(geo_full, w, ev, out, dnn=(n_feat, n_hidden))
    assert c["t5c"] > 500


def _dup_hits(ev, sel, times):
    """append `times` copies of the hits `sel` (same sensor, same position): every object built on them multiplies"""
    for name in ("x", "y", "z", "key", "hit_particle"):
        a = getattr(ev, name)
        setattr(ev, name, np.concatenate([a] + [a[sel]] * times))


def test_rows_with_many_partners(P, geo_barrel):
    """a3 / a4 keep the first TUPLE_STASH = 3 passing partners of a row in registers and evaluate the row again when there
    are more.  Hits of layers 3-5 of clean muons duplicated twice -> 9 MDs per layer and muon -> LS rows with 9 passing
    partners, T3 rows with 9: the re-evaluation path is what produces these lists."""
    w = xavier_weights(1)
    ev = make_event(geo_barrel, 81, origin_muons=3, smear=False)
    r = np.hypot(ev.x, ev.y)
    _dup_hits(ev, np.flatnonzero((r > 50) & (r < 90)), 2)
    out = _run_one(P, geo_barrel, w, ev)
    c = parity.compare(geo_barrel, w, ev, out)
    t3_per_row = np.bincount(out["t3"]["abc"][:, 3])
    t5_per_row = np.bincount(out["t5c"]["t3"][:, 0])
    assert t3_per_row.max() > 3 and t5_per_row.max() > 3, (t3_per_row.max(), t5_per_row.max())


def test_csr_row_with_many_runs(P, geo_barrel):
    """a2 caches the non-empty runs of a CSR row 32 at a time; a row with more runs than that takes the chunked path.  The
    rows of the occupied layer-1 modules get 40 extra, non-consecutive columns (every second module of layer 2)."""
    import dataclasses
    w = xavier_weights(1)
    ev = make_event(geo_barrel, 82, origin_muons=10)
    l2 = int(geo_barrel.barrel_base[1])
    occupied = set(int(k) >> 1 for k in ev.key if (int(k) >> 1) < l2)
    # every second module of a stretch of layer 2 (mostly empty: runs that hold no MD) plus every occupied module beyond layer 1
    extra = set(range(l2, l2 + 160, 2)) | set(range(l2 + 401, l2 + 481, 2)) | set(int(k) >> 1 for k in ev.key if (int(k) >> 1) >= l2)
    rows = []
    for m in range(geo_barrel.n_modules):
        cols = set(geo_barrel.conn_col[geo_barrel.conn_rowptr[m]:geo_barrel.conn_rowptr[m + 1]].tolist())
        if m in occupied:
            cols |= extra
        rows.append(sorted(cols))
    rowptr = np.zeros(geo_barrel.n_modules + 1, np.int32)
    rowptr[1:] = np.cumsum([len(c) for c in rows])
    g2 = dataclasses.replace(geo_barrel, conn_rowptr=rowptr, conn_col=np.array([c for r in rows for c in r], np.int32))
    n_runs = max(sum(1 for i, c in enumerate(r) if i == 0 or r[i - 1] != c - 1) for r in rows)
    assert n_runs > 64
    out = _run_one(P, g2, w, ev)
    c = parity.compare(g2, w, ev, out)
    assert c["ls_pairs"] > 400 and c["ls"] > 40


def test_dense_module_takes_the_big_path(P, geo_barrel):
    """a1 packs the cells of 32 modules into one flat index space unless a module alone has more than 2^20 cells; such a
    module (1100 x 1100 hits here) is swept on its own with a 64-bit sweep counter.  Expect plain parity, no flag."""
    w = xavier_weights(1)
    ev = make_event(geo_barrel, 83, origin_muons=4)
    rng = np.random.default_rng(9)
    m = 5 * 24 + 12                                   # a layer-1 module: phi sector 5, central z tile
    nphi = int(geo_barrel.barrel_nphi[0])
    n = 1100
    for up, rr in ((0, 23.0), (1, 23.26)):
        ph = (5 + rng.uniform(0.05, 0.95, n)) * 2 * np.pi / nphi
        ev.x = np.concatenate([ev.x, (rr * np.cos(ph)).astype(np.float32)]); ev.y = np.concatenate([ev.y, (rr * np.sin(ph)).astype(np.float32)])
        ev.z = np.concatenate([ev.z, rng.uniform(0.5, 9.5, n).astype(np.float32)])
        ev.key = np.concatenate([ev.key, np.full(n, 2 * m + up, np.uint32)])
        ev.hit_particle = np.concatenate([ev.hit_particle, np.full(n, -1, np.int32)])
    out = _run_one(P, geo_barrel, w, ev, P.Caps(n_slots=1, max_hits=8192, max_md=65536, max_ls=65536, max_t3=65536, max_t5c=65536, max_t5=65536, max_pls=64))
    assert out["status"] == 0
    c = parity.compare(geo_barrel, w, ev, out)
    assert c["md_pairs"] > (1 << 20) and c["md"] > 1000


def test_graphs_on_off_and_determinism(P, geo_full):
    """The CUDA-graph replay (default on a non-default stream) and direct launches (LST_GRAPHS=0) give identical bytes, and
    one PU200 event run 100 times gives the same bytes every time."""
    import os, torch
    w = xavier_weights(3)
    ev = config_event(geo_full, 2)
    names = ("md", "ls", "t3", "t5c", "t5", "tc", "match5", "tcc", "tcx")

    def snap(lst):
        o = lst.fetch(0)
        return {(n, k): v.copy().view(np.uint8) for n in names for k, v in o[n].items()}

    st = torch.cuda.Stream()
    lst = P.LST(geo_full, w, P.default_caps(1))
    lst.load_numpy_event(0, ev)
    torch.cuda.synchronize()
    lst.lst_run(0, st)
    torch.cuda.synchronize()
    ref = snap(lst)
    for _ in range(100):
        lst.lst_run(0, st)
    torch.cuda.synchronize()
    again = snap(lst)
    assert all(np.array_equal(ref[k], again[k]) for k in ref)
    for rep in range(4):                 # a few full comparisons along the way as well
        lst.lst_run(0, st)
        torch.cuda.synchronize()
        again = snap(lst)
        assert all(np.array_equal(ref[k], again[k]) for k in ref), rep
    lst.close()
    os.environ["LST_GRAPHS"] = "0"
    try:
        lst = P.LST(geo_full, w, P.default_caps(1))
        lst.load_numpy_event(0, ev)
        torch.cuda.synchronize()
        lst.lst_run(0, st)
        torch.cuda.synchronize()
        direct = snap(lst)
        lst.close()
    finally:
        del os.environ["LST_GRAPHS"]
    assert all(np.array_equal(ref[k], direct[k]) for k in ref)
    # and the bytes that never changed are the right ones
    lst = P.LST(geo_full, w, P.default_caps(1))
    lst.load_numpy_event(0, ev)
    torch.cuda.synchronize()
    lst.lst_run(0, st)
    torch.cuda.synchronize()
    out = lst.fetch(0)
    lst.close()
    assert all(np.array_equal(ref[(n, k)], v.view(np.uint8)) for n in names for k, v in out[n].items())
    parity.compare(geo_full, w, ev, out)


def _odd_pls(ev, rng):
    """Overwrite a fifth of the seeds with values the a6 bins cannot hold (overflow bins): pT below the bucketed range, |z0| > 20 cm,
    |cot| > 8, q = 0, and a few that curl up before the outer layers (r h > 0.88 there)."""
    n = ev.n_pls
    idx = rng.choice(n, max(5, n // 5), replace=False)
    for k, p in enumerate(idx):
        pt = float(np.hypot(ev.pls_px[p], ev.pls_py[p]))
        mode = k % 5
        if mode == 0: s = 0.5 / pt; ev.pls_px[p] *= s; ev.pls_py[p] *= s; ev.pls_pz[p] *= s      # pT = 0.5 GeV: h > HMAX
        elif mode == 1: ev.pls_z0[p] = np.float32(25.0 if k % 2 else -31.0)
        elif mode == 2: ev.pls_pz[p] = np.float32(9.5 * pt * (1 if k % 2 else -1))
        elif mode == 3: ev.pls_q[p] = 0
        else: s = 0.78 / pt; ev.pls_px[p] *= s; ev.pls_py[p] *= s; ev.pls_pz[p] *= s           # pT = 0.78 GeV: still bucketed, r h up to 0.8
    return ev


def test_a6_layer_label_255(P, geo_full):
    """Any uint8 is a legal layer label (include/lst.h: "any labelling, or none, gives the same matches").  255 used to double as the
    library's internal "no T3 / T5 starts here" mark, so the surfaces of modules labelled 255 were never measured and their objects
    were matched against stale bins.  Barrel layer 1 (where most T5s start) relabelled 255, then everything relabelled 255."""
    import dataclasses
    w = xavier_weights(3)
    ev = config_event(geo_full, 2, seed=37)
    base = parity.compare(geo_full, w, ev, _run_one(P, geo_full, w, ev))
    assert base["tc"] > 2000
    lab = geo_full.layer.copy()
    lab[lab == 1] = 255
    g1 = dataclasses.replace(geo_full, layer=lab)
    parity.compare(g1, w, ev, _run_one(P, g1, w, ev))
    g2 = dataclasses.replace(geo_full, layer=np.full_like(geo_full.layer, 255))
    parity.compare(g2, w, ev, _run_one(P, g2, w, ev))


def test_a6_generic_buckets_relabelled_layers_and_odd_seeds(P, geo_full):
    """a6 has two exact prefilters: per-surface crossing keys (geometry with a layer per module) and the generic (h, zeta, psi)
    buckets (no layers, or LST_XS=0).  Both must give the oracle's lists: with the real layers, without layers, with every module
    relabelled to ONE layer (surfaces 87 cm / 134 cm thick: windows open up, nothing may be lost), with a layer labelling that mixes
    two barrel layers, and with seeds the bins cannot hold."""
    import dataclasses, os
    w = xavier_weights(3)
    rng = np.random.default_rng(5)
    ev = _odd_pls(config_event(geo_full, 2, seed=31), rng)
    base = parity.compare(geo_full, w, ev, _run_one(P, geo_full, w, ev))
    assert base["tc"] > 2000
    g_none = dataclasses.replace(geo_full, layer=None)
    parity.compare(g_none, w, ev, _run_one(P, g_none, w, ev))
    g_one = dataclasses.replace(geo_full, layer=np.ones_like(geo_full.layer))
    parity.compare(g_one, w, ev, _run_one(P, g_one, w, ev))
    mixed = geo_full.layer.copy()
    mixed[mixed == 3] = 2                      # layers 2 and 3 share a surface: 15 cm thick
    mixed[mixed == 9] = 8                      # two disks share a surface: 29 cm thick
    g_mix = dataclasses.replace(geo_full, layer=mixed)
    parity.compare(g_mix, w, ev, _run_one(P, g_mix, w, ev))
    os.environ["LST_XS"] = "0"
    try:
        parity.compare(geo_full, w, ev, _run_one(P, geo_full, w, ev))
    finally:
        del os.environ["LST_XS"]
    ev4 = _odd_pls(config_event(geo_full, 4, seed=207, pileup=100), rng)          # displaced tracks as well
    parity.compare(geo_full, w, ev4, _run_one(P, geo_full, w, ev4))
    parity.compare(g_one, w, ev4, _run_one(P, g_one, w, ev4))


def test_a2_module_with_more_than_eight_nonempty_runs(P, geo_barrel):
    """a2 reads a per-module column table of up to 8 non-empty runs written by k_md_finish; a module whose CSR row holds more
    non-empty runs builds its run table in the sweep.  Occupied layer-1 modules get every second OCCUPIED module beyond layer 1
    as extra columns, so their rows hold 9 .. 32 non-empty runs (the 64+ case is test_csr_row_with_many_runs)."""
    import dataclasses
    w = xavier_weights(1)
    ev = make_event(geo_barrel, 84, origin_muons=12)
    l2 = int(geo_barrel.barrel_base[1])
    occ = sorted(set(int(k) >> 1 for k in ev.key))
    occupied_l1 = [m for m in occ if m < l2]
    beyond = [m for m in occ if m >= l2]
    extra = set(m for m in beyond if (m + 1) not in set(beyond) or m % 2 == 0)
    rows = []
    for m in range(geo_barrel.n_modules):
        cols = set(geo_barrel.conn_col[geo_barrel.conn_rowptr[m]:geo_barrel.conn_rowptr[m + 1]].tolist())
        if m in occupied_l1:
            cols |= extra
        rows.append(sorted(cols))
    rowptr = np.zeros(geo_barrel.n_modules + 1, np.int32)
    rowptr[1:] = np.cumsum([len(c) for c in rows])
    g2 = dataclasses.replace(geo_barrel, conn_rowptr=rowptr, conn_col=np.array([c for r in rows for c in r], np.int32))
    out = _run_one(P, g2, w, ev)
    c = parity.compare(g2, w, ev, out)
    # non-empty runs of the occupied layer-1 rows, from the oracle's own MD list
    md_mod = set((out["md"]["modt"] >> 2).tolist())
    n_ne = []
    for m in occupied_l1:
        r = rows[m]
        runs = [[r[0]]]
        for a, b in zip(r, r[1:]):
            if b == a + 1: runs[-1].append(b)
            else: runs.append([b])
        n_ne.append(sum(1 for run in runs if any(x in md_mod for x in run)))
    assert max(n_ne) > 8, max(n_ne)
    assert c["ls"] > 40


def test_one_launch_over_more_than_32_events(P, geo_full):
    """a2 hands out the chunks of up to 32 events by one ticket (one persistent grid per 32 events); a 45-event batch takes two
    groups (32 + 13), mixed sizes incl. empty events, and offsets other than 0.  Every event against the oracle."""
    w = xavier_weights(3)
    evs = []
    for i in range(45):
        if i % 9 == 4: evs.append(make_event(geo_full, 300 + i))                     # empty
        elif i % 3 == 0: evs.append(config_event(geo_full, 1, seed=300 + i))          # PU50
        elif i % 3 == 1: evs.append(make_event(geo_full, 300 + i, origin_muons=5, n_noise=300))
        else: evs.append(config_event(geo_full, 4, seed=300 + i, pileup=100 if i % 2 else 0))
    caps = P.default_caps(48)
    lst = P.LST(geo_full, w, caps)
    for i, ev in enumerate(evs):
        lst.load_numpy_event(i + 2, ev)          # slots 2 .. 46
    lst.lst_run_batch(2, len(evs))
    for i, ev in enumerate(evs):
        parity.compare(geo_full, w, ev, lst.fetch(i + 2))
    lst.close()


def test_a6_prefilters_agree_on_many_events(P, geo_full):
    """Both a6 prefilters only select which (pLS, object) pairs get the exact test, so they must produce identical bytes.  24 events
    (PU200 / PU300 + displaced, a fifth of the seeds pushed to the edges of the binned range) through both, match tables and TC
    lists compared byte by byte; four of the events also against the oracle."""
    import os
    w = xavier_weights(3)
    rng = np.random.default_rng(11)
    evs = []
    for i in range(24):
        ev = config_event(geo_full, 4, seed=400 + i, pileup=300 if i % 3 == 0 else 200)
        n = ev.n_pls
        idx = rng.choice(n, n // 5, replace=False)
        for k, p in enumerate(idx):
            pt = float(np.hypot(ev.pls_px[p], ev.pls_py[p]))
            if k % 4 == 0: ev.pls_z0[p] = np.float32(rng.choice([-19.9, 19.9, -20.5, 20.5]))
            elif k % 4 == 1: ev.pls_pz[p] = np.float32(rng.uniform(6.5, 8.5) * pt * rng.choice([-1, 1]))          # |cot| up to the cap
            elif k % 4 == 2: s = rng.uniform(0.76, 0.85) / pt; ev.pls_px[p] *= s; ev.pls_py[p] *= s; ev.pls_pz[p] *= s      # around pT = 0.8
            else: ev.pls_pz[p] = np.float32(rng.uniform(-0.05, 0.05) * pt)                                          # central: both circle intersections matter
        evs.append(ev)
    caps = P.Caps(n_slots=24, max_hits=196608, max_md=98304, max_ls=98304, max_t3=65536, max_t5c=32768, max_t5=32768, max_pls=8192)

    def run():
        lst = P.LST(geo_full, w, caps)
        for i, ev in enumerate(evs):
            lst.load_numpy_event(i, ev)
        lst.lst_run_batch(0, len(evs))
        out = [lst.fetch(i) for i in range(len(evs))]
        lst.close()
        return out

    a = run()
    os.environ["LST_XS"] = "0"
    try:
        b = run()
    finally:
        del os.environ["LST_XS"]
    for i, (x, y) in enumerate(zip(a, b)):
        assert x["status"] == 0 and y["status"] == 0, (i, x["status"], y["status"])
        for obj in ("match5", "tc", "tcc", "tcx"):
            for k in x[obj]:
                assert np.array_equal(x[obj][k].view(np.uint8), y[obj][k].view(np.uint8)), (i, obj, k)
    for i in (0, 7, 12, 23):
        parity.compare(geo_full, w, evs[i], a[i])
