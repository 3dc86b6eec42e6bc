"""Edge cases of the CUDA path against the oracle: non-finite inputs, capacity overflow inside a batched launch.  `-m gpu` only.

SPEC.md 1: "a NaN fails every cut" -- every selection of PAPER.md:39 is written as `!(lhs <= rhs)` so that an operand that is
not a number rejects.  The kernels' prefilters are allowed to let such pairs through to the exact test but never to accept
them, and nothing downstream (binning keys, argmin keys, compaction) may trip on them."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from lstgen import config_event, xavier_weights
import parity


@pytest.fixture(scope="module")
def P():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2403_13166_b200 as P
    P.load_library()
    return P


def _run_one(P, geo, w, ev, caps=None):
    lst = P.LST(geo, w, caps or P.default_caps(1))
    lst.load_numpy_event(0, ev)
    lst.lst_run(0)
    out = lst.fetch(0)
    lst.close()
    return out


BAD = [np.float32(np.nan), np.float32(np.inf), np.float32(-np.inf)]


def _poison(ev, rng, n_hits, n_pls):
    """NaN / +inf / -inf written into x, y or z of `n_hits` hits and into px, py, pz or z0 of `n_pls` seeds."""
    for k, i in enumerate(rng.choice(ev.n_hits, n_hits, replace=False)):
        (ev.x, ev.y, ev.z)[k % 3][i] = BAD[(k // 3) % 3]
    for k, p in enumerate(rng.choice(ev.n_pls, n_pls, replace=False)):
        (ev.pls_px, ev.pls_py, ev.pls_pz, ev.pls_z0)[k % 4][p] = BAD[(k // 4) % 3]
    return ev


@pytest.mark.parametrize("cfg,seed", [(1, 3), (2, 41)])
def test_non_finite_inputs(P, geo_full, cfg, seed):
    """No object may sit on a poisoned hit, a poisoned seed matches nothing and ends as a plain pLS candidate (or is dropped where
    SPEC.md 4.6 drops it), no flag is raised, no CUDA error -- and every list equals the oracle's, through both a6 prefilters."""
    import dataclasses
    w = xavier_weights(3)
    rng = np.random.default_rng(seed)
    clean = config_event(geo_full, cfg, seed=seed)
    ev = _poison(config_event(geo_full, cfg, seed=seed), rng, clean.n_hits // 40, clean.n_pls // 10)
    out = _run_one(P, geo_full, w, ev)
    assert out["status"] == 0
    c = parity.compare(geo_full, w, ev, out)
    # a NaN coordinate fails every cut (SPEC.md 1): no MD on such a hit.  An infinite one is a number: SPEC.md 4.1 as written accepts
    # e.g. an endcap upper hit at z = inf (Ls = inf, every bound inf, c_md = -+0) and a barrel upper hit at x = inf (c_md = inf / inf =
    # NaN) -- on both sides alike, which compare() has just checked -- but such an MD never gets into an LS (L1 / L3 see c or a NaN).
    nan_hit = np.isnan(ev.x) | np.isnan(ev.y) | np.isnan(ev.z)
    bad_hit = ~(np.isfinite(ev.x) & np.isfinite(ev.y) & np.isfinite(ev.z))
    assert nan_hit.sum() >= 30 and bad_hit.sum() >= 100 and not nan_hit[out["md"]["hits"]].any()
    assert not bad_hit[out["md"]["hits"][out["ls"]["ab"]]].any()
    bad_pls = ~(np.isfinite(ev.pls_px) & np.isfinite(ev.pls_py) & np.isfinite(ev.pls_pz) & np.isfinite(ev.pls_z0))
    tc = out["tc"]["tc"]
    assert bad_pls.sum() >= 20 and not bad_pls[tc[tc[:, 0] % 2 == 0, 1]].any()      # no pT5 (type 0) / pT3 (type 2) on a poisoned seed
    assert c["md"] > 0 and c["tc"] > 0
    g_none = dataclasses.replace(geo_full, layer=None)                                 # the generic (h, zeta, psi) buckets
    parity.compare(g_none, w, ev, _run_one(P, g_none, w, ev))


def O_counts(geo, w, ev):
    from oracle import lst_oracle as O
    return O.run(geo, w, ev, counts_only=True)


def test_overflow_of_one_event_inside_a_batch(P, geo_full):
    """configs[4] asks for every overflow flag; here the overflow happens to ONE event of a 16-event lst_run_batch (a PU200 event
    among PU50 events, capacities in between), which exercises the in-place re-run of that slot's rows inside the batched launch
    (k_md_finish / k_ls_finish) next to slots that do not overflow.  The neighbours must equal the oracle in full; the overflowing
    event keeps the oracle's first `cap` objects in build order, reports the unclamped total and raises only its own flag."""
    from oracle import lst_oracle as O
    w = xavier_weights(3)
    big_slot = 7
    evs = [config_event(geo_full, 1, seed=60 + i) for i in range(16)]
    evs[big_slot] = config_event(geo_full, 2, seed=77)
    ref_big = O.run(geo_full, w, evs[big_slot])
    small_max = {k: max(O_counts(geo_full, w, ev)[k] for i, ev in enumerate(evs) if i != big_slot) for k in ("md", "ls", "t3")}
    for name, bit, cnt in [("max_md", "ovf_md", "md"), ("max_ls", "ovf_ls", "ls"), ("max_t3", "ovf_t3", "t3")]:
        cap = (small_max[cnt] + ref_big.counts[cnt]) // 2
        assert small_max[cnt] < cap < ref_big.counts[cnt]
        kw = dict(n_slots=16, max_hits=131072, max_pls=4096, max_md=32768, max_ls=32768, max_t3=32768, max_t5c=32768, max_t5=32768)
        kw[name] = cap
        lst = P.LST(geo_full, w, P.Caps(**kw))
        for i, ev in enumerate(evs):
            lst.load_numpy_event(i, ev)
        lst.lst_run_batch(0, 16)
        outs = [lst.fetch(i) for i in range(16)]
        lst.close()
        for i, ev in enumerate(evs):
            if i != big_slot:
                assert outs[i]["status"] == 0, (name, i)
                parity.compare(geo_full, w, ev, outs[i])
        o = outs[big_slot]
        assert o["status"] == P.STATUS_BITS[bit], name
        assert o["counts"][cnt] == cap and o["counts"]["raw_" + cnt] == ref_big.counts[cnt]
        assert np.array_equal(o["md"]["hits"], ref_big.md_hits[:o["counts"]["md"]])          # MDs: always a prefix (the whole list unless MD overflows)
        if name == "max_ls":
            assert np.array_equal(o["ls"]["ab"], ref_big.ls[:cap])
        if name == "max_t3":
            assert np.array_equal(o["ls"]["ab"], ref_big.ls)
            assert np.array_equal(o["t3"]["abc"][:, :3], ref_big.t3[:cap, :3]) and np.array_equal(o["t3"]["l1"], ref_big.t3[:cap, 4])
