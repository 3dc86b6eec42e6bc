"""f2: the truth matcher / efficiency tally (paper_2403_13166_b200/evaluate.py) on candidates whose truth is known by
construction.  CPU: candidates come from the oracle here; the -m gpu test feeds it the CUDA output."""
import numpy as np
import pytest

from lstgen import make_event, config_event, xavier_weights
from oracle import lst_oracle as O
from paper_2403_13166_b200 import evaluate as E


def test_truth_match_rule():
    """> 75 % of the hits from one particle: 8 of 10 matches, 7 of 10 does not; noise hits count against; pLS follow their seed"""
    class Ev: pass
    ev = Ev()
    ev.hit_particle = np.array([5] * 8 + [6] * 2 + [-1] * 3 + [7] * 10)
    ev.pls_particle = np.array([3, 4])
    h = lambda *idx: list(idx) + [-1] * (10 - len(idx))
    hits = np.array([h(*range(0, 10)),                 # 8 x particle 5 + 2 x particle 6 -> 5
                     h(*range(1, 11)),                 # 7 x 5, 2 x 6, 1 noise -> none
                     h(0, 1, 2, 3, 4, 10),             # T3: 5 of 6 from 5 -> 5
                     h(0, 1, 2, 3, 10, 11),            # T3: 4 of 6 -> none
                     h(*range(13, 23)),                # all from 7
                     h()])
    m = E.truth_match(ev, np.array([0, 1, 2, 2, 1, 3]), np.array([0, -1, 1, 1, -1, 1]), hits)
    assert m.tolist() == [5, -1, 5, -1, 7, 4]


def test_clean_muons_are_fully_efficient(geo_barrel):
    """noise-free barrel muons with exact seeds: every muon is found, nothing is fake; the raw list holds no duplicates
    (one pT5 per muon: the second T5 is a matched loser) -- and the tally's denominators see all 10 muons"""
    t = E.Tally()
    for seed in (71, 72, 73):
        ev = make_event(geo_barrel, seed, origin_muons=10, smear=False)
        r = O.run(geo_barrel, xavier_weights(1), ev)
        t.add(ev, r.tc[:, 0], r.tc[:, 1], r.tc_hits)
    s = t.summary()
    assert s["n_particles"] == 30 and s["efficiency"] == 1.0 and s["fake_rate"] == 0.0 and s["duplicate_rate"] == 0.0
    assert sum(b["n"] for b in s["vs"]["pt"]) == 30 and all(b["eff"] in (None, 1.0) for b in s["vs"]["eta"])
    # every muon is found by a candidate with outer-tracker hits (a pT5), none through a bare seed
    assert s["efficiency_outer_tracker"] == 1.0 and s["efficiency_by_type"] == {"pT5": 1.0, "T5": 0.0, "pT3": 0.0, "pLS": 0.0}


def test_seed_only_candidates_do_not_count_for_the_outer_tracker(geo_barrel):
    """The pooled efficiency is nearly tautological on this generator (every prompt particle has a seed, a pLS candidate is matched
    through the seed's label): a candidate list made of bare seeds 'finds' every muon although the outer-tracker chain built
    nothing.  The outer-tracker headline must read 0 for it."""
    ev = make_event(geo_barrel, 71, origin_muons=10, smear=False)
    n = ev.n_pls
    t = E.Tally()
    t.add(ev, np.full(n, 3), np.arange(n), -np.ones((n, 10), dtype=np.int64))
    s = t.summary()
    assert s["efficiency"] == 1.0 and s["efficiency_outer_tracker"] == 0.0 and s["fake_rate_outer_tracker"] is None
    assert s["efficiency_by_type"]["pLS"] == 1.0


def test_pileup_event_numbers_are_sane(geo_full):
    """PU50 with smearing and noise: high efficiency, and the duplicate cleaning (f1) removes duplicates without
    costing efficiency"""
    ev = config_event(geo_full, 1)
    w = E.pass_all_weights()
    r = O.run(geo_full, w, ev)
    raw, cl = E.Tally(), E.Tally()
    raw.add(ev, r.tc[:, 0], r.tc[:, 1], r.tc_hits)
    k = r.tc_keep.astype(bool)
    cl.add(ev, r.tc[k, 0], r.tc[k, 1], r.tc_hits[k])
    a, b = raw.summary(), cl.summary()
    assert a["efficiency"] > 0.9 and b["efficiency"] >= a["efficiency"] - 0.01
    assert b["duplicate_rate"] < a["duplicate_rate"] and a["duplicate_rate"] > 0.02
    assert a["fake_rate"] < 0.2
    assert len(r.t5) == len(r.t5c)                  # the pass-all weights really switch the DNN cut off


@pytest.mark.gpu
def test_gpu_candidates_give_the_same_tally(geo_full):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    evs = [config_event(geo_full, 1, seed=40 + i) for i in range(2)]
    w = xavier_weights(3)
    for cleaned in (False, True):
        g = E.run_gpu(evs, geo_full, w, cleaned).summary()
        t = E.Tally()
        for ev in evs:
            r = O.run(geo_full, w, ev)
            k = r.tc_keep.astype(bool) if cleaned else np.ones(len(r.tc), bool)
            t.add(ev, r.tc[k, 0], r.tc[k, 1], r.tc_hits[k])
        assert g == t.summary()
