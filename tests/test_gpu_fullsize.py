"""-m gpu: parity at the sizes and in the launch shapes bench.py runs (BASELINE.json configs 3 and 4; B:L5 "bit-exact
to the CPU oracle on all five configs"), plus the stress tests of the fast path's error bound.

The oracle stays single-threaded; independent units of the same definition (events, d0 slabs, hit ranges) are given to
several host threads so that the full-size comparisons finish in a minute.
"""
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest
import torch

from oracle import Oracle, OracleCandidates
from workloads import HoughBinning, generate_events, get_workload, LAYERS_10
from workloads.configs import ACC_I32, ACC_U16

pytestmark = pytest.mark.gpu

from gpu_util import (assert_centroids_close, n_threads, oracle_peaks_parallel, oracle_vote_parallel, run_cuda, run_vote)  # noqa: E402
from paper_1311_2769_b200 import HoughPlan, alloc_candidates, candidates_to_numpy  # noqa: E402


def test_config_3_one_256_event_call_bit_exact():
    """One hough_vote / hough_find_peaks / hough_assign_hits call over events 0..255 of config 3 -- the call shape of
    bench.py's device-resident loop (grid 8192 tiles, 2.19 M staged hits) -- against the oracle run event by event."""
    w = get_workload(3)
    bn = w.binning
    n_ev = 256
    batch = generate_events(w, events=list(range(n_ev)))
    cap = 32768 * n_ev
    got = run_cuda(bn, w.bz_tesla, w.layers, batch.hits_xy, batch.event_offsets, w.threshold, w.assoc_dj, w.min_hits, cap,
                   options=("reuse_staging",))
    assert got.total <= cap
    o = Oracle.from_binning(bn, w.bz_tesla)

    def one(e):
        ev = batch.select([e])
        acc, votes = o.vote(ev.hits_xy, ev.event_offsets)
        assert acc.max() <= 65535
        ref = o.find_peaks(acc, w.threshold)
        h2c, nh, keep = o.assign_indexed(ev.hits_xy, ev.event_offsets, ref, w.assoc_dj, w.min_hits)
        c0, c1 = int(got.offsets[e]), int(got.offsets[e + 1])
        h0, h1 = int(batch.event_offsets[e]), int(batch.event_offsets[e + 1])
        assert np.array_equal(got.accum[e], acc[0].astype(np.uint16)), ("accum", e)
        assert c1 - c0 == ref.total, ("count", e)
        rec = got.records[c0:c1]
        assert np.all(rec["event"] == e)
        for f in ("k", "i", "j", "votes"):
            assert np.array_equal(rec[f], ref.records[f]), (f, e)
        assert_centroids_close(rec, ref.records, bn)
        assert np.array_equal(got.hit_to_cand[h0:h1], np.where(h2c >= 0, h2c + c0, -1)), ("hit_to_cand", e)
        assert np.array_equal(got.cand_nhits[c0:c1], nh) and np.array_equal(got.cand_keep[c0:c1], keep), ("dedup", e)
        return votes, int(keep.sum())

    with ThreadPoolExecutor(n_threads()) as ex:
        res = list(ex.map(one, range(n_ev)))
    assert sum(r[0] for r in res) == int(got.accum.astype(np.int64).sum())
    assert sum(r[1] for r in res) > 100 * n_ev            # ~195 kept candidates per event (SURVEY table D)
    assert not got.cand_nhits[got.total:].any() and not got.cand_keep[got.total:].any()


def test_config_4_full_size_all_outputs_bit_exact():
    """Config 4 at full size (162 k hits, 1024 x 512 x 128 u16): the whole accumulator, the whole candidate list and every
    hit's assignment against the oracle (vote and peaks by d0 slabs, association by hit ranges on host threads), plus the
    brute-force association (all candidates x sampled hits) as the independent check SURVEY 8(c) D9 prescribes."""
    w = get_workload(4)
    bn = w.binning
    batch = generate_events(w)
    cap = bn.n_bins // 16
    got = run_cuda(bn, w.bz_tesla, w.layers, batch.hits_xy, batch.event_offsets, w.threshold, w.assoc_dj, w.min_hits, cap)
    o = Oracle.from_binning(bn, w.bz_tesla)
    acc, votes = oracle_vote_parallel(o, batch.hits_xy, batch.event_offsets)
    assert acc.max() <= 65535
    assert np.array_equal(got.accum, acc.astype(np.uint16)), "accumulator differs"
    assert votes == int(got.accum.astype(np.int64).sum())
    ref = oracle_peaks_parallel(o, acc, w.threshold)
    del acc
    assert got.total == ref.total <= cap and list(got.offsets) == [0, ref.total]
    for f in ("event", "k", "i", "j", "votes"):
        assert np.array_equal(got.records[f], ref.records[f]), f
    assert_centroids_close(got.records, ref.records, bn)

    # association: raw best candidate of every hit (indexed oracle, hits split over threads), then D9 here
    nt = max(1, min(8, n_threads()))                       # each thread holds a 268 MB bin -> candidate index
    bounds = np.linspace(0, batch.n_hits, nt + 1).astype(int)

    def part(t):
        h0, h1 = int(bounds[t]), int(bounds[t + 1])
        off = np.array([0, h1 - h0], np.int32)
        return o.assign_indexed(batch.hits_xy[h0:h1], off, ref, w.assoc_dj, w.min_hits, apply_dedup=False)[0]

    with ThreadPoolExecutor(nt) as ex:
        raw = np.concatenate(list(ex.map(part, range(nt))))
    nh = np.bincount(raw[raw >= 0], minlength=ref.total).astype(np.int32)
    keep = nh >= w.min_hits
    h2c = np.where((raw >= 0) & keep[np.maximum(raw, 0)], raw, -1)
    assert np.array_equal(got.cand_nhits[:ref.total], nh), "cand_nhits differs"
    assert np.array_equal(got.cand_keep[:ref.total].astype(bool), keep)
    assert np.array_equal(got.hit_to_cand, h2c), "hit_to_cand differs"
    assert keep.sum() > 1000 and (h2c >= 0).sum() > 10000

    # brute force over all candidates for sampled hits (D9's prescription): 512 hits x 2.2 M candidates
    rng = np.random.default_rng(44)
    sample = np.sort(rng.choice(batch.n_hits, 512, replace=False))
    chunks = np.array_split(sample, nt)

    def brute(idx):
        off = np.array([0, len(idx)], np.int32)
        return o.assign_brute(batch.hits_xy[idx], off, ref, w.assoc_dj, w.min_hits, apply_dedup=False)[0]

    with ThreadPoolExecutor(nt) as ex:
        raw_b = np.concatenate(list(ex.map(brute, chunks)))
    assert np.array_equal(raw_b, raw[sample])


def _vote_keys_default_vs_exact(w, batch, n_ev_call):
    """Accumulators and final assignments of the default (error-bounded fast path) and the exact_walk (D3 at every
    window column; oracle-validated elsewhere) walks over the same input, call by call."""
    bn = w.binning
    n_ev = batch.n_events
    cap_ev = bn.n_bins // 16 if n_ev == 1 else 32768
    starts = list(range(0, n_ev, n_ev_call))
    max_hits = max(int(batch.event_offsets[min(s + n_ev_call, n_ev)] - batch.event_offsets[s]) for s in starts)
    plans = []
    for exact in (0, 1):
        p = HoughPlan.from_workload(w, max_hits=max_hits, max_events=n_ev_call)
        p.set_option("exact_walk", exact)
        p.set_option("reuse_staging", 1)
        plans.append(p)
    d_hits = torch.from_numpy(batch.hits_xy).cuda()
    n_diff = 0
    for s in starts:
        ne = min(n_ev_call, n_ev - s)
        h0, h1 = int(batch.event_offsets[s]), int(batch.event_offsets[s + ne])
        d_off = torch.from_numpy((batch.event_offsets[s:s + ne + 1] - h0).astype(np.int32)).cuda()
        outs = []
        for p in plans:
            accum = p.alloc_accum(ne)
            cap = cap_ev * ne
            cands = alloc_candidates(cap)
            coff = torch.zeros(ne + 1, dtype=torch.int32, device="cuda")
            h2c = torch.empty(h1 - h0, dtype=torch.int32, device="cuda")
            nh = torch.empty(cap, dtype=torch.int32, device="cuda")
            keep = torch.empty(cap, dtype=torch.uint8, device="cuda")
            p.vote(d_hits[h0:h1], d_off, accum)
            p.find_peaks(accum, ne, w.threshold, cands, cap, coff)
            p.assign_hits(d_hits[h0:h1], d_off, cands, coff, cap, w.assoc_dj, w.min_hits, h2c, nh, keep)
            outs.append((accum, h2c, nh, coff))
        torch.cuda.synchronize()
        (a0, h0_, n0, c0), (a1, h1_, n1, c1) = outs
        assert torch.equal(c0, c1)
        n_diff += int((a0.view(torch.int16) != a1.view(torch.int16)).sum().item()) if a0.dtype == torch.uint16 else \
            int((a0 != a1).sum().item())
        assert torch.equal(h0_, h1_), ("hit_to_cand", s)
        tot = int(c0[-1].item())
        assert torch.equal(n0[:tot], n1[:tot]), ("cand_nhits", s)
        del outs, a0, a1
    for p in plans:
        p.close()
    return n_diff


def test_config_3_all_1024_events_default_equals_exact_walk():
    """Stress test of the fast path's error bound: 6.6e9 votes, 7.6e9 fast evaluations (one bench step)."""
    w = get_workload(3)
    batch = generate_events(w)
    assert batch.n_events == 1024
    assert _vote_keys_default_vs_exact(w, batch, 256) == 0


def test_config_4_default_equals_exact_walk():
    w = get_workload(4)
    assert _vote_keys_default_vs_exact(w, generate_events(w), 1) == 0


def test_event_with_300k_hits_redo_on_the_spot():
    """An event above 2^18 hits: the walk's redo-queue entries no longer fit 32 bits and uncertain pairs are redone on
    the spot (walk.cuh wq_ok == false).  Small binning so the oracle stays cheap; both accumulator dtypes' tiles."""
    rng = np.random.default_rng(300)
    n = 300_000
    r = rng.choice(np.asarray(LAYERS_10), n) * (1.0 + rng.normal(0, 2e-5, n))
    ph = rng.uniform(0, 2 * np.pi, n)
    hits = np.stack([r * np.cos(ph), r * np.sin(ph)], 1).astype(np.float32)
    off = np.array([0, n], np.int32)
    for shape, dtype in (((64, 32, 2), ACC_I32), ((128, 64, 1), ACC_I32)):
        bn = HoughBinning(*shape, accum_dtype=dtype)
        o = Oracle.from_binning(bn, 3.8)
        acc, votes = oracle_vote_parallel(o, hits, off)
        got = run_vote(bn, 3.8, LAYERS_10, hits, off)
        assert votes > 5 * n and np.array_equal(got, acc)
        thr = int(acc.max()) - 50
        ref = o.find_peaks(acc, thr)
        res = run_cuda(bn, 3.8, LAYERS_10, hits, off, thr, 1, 1, ref.total + 3)
        h2c, nh, keep = o.assign_indexed(hits, off, ref, 1, 1)
        assert res.total == ref.total and np.array_equal(res.hit_to_cand, h2c) and np.array_equal(res.cand_nhits[:ref.total], nh)
