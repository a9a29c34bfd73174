"""-m gpu: config 3 in full -- all 1024 events -- in the two shapes bench.py times, against the oracle event by event
(B:L5 "bit-exact to the CPU oracle on all five configs"; B:L10 is the config the metric is quoted on).

(a) the device-resident loop: four calls of 256 events (plan option reuse_staging, as bench.py's DeviceRun);
(b) hough_pipeline_run_host with bench.py's e2e arguments: 32-event tiles on 4 streams, graphs on, per-tile capacity
    n_bins * 32 / 16 + 1024, pinned host buffers; full output and "kept_only".
The oracle stays single-threaded; events are independent units of the same definition and are given to host threads."""
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest
import torch

from oracle import Oracle
from workloads import generate_events, get_workload

pytestmark = pytest.mark.gpu

from gpu_util import assert_centroids_close, n_threads, run_cuda  # noqa: E402
from paper_1311_2769_b200 import CAND_DTYPE, HoughPipeline  # noqa: E402

_CACHE = {}          # event -> (records, hit_to_cand (event-local candidate ranks), cand_nhits, cand_keep); filled by (a) or (b)


def _oracle_event(o, w, batch, e, want_acc):
    ev = batch.select([e])
    acc, votes = o.vote(ev.hits_xy, ev.event_offsets)
    ref = o.find_peaks(acc, w.threshold)
    h2c, nh, keep = o.assign_indexed(ev.hits_xy, ev.event_offsets, ref, w.assoc_dj, w.min_hits)
    _CACHE[e] = (ref.records, h2c, nh, keep)
    return (acc[0].astype(np.uint16) if want_acc else None), votes


def _batch():
    w = get_workload(3)
    if "batch" not in _CACHE:
        _CACHE["batch"] = generate_events(w)
    assert _CACHE["batch"].n_events == 1024
    return w, _CACHE["batch"]


def test_config_3_all_1024_events_in_four_256_event_calls_bit_exact():
    w, batch = _batch()
    bn = w.binning
    o = Oracle.from_binning(bn, w.bz_tesla)
    kept_total = 0
    for t in range(4):
        e0, n_ev = 256 * t, 256
        tile = batch.select(list(range(e0, e0 + n_ev)))
        cap = int(bn.n_bins * n_ev / 16) + 1024                 # bench.py DeviceRun.cap
        got = run_cuda(bn, w.bz_tesla, w.layers, tile.hits_xy, tile.event_offsets, w.threshold, w.assoc_dj, w.min_hits, cap,
                       options=("reuse_staging",))
        assert got.total <= cap

        def one(le):
            acc, votes = _oracle_event(o, w, batch, e0 + le, True)
            rec_ref, h2c, nh, keep = _CACHE[e0 + le]
            assert np.array_equal(got.accum[le], acc), ("accum", e0 + le)
            c0, c1 = int(got.offsets[le]), int(got.offsets[le + 1])
            h0, h1 = int(tile.event_offsets[le]), int(tile.event_offsets[le + 1])
            assert c1 - c0 == len(rec_ref), ("count", e0 + le)
            rec = got.records[c0:c1]
            assert np.all(rec["event"] == le)
            for f in ("k", "i", "j", "votes"):
                assert np.array_equal(rec[f], rec_ref[f]), (f, e0 + le)
            assert_centroids_close(rec, rec_ref, bn)
            assert np.array_equal(got.hit_to_cand[h0:h1], np.where(h2c >= 0, h2c + c0, -1)), ("hit_to_cand", e0 + le)
            assert np.array_equal(got.cand_nhits[c0:c1], nh) and np.array_equal(got.cand_keep[c0:c1], keep), ("dedup", e0 + le)
            return votes, int(keep.sum())

        with ThreadPoolExecutor(n_threads()) as ex:
            res = list(ex.map(one, range(n_ev)))
        assert sum(r[0] for r in res) == int(got.accum.astype(np.int64).sum())
        kept_total += sum(r[1] for r in res)
        del got
    assert kept_total > 100 * 1024


@pytest.mark.parametrize("kept_only", [False, True])
def test_config_3_all_1024_events_through_the_pipeline_as_bench_runs_it(kept_only):
    w, batch = _batch()
    bn = w.binning
    missing = [e for e in range(batch.n_events) if e not in _CACHE]
    if missing:                                                 # run alone: the oracle results of test (a) are not there
        o = Oracle.from_binning(bn, w.bz_tesla)
        with ThreadPoolExecutor(n_threads()) as ex:
            list(ex.map(lambda e: _oracle_event(o, w, batch, e, False), missing))
    counts = np.array([len(_CACHE[e][0]) for e in range(batch.n_events)], np.int64)
    off_ref = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
    total = int(off_ref[-1])
    keep_ref = np.concatenate([_CACHE[e][3] for e in range(batch.n_events)])
    nh_ref = np.concatenate([_CACHE[e][2] for e in range(batch.n_events)])
    h2c_ref = np.concatenate([np.where(_CACHE[e][1] >= 0, _CACHE[e][1] + off_ref[e], -1) for e in range(batch.n_events)]).astype(np.int32)

    tile_events, n_streams = 32, 4                              # bench.py --e2e-tile-events, --streams
    off = batch.event_offsets.astype(np.int64)
    max_hits = max(int(off[e0 + tile_events] - off[e0]) for e0 in range(0, batch.n_events, tile_events))
    tile_cap = int(bn.n_bins * tile_events / 16) + 1024
    total_cap = total + 1024
    pipe = HoughPipeline.from_workload(w, tile_events, max_hits, tile_cap, n_streams)
    if kept_only:
        pipe.set_option("kept_only", 1)
    hits = torch.from_numpy(batch.hits_xy).pin_memory()
    offs = torch.from_numpy(batch.event_offsets.astype(np.int32)).pin_memory()
    h2c = torch.full((batch.n_hits,), -7, dtype=torch.int32).pin_memory()
    coff = torch.full((batch.n_events + 1,), -5, dtype=torch.int32).pin_memory()
    cands = torch.zeros((total_cap, 32), dtype=torch.uint8).pin_memory()
    nh = torch.zeros(total_cap, dtype=torch.int32).pin_memory()
    keep = torch.zeros(total_cap, dtype=torch.uint8).pin_memory()
    for _ in range(2):                                          # warm-up step, then the replayed graphs of a timed step
        over = pipe.run_host(hits, offs, w.threshold, w.assoc_dj, w.min_hits, h2c, coff, cands, total_cap, nh, keep)
        assert not over
    pipe.close()
    got = cands.numpy().view(CAND_DTYPE).reshape(-1)
    h2c, coff, nh, keep = h2c.numpy(), coff.numpy(), nh.numpy(), keep.numpy()
    ev_of = np.repeat(np.arange(batch.n_events, dtype=np.int32), counts)
    if not kept_only:
        assert np.array_equal(coff, off_ref)
        assert np.array_equal(got["event"][:total], ev_of)
        for f in ("k", "i", "j", "votes"):
            assert np.array_equal(got[f][:total], np.concatenate([_CACHE[e][0][f] for e in range(batch.n_events)])), f
        assert_centroids_close(got[:total], np.concatenate([_CACHE[e][0] for e in range(batch.n_events)]), bn)
        assert np.array_equal(h2c, h2c_ref)
        assert np.array_equal(nh[:total], nh_ref) and np.array_equal(keep[:total], keep_ref)
    else:
        kmask = keep_ref.astype(bool)
        n_kept = int(kmask.sum())
        new_index = (np.cumsum(kmask) - 1).astype(np.int32)
        kept_off = np.concatenate([[0], np.cumsum(kmask)])[off_ref].astype(np.int32)
        assert np.array_equal(coff, kept_off)
        rec = np.concatenate([_CACHE[e][0] for e in range(batch.n_events)])[kmask]
        assert np.array_equal(got["event"][:n_kept], ev_of[kmask])
        for f in ("k", "i", "j", "votes"):
            assert np.array_equal(got[f][:n_kept], rec[f]), f
        assert_centroids_close(got[:n_kept], rec, bn)
        assert np.array_equal(h2c, np.where(h2c_ref >= 0, new_index[np.maximum(h2c_ref, 0)], -1))
        assert np.array_equal(nh[:n_kept], nh_ref[kmask]) and (keep[:n_kept] == 1).all()
