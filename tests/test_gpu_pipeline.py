"""-m gpu: the batched multi-event path (hough_pipeline_run_host, A6) vs the CPU oracle, event by event."""
import numpy as np
import pytest
import torch

from oracle import Oracle
from workloads import generate_events, get_workload

pytestmark = pytest.mark.gpu

from gpu_util import assert_centroids_close  # noqa: E402
from paper_1311_2769_b200 import CAND_DTYPE, HoughPipeline  # noqa: E402


def _run_pipeline(w, batch, tile_events, n_streams, tile_cap, cand_capacity, pinned=True, kept_only=False, reassign=False):
    off = batch.event_offsets.astype(np.int64)
    tiles = [(e0, min(e0 + tile_events, batch.n_events)) for e0 in range(0, batch.n_events, tile_events)]
    max_hits = max(int(off[e1] - off[e0]) for e0, e1 in tiles)
    pipe = HoughPipeline.from_workload(w, tile_events, max(max_hits, 1), tile_cap, n_streams)
    if kept_only:
        pipe.set_option("kept_only", 1)
    if reassign:
        pipe.set_option("reassign", 1)

    def host(t):
        return t.pin_memory() if pinned else t
    hits = host(torch.from_numpy(batch.hits_xy.copy()))
    offs = host(torch.from_numpy(batch.event_offsets.astype(np.int32)))
    h2c = host(torch.full((max(batch.n_hits, 1),), -7, dtype=torch.int32))
    coff = host(torch.full((batch.n_events + 1,), -5, dtype=torch.int32))
    cands = host(torch.zeros((max(cand_capacity, 1), 32), dtype=torch.uint8))
    nh = host(torch.zeros(max(cand_capacity, 1), dtype=torch.int32))
    keep = host(torch.zeros(max(cand_capacity, 1), dtype=torch.uint8))
    over = None
    for _ in range(2):                                   # second run: every lane replays / updates its graph
        over = pipe.run_host(hits, offs, w.threshold, w.assoc_dj, w.min_hits, h2c[:batch.n_hits], coff, cands, cand_capacity,
                             nh, keep)
    pipe.close()
    return over, h2c.numpy()[:batch.n_hits], coff.numpy(), cands.numpy().view(CAND_DTYPE).reshape(-1), nh.numpy(), keep.numpy()


def _oracle_per_event(w, batch, rounds=False):
    o = Oracle.from_binning(w.binning, w.bz_tesla)
    recs, h2cs, nhs, keeps, offs = [], [], [], [], [0]
    for e in range(batch.n_events):
        ev = batch.select([e])
        acc, _ = o.vote(ev.hits_xy, ev.event_offsets)
        ref = o.find_peaks(acc, w.threshold)
        if rounds:                                       # D12: the fixed point of the re-assignment rounds
            h2c, nh, keep, _ = o.assign_rounds(ev.hits_xy, ev.event_offsets, ref, w.assoc_dj, w.min_hits, max_rounds=4)
        else:
            h2c, nh, keep = o.assign_indexed(ev.hits_xy, ev.event_offsets, ref, w.assoc_dj, w.min_hits)
        r = ref.records.copy()
        r["event"] = e
        recs.append(r)
        h2cs.append(np.where(h2c >= 0, h2c + offs[-1], -1))
        nhs.append(nh)
        keeps.append(keep)
        offs.append(offs[-1] + ref.total)
    return (np.concatenate(recs), np.concatenate(h2cs).astype(np.int32), np.concatenate(nhs), np.concatenate(keeps),
            np.array(offs, np.int32))


@pytest.mark.parametrize("tile_events,n_streams,pinned", [(3, 2, True), (4, 4, True), (16, 3, False)])
def test_pipeline_matches_oracle_on_config_3_events(tile_events, n_streams, pinned):
    w = get_workload(3)
    batch = generate_events(w, events=list(range(11)))   # ragged: 11 events over tiles of 3 / 4 / 16
    rec, h2c_ref, nh_ref, keep_ref, off_ref = _oracle_per_event(w, batch)
    total = int(off_ref[-1])
    cap = total + 5
    tile_cap = int(max(off_ref[min(e0 + tile_events, 11)] - off_ref[e0] for e0 in range(0, 11, tile_events))) + 3
    over, h2c, coff, cands, nh, keep = _run_pipeline(w, batch, tile_events, n_streams, tile_cap, cap, pinned)
    assert not over
    assert np.array_equal(coff, off_ref)
    for f in ("event", "k", "i", "j", "votes"):
        assert np.array_equal(cands[f][:total], rec[f]), f
    assert_centroids_close(cands[:total], rec, w.binning)
    assert np.array_equal(h2c, h2c_ref)
    assert np.array_equal(nh[:total], nh_ref) and np.array_equal(keep[:total], keep_ref)


def test_pipeline_reports_overflow_and_keeps_true_offsets():
    w = get_workload(3)
    batch = generate_events(w, events=[0, 1, 2, 3])
    rec, h2c_ref, nh_ref, keep_ref, off_ref = _oracle_per_event(w, batch)
    total = int(off_ref[-1])
    over, h2c, coff, cands, nh, keep = _run_pipeline(w, batch, 2, 2, 1 << 20, total // 2)
    assert over                                            # caller's capacity exceeded
    assert np.array_equal(coff, off_ref)                   # true counts all the same
    n = total // 2
    for f in ("event", "k", "i", "j", "votes"):
        assert np.array_equal(cands[f][:n], rec[f][:n]), f
    over2, *_ = _run_pipeline(w, batch, 2, 2, 100, total + 5)
    assert over2                                           # per-tile capacity exceeded


def test_pipeline_empty_batch_and_empty_events():
    w = get_workload(0)
    batch = generate_events(w)
    hits = np.concatenate([batch.hits_xy, batch.hits_xy])
    offs = np.array([0, 0, batch.n_hits, batch.n_hits, 2 * batch.n_hits, 2 * batch.n_hits], np.int32)   # events 0, 2, 4 empty

    class B:
        pass
    b = B()
    b.hits_xy, b.event_offsets, b.n_hits, b.n_events = hits, offs, 2 * batch.n_hits, 5
    over, h2c, coff, cands, nh, keep = _run_pipeline(w, b, 2, 2, 4096, 4096)
    o = Oracle.from_binning(w.binning, w.bz_tesla)
    acc, _ = o.vote(batch.hits_xy, batch.event_offsets)
    ref = o.find_peaks(acc, w.threshold)
    assert not over
    assert list(coff) == [0, 0, ref.total, ref.total, 2 * ref.total, 2 * ref.total]
    assert list(cands["event"][:2 * ref.total]) == [1] * ref.total + [3] * ref.total
    h_ref, _, _ = o.assign_indexed(batch.hits_xy, batch.event_offsets, ref, w.assoc_dj, w.min_hits)
    assert np.array_equal(h2c[:batch.n_hits], h_ref)
    assert np.array_equal(h2c[batch.n_hits:], np.where(h_ref >= 0, h_ref + ref.total, -1))


@pytest.mark.parametrize("tile_events,n_streams", [(3, 2), (16, 3)])
def test_pipeline_kept_only_returns_the_compacted_kept_list(tile_events, n_streams):
    """include/hough.h "kept_only": same work, only the candidates with cand_keep = 1 come back, compacted."""
    w = get_workload(3)
    batch = generate_events(w, events=list(range(20, 31)))
    rec, h2c_ref, nh_ref, keep_ref, off_ref = _oracle_per_event(w, batch)
    kmask = keep_ref.astype(bool)
    new_index = np.cumsum(kmask) - 1
    n_kept = int(kmask.sum())
    assert 0 < n_kept < len(kmask)
    koff = np.array([int(kmask[:o].sum()) for o in off_ref], np.int32)
    h2c_kept = np.where(h2c_ref >= 0, new_index[np.maximum(h2c_ref, 0)], -1).astype(np.int32)
    tile_cap = int(max(off_ref[min(e0 + tile_events, 11)] - off_ref[e0] for e0 in range(0, 11, tile_events))) + 3
    over, h2c, coff, cands, nh, keep = _run_pipeline(w, batch, tile_events, n_streams, tile_cap, n_kept + 4, kept_only=True)
    assert not over
    assert np.array_equal(coff, koff)
    for f in ("event", "k", "i", "j", "votes"):
        assert np.array_equal(cands[f][:n_kept], rec[f][kmask]), f
    assert_centroids_close(cands[:n_kept], rec[kmask], w.binning)
    assert np.array_equal(h2c, h2c_kept)
    assert np.array_equal(nh[:n_kept], nh_ref[kmask]) and (keep[:n_kept] == 1).all()


@pytest.mark.parametrize("kept_only", [False, True])
def test_pipeline_reassign_option_runs_the_d12_round(kept_only):
    """Pipeline option "reassign": hit_to_cand / cand_nhits are the fixed point of the re-assignment rounds (D12)."""
    w = get_workload(3)
    batch = generate_events(w, events=[5, 6, 7])
    rec, h2c_ref, nh_ref, keep_ref, off_ref = _oracle_per_event(w, batch, rounds=True)
    total = int(off_ref[-1])
    tile_cap = int(max(off_ref[min(e0 + 2, 3)] - off_ref[e0] for e0 in range(0, 3, 2))) + 3
    over, h2c, coff, cands, nh, keep = _run_pipeline(w, batch, 2, 2, tile_cap, total + 5, kept_only=kept_only, reassign=True)
    assert not over
    if not kept_only:
        assert np.array_equal(coff, off_ref) and np.array_equal(h2c, h2c_ref)
        assert np.array_equal(nh[:total], nh_ref) and np.array_equal(keep[:total], keep_ref)
    else:
        kmask = keep_ref.astype(bool)
        new_index = np.cumsum(kmask) - 1
        assert np.array_equal(h2c, np.where(h2c_ref >= 0, new_index[np.maximum(h2c_ref, 0)], -1))
        assert np.array_equal(nh[:int(kmask.sum())], nh_ref[kmask])
    assert (h2c >= 0).sum() > (_oracle_per_event(w, batch)[1] >= 0).sum()     # the round did recover hits


@pytest.mark.parametrize("kept_only", [False, True])
def test_pipeline_reassign_when_every_lane_starts_on_an_empty_tile(kept_only):
    """Graphs on, option "reassign", and the FIRST tile of each lane has no hits (that tile runs un-captured and returns
    before the D12 round): the round's table is built by set_option, so the following, captured tiles must not allocate."""
    from workloads.generator import EventBatch
    w = get_workload(3)
    real = generate_events(w, events=[5, 6, 7])
    n = [int(real.event_offsets[i + 1] - real.event_offsets[i]) for i in range(3)]
    # events: empty, empty, e5, e6, empty, e7 -- tiles of one event on two lanes
    off = np.cumsum([0, 0, 0, n[0], n[1], 0, n[2]]).astype(np.int32)
    batch = EventBatch(real.hits_xy, off, None)
    rec, h2c_ref, nh_ref, keep_ref, off_ref = _oracle_per_event(w, batch, rounds=True)
    total = int(off_ref[-1])
    tile_cap = int(np.diff(off_ref).max()) + 3
    over, h2c, coff, cands, nh, keep = _run_pipeline(w, batch, 1, 2, tile_cap, total + 5, kept_only=kept_only, reassign=True)
    assert not over
    if not kept_only:
        assert np.array_equal(coff, off_ref) and np.array_equal(h2c, h2c_ref)
        assert np.array_equal(nh[:total], nh_ref) and np.array_equal(keep[:total], keep_ref)
        assert np.array_equal(cands["event"][:total], rec["event"])
    else:
        kmask = keep_ref.astype(bool)
        new_index = np.cumsum(kmask) - 1
        assert np.array_equal(h2c, np.where(h2c_ref >= 0, new_index[np.maximum(h2c_ref, 0)], -1))
        assert np.array_equal(nh[:int(kmask.sum())], nh_ref[kmask])
