"""-m gpu: hough_reassign_hits (D12 re-assignment rounds, P:L33 / P:L29) through the C ABI vs orc_assign_rounds.

Bar: hit_to_cand, cand_nhits, cand_keep bit-exact, on all three association paths (candidate-centric default,
plan option "reassign_walk", full scan)."""
import numpy as np
import pytest
import torch

from oracle import Oracle, OracleCandidates
from workloads import generate_events, get_workload

pytestmark = pytest.mark.gpu

from gpu_util import oracle_vote_parallel  # noqa: E402
from paper_1311_2769_b200 import HoughPlan, alloc_candidates, candidates_to_numpy  # noqa: E402


def _run(w, batch, max_rounds, options=(), min_hits=None, assoc_dj=None, capacity=None, threshold=None, plan_events=None):
    bn = w.binning
    n_hits, n_ev = batch.n_hits, len(batch.event_offsets) - 1
    min_hits = w.min_hits if min_hits is None else min_hits
    assoc_dj = w.assoc_dj if assoc_dj is None else assoc_dj
    threshold = w.threshold if threshold is None else threshold
    plan = HoughPlan.from_workload(w, max_hits=n_hits, max_events=n_ev if plan_events is None else plan_events)
    for key in options:
        plan.set_option(key, 1)
    d_hits = torch.from_numpy(batch.hits_xy).cuda()
    d_off = torch.from_numpy(batch.event_offsets).cuda()
    accum = plan.alloc_accum(n_ev)
    plan.vote(d_hits, d_off, accum)
    cand_off = torch.zeros(n_ev + 1, dtype=torch.int32, device="cuda")
    plan.find_peaks(accum, n_ev, threshold, None, 0, cand_off)
    total = int(cand_off[n_ev].item())
    cap = total + 5 if capacity is None else capacity
    cands = alloc_candidates(max(cap, 1))
    plan.find_peaks(accum, n_ev, threshold, cands, cap, cand_off)
    h2c = torch.full((n_hits,), -7, dtype=torch.int32, device="cuda")
    nh = torch.full((max(cap, 1),), -3, dtype=torch.int32, device="cuda")
    keep = torch.full((max(cap, 1),), 9, dtype=torch.uint8, device="cuda")
    plan.assign_hits(d_hits, d_off, cands, cand_off, cap, assoc_dj, min_hits, h2c, nh, keep)
    keep_before = keep.clone()
    plan.reassign_hits(d_hits, d_off, cands, cand_off, cap, assoc_dj, max_rounds, h2c, nh, keep)
    torch.cuda.synchronize()
    assert torch.equal(keep, keep_before)                      # the kept set is not touched
    n_c = min(total, cap)
    rec = candidates_to_numpy(cands, n_c)
    out = (h2c.cpu().numpy(), nh[:n_c].cpu().numpy(), keep[:n_c].cpu().numpy(), rec, cand_off.cpu().numpy(), cap)
    plan.close()
    return out


def _check(w, batch, max_rounds=4, options=(), **kw):
    h2c, nh, keep, rec, off, cap = _run(w, batch, max_rounds, options, **kw)
    o = Oracle.from_binning(w.binning, w.bz_tesla)
    ref_c = OracleCandidates(rec, off, int(off[-1]))            # the list itself is covered by the peak parity tests
    rh, rn, rk, rounds = o.assign_rounds(batch.hits_xy, batch.event_offsets, ref_c, kw.get("assoc_dj", w.assoc_dj),
                                         kw.get("min_hits", w.min_hits), max_rounds=max_rounds, capacity=cap)
    kw.pop("plan_events", None)
    assert rounds <= 2
    assert np.array_equal(h2c, rh), "hit_to_cand differs"
    assert np.array_equal(nh, rn) and np.array_equal(keep, rk)
    return h2c, rh


@pytest.mark.parametrize("options", [(), ("reassign_walk",), ("fullscan",)])
@pytest.mark.parametrize("cfg", [0, 1, 5])
def test_reassign_bit_exact_single_events(cfg, options):
    w = get_workload(cfg)
    b = generate_events(w)
    h2c, _ = _check(w, b, options=options)
    if cfg != 0:
        h9 = _run(w, b, 1, options)[0]                          # max_rounds = 1: the call returns at once (D9)
        assert (h2c >= 0).sum() > (h9 >= 0).sum()               # the extra round does recover hits


@pytest.mark.parametrize("options", [(), ("reassign_walk",)])
def test_reassign_batched_config3_events(options):
    w = get_workload(3).scaled(3)
    _check(w, generate_events(w), options=options)


@pytest.mark.parametrize("options", [(), ("reassign_walk",), ("fullscan",)])
def test_reassign_variants(options):
    w = get_workload(1)
    b = generate_events(w)
    _check(w, b, options=options, assoc_dj=3, min_hits=5, threshold=6)       # wide association window, many candidates
    _check(w, b, options=options, assoc_dj=0, min_hits=9)                    # exact-bin association
    _check(w, b, options=options, min_hits=100)                              # nothing survives: nothing to re-assign
    _check(w, b, options=options, capacity=40)                               # truncated list: only ranks < capacity take part


@pytest.mark.parametrize("options", [(), ("prepare_reassign",)])
def test_reassign_on_a_plan_sized_for_many_events_uses_coarse_sectors(options):
    """A plan declared for 2048 events keeps its per-call key-start table small by staging with fewer phi sectors than phi0
    columns (plan.cu, HOUGH_STAGE_TABLE_BYTES): the candidate-centric D12 round must not depend on the sector count."""
    w = get_workload(3).scaled(3)
    _check(w, generate_events(w), options=options, plan_events=2048)


def test_reassign_captured_in_a_graph_on_its_first_call():
    """include/hough.h: a hough_reassign_hits call on a capturing stream never allocates or synchronises.  First call of a
    fresh plan under stream capture (no table yet: the columns are re-walked), replayed, then the same call un-captured
    (builds the table, candidate-centric path): both must give the oracle's fixed point."""
    w = get_workload(3).scaled(2)
    batch = generate_events(w)
    n_hits, n_ev = batch.n_hits, batch.n_events
    plan = HoughPlan.from_workload(w, max_hits=n_hits, max_events=n_ev)
    d_hits = torch.from_numpy(batch.hits_xy).cuda()
    d_off = torch.from_numpy(batch.event_offsets).cuda()
    accum = plan.alloc_accum(n_ev)
    plan.vote(d_hits, d_off, accum)
    cand_off = torch.zeros(n_ev + 1, dtype=torch.int32, device="cuda")
    plan.find_peaks(accum, n_ev, w.threshold, None, 0, cand_off)
    cap = int(cand_off[n_ev].item()) + 5
    cands = alloc_candidates(cap)
    plan.find_peaks(accum, n_ev, w.threshold, cands, cap, cand_off)
    h2c = torch.empty(n_hits, dtype=torch.int32, device="cuda")
    nh = torch.empty(cap, dtype=torch.int32, device="cuda")
    keep = torch.empty(cap, dtype=torch.uint8, device="cuda")
    plan.assign_hits(d_hits, d_off, cands, cand_off, cap, w.assoc_dj, w.min_hits, h2c, nh, keep)
    torch.cuda.synchronize()
    h2c0, nh0 = h2c.clone(), nh.clone()
    rec = candidates_to_numpy(cands, cap - 5)
    off = cand_off.cpu().numpy()
    o = Oracle.from_binning(w.binning, w.bz_tesla)
    rh, rn, rk, _ = o.assign_rounds(batch.hits_xy, batch.event_offsets, OracleCandidates(rec, off, int(off[-1])), w.assoc_dj,
                                    w.min_hits, max_rounds=2, capacity=cap)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):                                   # capture_error_mode "global": a cudaMalloc here would fail
        plan.reassign_hits(d_hits, d_off, cands, cand_off, cap, w.assoc_dj, 2, h2c, nh, keep)
    for _ in range(2):                                          # the graph is replayable on restored inputs
        h2c.copy_(h2c0)
        nh.copy_(nh0)
        g.replay()
        torch.cuda.synchronize()
        assert np.array_equal(h2c.cpu().numpy(), rh) and np.array_equal(nh[:cap - 5].cpu().numpy(), rn)
    h2c.copy_(h2c0)
    nh.copy_(nh0)
    plan.reassign_hits(d_hits, d_off, cands, cand_off, cap, w.assoc_dj, 2, h2c, nh, keep)      # un-captured: table path
    torch.cuda.synchronize()
    assert np.array_equal(h2c.cpu().numpy(), rh) and np.array_equal(nh[:cap - 5].cpu().numpy(), rn)
    assert (h2c >= 0).sum().item() > (h2c0 >= 0).sum().item()
    plan.close()


def test_reassign_argument_errors():
    from paper_1311_2769_b200 import HoughError
    w = get_workload(0)
    b = generate_events(w)
    plan = HoughPlan.from_workload(w, max_hits=b.n_hits, max_events=1)
    d_hits = torch.from_numpy(b.hits_xy).cuda()
    d_off = torch.from_numpy(b.event_offsets).cuda()
    cands = alloc_candidates(16)
    off = torch.zeros(2, dtype=torch.int32, device="cuda")
    h2c = torch.full((b.n_hits,), -1, dtype=torch.int32, device="cuda")
    nh = torch.zeros(16, dtype=torch.int32, device="cuda")
    keep = torch.zeros(16, dtype=torch.uint8, device="cuda")
    with pytest.raises(HoughError):
        plan.reassign_hits(d_hits, d_off, cands, off, 16, 1, 0, h2c, nh, keep)          # max_rounds < 1
    with pytest.raises(HoughError):
        plan.reassign_hits(d_hits, d_off, cands, off, 16, 16, 2, h2c, nh, keep)         # assoc_dj > 15
    plan.reassign_hits(d_hits, d_off, cands, off, 16, 1, 2, h2c, nh, keep)              # empty list: no-op
    torch.cuda.synchronize()
    assert (h2c == -1).all()
    plan.close()
