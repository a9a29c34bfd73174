"""-m gpu: hough_event_run (one event, one launch of a thread-block cluster) vs the CPU oracle, element by element, and vs the
three general calls.  Bar: accumulator, candidate list, hit_to_cand, cand_nhits, cand_keep bit-exact; centroids 1e-5."""
from dataclasses import replace

import numpy as np
import pytest
import torch

from oracle import Oracle
from workloads import HoughBinning, generate_events, get_workload
from workloads.configs import ACC_I32, ACC_U16

pytestmark = pytest.mark.gpu

from gpu_util import assert_centroids_close  # noqa: E402
from paper_1311_2769_b200 import HoughPlan, alloc_candidates, candidates_to_numpy, kernel_launches  # noqa: E402


def _run(w, batch, capacity, general=False, threshold=None, assoc_dj=None, min_hits=None, cluster=True):
    bn = w.binning
    plan = HoughPlan.from_workload(w, max_hits=max(batch.n_hits, 1), max_events=1)
    if general:
        plan.set_option("event_general", 1)
    elif cluster:
        plan.set_option("event_cluster", 1)                        # the cluster kernel whenever it fits (no work gate)
    d_hits = torch.from_numpy(batch.hits_xy).cuda() if batch.n_hits else torch.zeros((1, 2), dtype=torch.float32, device="cuda")[:0]
    d_off = torch.from_numpy(batch.event_offsets).cuda()
    accum = plan.alloc_accum(1)
    accum.fill_(5)
    cands = alloc_candidates(max(capacity, 1))
    coff = torch.full((2,), -3, dtype=torch.int32, device="cuda")
    h2c = torch.full((max(batch.n_hits, 1),), -7, dtype=torch.int32, device="cuda")
    nh = torch.full((max(capacity, 1),), -3, dtype=torch.int32, device="cuda")
    keep = torch.full((max(capacity, 1),), 9, dtype=torch.uint8, device="cuda")
    n0 = kernel_launches()
    plan.event_run(d_hits, d_off, accum, w.threshold if threshold is None else threshold, cands, capacity, coff,
                   w.assoc_dj if assoc_dj is None else assoc_dj, w.min_hits if min_hits is None else min_hits, h2c, nh, keep)
    torch.cuda.synchronize()
    launches = kernel_launches() - n0
    off = coff.cpu().numpy()
    n_c = min(int(off[1]), capacity)
    out = dict(accum=accum.cpu().numpy(), off=off, rec=candidates_to_numpy(cands, n_c), h2c=h2c[:batch.n_hits].cpu().numpy(),
               nh=nh[:capacity].cpu().numpy(), keep=keep[:capacity].cpu().numpy(), launches=launches)
    plan.close()
    return out


def _check(w, batch, capacity=None, **kw):
    bn = w.binning
    o = Oracle.from_binning(bn, w.bz_tesla)
    thr = kw.get("threshold", w.threshold)
    dj = kw.get("assoc_dj", w.assoc_dj)
    mh = kw.get("min_hits", w.min_hits)
    acc, votes = o.vote(batch.hits_xy, batch.event_offsets)
    ref = o.find_peaks(acc, thr)
    cap = ref.total + 3 if capacity is None else capacity
    got = _run(w, batch, cap, **kw)
    exp_acc = acc.astype(np.uint16) if bn.accum_dtype == ACC_U16 else acc
    assert np.array_equal(got["accum"].reshape(exp_acc.shape), exp_acc), "accumulator differs"
    assert list(got["off"]) == [0, ref.total]
    n_c = min(cap, ref.total)
    for f in ("event", "k", "i", "j", "votes"):
        assert np.array_equal(got["rec"][f], ref.records[f][:n_c]), f
    assert_centroids_close(got["rec"], ref.records[:n_c], bn)
    ref_c = ref if n_c == ref.total else o.find_peaks(acc, thr, capacity=cap)
    h2c, nh, keep = o.assign_indexed(batch.hits_xy, batch.event_offsets, ref_c, dj, mh, capacity=cap)
    assert np.array_equal(got["h2c"], h2c), "hit_to_cand differs"
    assert np.array_equal(got["nh"][:n_c], nh) and np.array_equal(got["keep"][:n_c], keep)
    assert not got["nh"][n_c:].any() and not got["keep"][n_c:].any()
    return got


@pytest.mark.parametrize("cfg", [0, 5, 6])
def test_event_run_two_parameter_workloads_one_launch(cfg):
    w = get_workload(cfg)
    if cfg == 5:
        w = w.with_tracks(200)                                    # 2000 hits: within the one-launch limit
    got = _check(w, generate_events(w))
    assert got["launches"] == 1                                   # the whole path was a single kernel launch
    gen = _run(w, generate_events(w), len(got["nh"]), general=True)
    assert gen["launches"] > 5
    for key in ("accum", "off", "h2c", "nh", "keep"):
        assert np.array_equal(got[key], gen[key]), key
    assert np.array_equal(got["rec"], gen["rec"])                 # records byte for byte, centroids included


def test_event_run_work_gate():
    """Without the test switch the cluster is taken only while hits x longest window stays small: config 0 yes, the
    zero-field workload (windows of up to 512 columns, 2200 hits) no.  Same results either way."""
    w0, w6 = get_workload(0), get_workload(6)
    assert _check(w0, generate_events(w0), cluster=False)["launches"] == 1
    assert _check(w6, generate_events(w6), cluster=False)["launches"] > 5


def test_event_run_three_parameter_space_takes_the_general_calls():
    w = get_workload(1)
    got = _check(w, generate_events(w))
    assert got["launches"] > 5


@pytest.mark.parametrize("n_tracks", [50, 200, 3000])
def test_event_run_toy_sizes(n_tracks):
    w = get_workload(5).with_tracks(n_tracks)
    got = _check(w, generate_events(w))
    assert (got["launches"] == 1) == (10 * n_tracks <= 2560)      # above 2560 hits: the three general calls


@pytest.mark.parametrize("shape", [(64, 32, ACC_I32), (256, 256, ACC_U16), (1024, 128, ACC_I32), (100, 77, ACC_I32),
                                   (2048, 64, ACC_U16), (4, 16, ACC_I32)])
def test_event_run_binnings_and_cluster_sizes(shape):
    """1, 2, 4 and 8 CTAs per cluster, odd sizes, slabs whose last CTA is short, both accumulator types."""
    n_phi, n_q, dt = shape
    w0 = get_workload(5)
    w = replace(w0, binning=HoughBinning(n_phi, n_q, 1, -0.9, 1.1, accum_dtype=dt), n_prompt=300, n_noise=200, threshold=6)
    b = generate_events(w)
    _check(w, b, min_hits=5)
    _check(w, b, capacity=7, min_hits=5)                          # truncated list: only ranks < capacity take part
    _check(w, b, assoc_dj=3, min_hits=4, threshold=5)


def test_event_run_degenerate_inputs():
    w = get_workload(0)
    b = generate_events(w)
    empty = type(b)(np.zeros((0, 2), np.float32), np.zeros(2, np.int32), None)
    got = _check(w, empty)
    assert list(got["off"]) == [0, 0]
    hits = b.hits_xy.copy()
    hits[3] = [np.nan, 1.0]; hits[4] = [np.inf, -np.inf]; hits[5] = [0.0, 0.0]; hits[6] = [1e30, 1e30]
    bad = type(b)(hits, b.event_offsets, None)
    _check(w, bad)
    _check(w, b, capacity=0)                                       # no candidate buffer at all
