"""-m gpu: second Hough transform (hough_vertex_vote, D10) vs the CPU oracle, bit for bit."""
import numpy as np
import pytest
import torch

from oracle import CAND_DTYPE, Oracle, OracleCandidates
from workloads import HoughBinning, generate_events, get_workload
from workloads.configs import ACC_I32

pytestmark = pytest.mark.gpu

from gpu_util import assert_centroids_close  # noqa: E402
from paper_1311_2769_b200 import HoughPlan, alloc_candidates, candidates_to_numpy, hough_vertex_vote  # noqa: E402


def _vertex_on_gpu(plan, rec, offsets, keep, capacity, d_abs_min, n_r, r_max):
    n_ev = len(offsets) - 1
    cands = alloc_candidates(max(capacity, 1))
    n_c = min(capacity, len(rec))
    if n_c:
        cands[:n_c].copy_(torch.from_numpy(np.ascontiguousarray(rec[:n_c]).view(np.uint8).reshape(n_c, 32)))
    d_off = torch.from_numpy(np.ascontiguousarray(offsets, np.int32)).cuda()
    d_keep = None if keep is None else torch.from_numpy(np.ascontiguousarray(keep, np.uint8)).cuda()
    vacc = torch.full((n_ev, plan.n_phi, n_r), 7, dtype=torch.int32, device="cuda")     # must be overwritten
    hough_vertex_vote(plan, cands, d_off, n_ev, capacity, d_keep, d_abs_min, n_r, r_max, vacc)
    torch.cuda.synchronize()
    return vacc


def test_vertex_chain_on_workload_6_bit_exact():
    """hits -> (phi0, d0) tracks -> (Phi_v, R_v) vertices, every stage on the GPU, compared with the oracle's chain."""
    w = get_workload(6)
    batch = generate_events(w)
    o = Oracle.from_binning(w.binning, w.bz_tesla)
    acc, _ = o.vote(batch.hits_xy, batch.event_offsets)
    ref = o.find_peaks(acc, w.threshold)
    h2c, nh, keep = o.assign_indexed(batch.hits_xy, batch.event_offsets, ref, w.assoc_dj, w.min_hits)
    n_r, r_max, thr_v = 32, 16.0, 6
    vacc_ref, votes = o.vertex_vote(ref, keep, 0.6, n_r, r_max)
    # GPU chain
    plan = HoughPlan.from_workload(w, max_hits=batch.n_hits, max_events=1)
    d_hits = torch.from_numpy(batch.hits_xy).cuda()
    d_off = torch.from_numpy(batch.event_offsets).cuda()
    accum = plan.alloc_accum(1)
    cap = ref.total + 9
    cands = alloc_candidates(cap)
    coff = torch.zeros(2, dtype=torch.int32, device="cuda")
    d_h2c = torch.empty(batch.n_hits, dtype=torch.int32, device="cuda")
    d_nh = torch.empty(cap, dtype=torch.int32, device="cuda")
    d_keep = torch.empty(cap, dtype=torch.uint8, device="cuda")
    plan.vote(d_hits, d_off, accum)
    plan.find_peaks(accum, 1, w.threshold, cands, cap, coff)
    plan.assign_hits(d_hits, d_off, cands, coff, cap, w.assoc_dj, w.min_hits, d_h2c, d_nh, d_keep)
    vacc = torch.empty((1, plan.n_phi, n_r), dtype=torch.int32, device="cuda")
    hough_vertex_vote(plan, cands, coff, 1, cap, d_keep, 0.6, n_r, r_max, vacc)
    vplan = HoughPlan(plan.n_phi, n_r, 1, 0.0, r_max, accum_dtype=ACC_I32, bz_tesla=0.0, max_hits=1, max_events=1, model=1)
    vcands = alloc_candidates(4096)
    vcoff = torch.zeros(2, dtype=torch.int32, device="cuda")
    vplan.find_peaks(vacc, 1, thr_v, vcands, 4096, vcoff)
    torch.cuda.synchronize()
    assert votes > 1000 and np.array_equal(vacc.cpu().numpy(), vacc_ref)
    vs = Oracle(plan.n_phi, n_r, 1, 0.0, r_max, bz_tesla=0.0, model=1)
    vref = vs.find_peaks(vacc_ref[:, None], thr_v)
    got = candidates_to_numpy(vcands, int(vcoff[1].item()))
    assert vref.total > 0 and len(got) == vref.total
    for f in ("event", "k", "i", "j", "votes"):
        assert np.array_equal(got[f], vref.records[f]), f
    assert_centroids_close(got, vref.records, HoughBinning(plan.n_phi, n_r, 1, 0.0, r_max, model=1))
    plan.close()
    vplan.close()


@pytest.mark.parametrize("shape,drange,n_r,r_max,use_keep", [
    ((256, 128), (-20.0, 20.0), 48, 25.0, True),
    ((100, 37), (-5.0, 9.0), 7, 3.0, False),               # odd sizes, asymmetric d0 range, all candidates vote
    ((1024, 64), (0.0, 30.0), 200, 40.0, True),
])
def test_vertex_vote_random_track_lists_bit_exact(shape, drange, n_r, r_max, use_keep):
    rng = np.random.default_rng(shape[0] + n_r)
    n_phi, n_d = shape
    o = Oracle(n_phi, n_d, 1, drange[0], drange[1], bz_tesla=0.0, model=1)
    counts = [150, 0, 333, 40]                              # four events, one without candidates
    offsets = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
    rec = np.zeros(offsets[-1], CAND_DTYPE)
    rec["i"] = rng.integers(0, n_phi, len(rec))
    rec["j"] = rng.integers(0, n_d, len(rec))
    keep = (rng.uniform(size=len(rec)) < 0.6).astype(np.uint8) if use_keep else None
    plan = HoughPlan(n_phi, n_d, 1, drange[0], drange[1], accum_dtype=ACC_I32, bz_tesla=0.0, max_hits=1, max_events=4, model=1)
    for capacity in (len(rec) + 5, 400):                    # 400: the list is truncated inside event 2
        cands = OracleCandidates(rec[:min(capacity, len(rec))], offsets, int(offsets[-1]))
        vacc_ref, votes = o.vertex_vote(cands, None if keep is None else keep[:min(capacity, len(rec))], 0.4, n_r, r_max,
                                        capacity=capacity)
        vacc = _vertex_on_gpu(plan, rec, offsets, keep, capacity, 0.4, n_r, r_max)
        assert votes > 0 and np.array_equal(vacc.cpu().numpy(), vacc_ref)
    plan.close()


def test_vertex_vote_rejects_a_helix_plan_and_handles_no_events():
    from paper_1311_2769_b200 import HoughError
    helix = HoughPlan(64, 32, 1, max_hits=1, max_events=1)
    with pytest.raises(HoughError):
        _vertex_on_gpu(helix, np.zeros(0, CAND_DTYPE), np.array([0, 0], np.int32), None, 0, 0.5, 8, 10.0)
    helix.close()
    line = HoughPlan(64, 32, 1, -10.0, 10.0, bz_tesla=0.0, max_hits=1, max_events=1, model=1)
    vacc = _vertex_on_gpu(line, np.zeros(0, CAND_DTYPE), np.array([0, 0], np.int32), None, 0, 0.5, 8, 10.0)
    assert not vacc.cpu().numpy().any()
    line.close()
