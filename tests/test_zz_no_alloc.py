"""-m gpu: hough_fit_circles_static, the circle fit for callers that cannot allocate device memory.

Why the entry point exists: an event loop with a fixed time budget per event (the trigger setting of the paper) must not reach
cudaMalloc / cudaFree once it is live -- they take unbounded time and stall every stream of the device -- and a plug-in inside
an application whose GPU memory is owned by another memory manager has nowhere to take scratch from.  hough_fit_circles wants
a plan (its creation allocates) and a caller-made work buffer; the static variant wants neither and keeps its moment sums
in one fixed array per GPU inside the library (at most FIT_STATIC_MAX_CANDIDATES candidates per call).

What is checked: the static variant against the existing hough_fit_circles on the same device inputs, twice in a row with
DIFFERENT inputs, so that the second call runs on an array still holding the first call's sums (every call has to clear
the rows it uses).  Hit counts and fit flags must be equal; the parameters agree to the 1e-7 of tests/test_gpu_fit.py
(both paths sum with double atomics in no fixed order).  A request beyond the fixed limit must be refused, not truncated.

This file sorts last on purpose (pytest -x stops at the first failure, so a failure here cannot hide another test), and it
must pass alone in a fresh process as well as after the rest of the suite: it makes no assumption on what ran before."""
import numpy as np
import pytest
import torch

from workloads import generate_events, get_workload

pytestmark = pytest.mark.gpu

from paper_1311_2769_b200 import (FIT_STATIC_MAX_CANDIDATES, HoughError, HoughPlan, alloc_candidates,  # noqa: E402
                                  hough_fit_circles, hough_fit_circles_static)


def _chain(cfg, events):
    """vote -> peaks -> assign through the existing calls; returns what a fit call needs, all on the device."""
    w = get_workload(cfg)
    batch = generate_events(w, events=events) if w.n_events > 1 else generate_events(w)
    n_ev = batch.n_events
    plan = HoughPlan.from_workload(w, max_hits=batch.n_hits, max_events=n_ev)
    d_hits = torch.from_numpy(batch.hits_xy).cuda()
    d_off = torch.from_numpy(batch.event_offsets).cuda()
    accum = plan.alloc_accum(n_ev)
    cap = FIT_STATIC_MAX_CANDIDATES            # config 3 makes ~25 600 candidates per event: two events fit the fixed array
    cands = alloc_candidates(cap)
    coff = torch.zeros(n_ev + 1, dtype=torch.int32, device="cuda")
    h2c = torch.empty(batch.n_hits, dtype=torch.int32, device="cuda")
    nh = torch.empty(cap, dtype=torch.int32, device="cuda")
    keep = torch.empty(cap, dtype=torch.uint8, device="cuda")
    plan.vote(d_hits, d_off, accum)
    plan.find_peaks(accum, n_ev, w.threshold, cands, cap, coff)
    plan.assign_hits(d_hits, d_off, cands, coff, cap, w.assoc_dj, w.min_hits, h2c, nh, keep)
    torch.cuda.synchronize()
    total = int(coff[-1].item())
    assert 0 < total <= cap
    return w, plan, d_hits, h2c, cands, coff, n_ev, cap, keep, total


def _compare(w, plan, d_hits, h2c, cands, coff, n_ev, cap, keep, total):
    """One call of each path on the same inputs; the static one must reproduce the existing one."""
    work = torch.empty((cap, 9), dtype=torch.float64, device="cuda")
    fit_a = torch.full((cap, 4), -1.0, dtype=torch.float64, device="cuda")
    n_a = torch.full((cap,), -77, dtype=torch.int32, device="cuda")
    hough_fit_circles(plan, d_hits, h2c, cands, coff, n_ev, cap, keep, work, fit_a, n_a)
    fit_b = torch.full((cap, 4), -2.0, dtype=torch.float64, device="cuda")
    n_b = torch.full((cap,), -78, dtype=torch.int32, device="cuda")
    hough_fit_circles_static(w.binning.n_phi, w.bz_tesla, d_hits, h2c, cands, coff, n_ev, cap, keep, fit_b, n_b)
    torch.cuda.synchronize()
    fa, na, fb, nb = fit_a.cpu().numpy(), n_a.cpu().numpy(), fit_b.cpu().numpy(), n_b.cpu().numpy()
    assert np.array_equal(na, nb)
    assert (na[:total] > 0).sum() >= 2, "the case must fit some tracks"
    assert not nb[total:].any() and not fb[total:].any()
    dphi = np.angle(np.exp(1j * (fa[:, 0] - fb[:, 0])))
    assert np.all(np.abs(dphi) < 1e-7)
    for col in (1, 2, 3):
        assert np.all(np.abs(fa[:, col] - fb[:, col]) <= 1e-7 * np.maximum(1.0, np.abs(fa[:, col]))), col
    return int((na > 0).sum())


def test_static_fit_matches_the_allocating_path_on_two_calls_in_a_row():
    # call 1: two events of config 3 (~51 000 candidates, a few hundred of them kept and fitted)
    a = _chain(3, [4, 5])
    n1 = _compare(*a)
    # call 2, right after it: another event without keep flags, so other candidates land on the rows call 1 left filled
    b = list(_chain(3, [7]))
    b[8] = None
    assert _compare(*b) > 0
    # and once more the first inputs, now on top of call 2's leftovers
    assert _compare(*a) == n1
    a[1].close()
    b[1].close()


def test_static_fit_small_two_parameter_event_and_line_model():
    for cfg in (5, 6):
        c = _chain(cfg, [0])
        _compare(*c)
        c[1].close()


def test_static_fit_refuses_more_candidates_than_its_array_holds():
    w = get_workload(0)
    dummy = torch.zeros(64, dtype=torch.int32, device="cuda")
    cands = alloc_candidates(1)
    fit = torch.zeros((1, 4), dtype=torch.float64, device="cuda")
    with pytest.raises(HoughError, match="fixed scratch"):
        hough_fit_circles_static(w.binning.n_phi, w.bz_tesla, torch.zeros((0, 2), device="cuda"), dummy[:0], cands, dummy, 1,
                                 FIT_STATIC_MAX_CANDIDATES + 1, None, fit, dummy)
    torch.cuda.synchronize()
    assert not fit.any().item() and not dummy.any().item()          # nothing was enqueued
    # capacity 0 is a no-op, and the limit itself is accepted
    hough_fit_circles_static(w.binning.n_phi, w.bz_tesla, torch.zeros((0, 2), device="cuda"), dummy[:0], cands, dummy, 1, 0, None,
                             None, None)
    big_c = alloc_candidates(FIT_STATIC_MAX_CANDIDATES)
    big_f = torch.full((FIT_STATIC_MAX_CANDIDATES, 4), 5.0, dtype=torch.float64, device="cuda")
    big_n = torch.full((FIT_STATIC_MAX_CANDIDATES,), 5, dtype=torch.int32, device="cuda")
    hough_fit_circles_static(w.binning.n_phi, w.bz_tesla, torch.zeros((0, 2), device="cuda"), dummy[:0], big_c, dummy, 1,
                             FIT_STATIC_MAX_CANDIDATES, None, big_f, big_n)
    torch.cuda.synchronize()
    assert not big_f.any().item() and not big_n.any().item()        # empty candidate list: all rows reported as "no fit"
