"""-m gpu: circle fit of the assigned hits (hough_fit_circles, D11) vs the CPU oracle.

Hit counts and fit flags are exact; the fitted parameters come from moment sums accumulated with double-precision atomics
(order not fixed), so they are compared to 1e-7 relative / absolute: rounding of the sums (~1e-16 relative) times the
conditioning of the 3x3 normal equations for ~10 hits at radii up to 110 cm (<= ~1e8)."""
import numpy as np
import pytest
import torch

from oracle import Oracle
from workloads import generate_events, get_workload

pytestmark = pytest.mark.gpu

from paper_1311_2769_b200 import HoughPlan, alloc_candidates, hough_fit_circles  # noqa: E402


@pytest.mark.parametrize("cfg,events", [(1, [0]), (5, [0]), (6, [0]), (3, [4, 5, 6])])
def test_fit_chain_matches_oracle(cfg, events):
    w = get_workload(cfg)
    batch = generate_events(w, events=events) if w.n_events > 1 else generate_events(w)
    n_ev = batch.n_events
    o = Oracle.from_binning(w.binning, w.bz_tesla)
    acc, _ = o.vote(batch.hits_xy, batch.event_offsets)
    ref = o.find_peaks(acc, w.threshold)
    h2c_ref, nh_ref, keep_ref = o.assign_indexed(batch.hits_xy, batch.event_offsets, ref, w.assoc_dj, w.min_hits)
    fit_ref, nfit_ref = o.fit_circles(batch.hits_xy, h2c_ref, ref, keep_ref)
    assert (nfit_ref > 0).sum() >= 2

    plan = HoughPlan.from_workload(w, max_hits=batch.n_hits, max_events=n_ev)
    d_hits = torch.from_numpy(batch.hits_xy).cuda()
    d_off = torch.from_numpy(batch.event_offsets).cuda()
    accum = plan.alloc_accum(n_ev)
    cap = ref.total + 11
    cands = alloc_candidates(cap)
    coff = torch.zeros(n_ev + 1, dtype=torch.int32, device="cuda")
    h2c = torch.empty(batch.n_hits, dtype=torch.int32, device="cuda")
    nh = torch.empty(cap, dtype=torch.int32, device="cuda")
    keep = torch.empty(cap, dtype=torch.uint8, device="cuda")
    plan.vote(d_hits, d_off, accum)
    plan.find_peaks(accum, n_ev, w.threshold, cands, cap, coff)
    plan.assign_hits(d_hits, d_off, cands, coff, cap, w.assoc_dj, w.min_hits, h2c, nh, keep)
    work = torch.full((cap, 9), 3.0, dtype=torch.float64, device="cuda")          # must be zeroed by the call
    fit = torch.full((cap, 4), -1.0, dtype=torch.float64, device="cuda")
    nfit = torch.full((cap,), -77, dtype=torch.int32, device="cuda")
    hough_fit_circles(plan, d_hits, h2c, cands, coff, n_ev, cap, keep, work, fit, nfit)
    torch.cuda.synchronize()
    got_fit, got_n = fit.cpu().numpy(), nfit.cpu().numpy()
    assert np.array_equal(got_n[:ref.total], nfit_ref) and not got_n[ref.total:].any() and not got_fit[ref.total:].any()
    ok = nfit_ref > 0
    dphi = np.angle(np.exp(1j * (got_fit[:ref.total, 0] - fit_ref[:, 0])))
    assert np.all(np.abs(dphi[ok]) < 1e-7)
    for col in (1, 2, 3):
        g, r = got_fit[:ref.total, col][ok], fit_ref[:, col][ok]
        assert np.all(np.abs(g - r) <= 1e-7 * np.maximum(1.0, np.abs(r))), col
    assert not got_fit[:ref.total][~ok].any()
    # the fitted circles describe the assigned hits: rms distance of the hits to their circle is small for real tracks
    plan.close()


def test_fit_without_keep_flags_and_empty_inputs():
    w = get_workload(0)
    batch = generate_events(w)
    o = Oracle.from_binning(w.binning, w.bz_tesla)
    acc, _ = o.vote(batch.hits_xy, batch.event_offsets)
    ref = o.find_peaks(acc, w.threshold)
    h2c_ref, _, _ = o.assign_indexed(batch.hits_xy, batch.event_offsets, ref, 1, 0, apply_dedup=False)
    fit_ref, nfit_ref = o.fit_circles(batch.hits_xy, h2c_ref, ref, None)
    plan = HoughPlan.from_workload(w, max_hits=batch.n_hits, max_events=1)
    cap = ref.total
    cands = alloc_candidates(cap)
    cands[:cap].copy_(torch.from_numpy(np.ascontiguousarray(ref.records).view(np.uint8).reshape(cap, 32)))
    coff = torch.from_numpy(ref.offsets.astype(np.int32)).cuda()
    d_hits = torch.from_numpy(batch.hits_xy).cuda()
    h2c = torch.from_numpy(h2c_ref).cuda()
    work = torch.empty((cap, 9), dtype=torch.float64, device="cuda")
    fit = torch.empty((cap, 4), dtype=torch.float64, device="cuda")
    nfit = torch.empty((cap,), dtype=torch.int32, device="cuda")
    hough_fit_circles(plan, d_hits, h2c, cands, coff, 1, cap, None, work, fit, nfit)
    hough_fit_circles(plan, d_hits[:0], h2c[:0], cands, coff, 1, 0, None, None, None, None)   # capacity 0: nothing to do
    torch.cuda.synchronize()
    assert np.array_equal(nfit.cpu().numpy(), nfit_ref)
    assert np.allclose(fit.cpu().numpy(), fit_ref, rtol=1e-7, atol=1e-7)
    plan.close()


def test_fit_recovers_analytic_helices_without_the_oracle():
    """The fit kernel against the geometry itself (no oracle on the expected side): noiseless helices generated from
    their D1 parameters (both charges, d0 of both signs and zero, all quadrants of phi0) must come back; the fp32
    rounding of the hit coordinates (~1e-7 relative) limits the agreement, not the solve."""
    import math
    from workloads import LAYERS_14, helix_hits
    rng = np.random.default_rng(11)
    bz = 3.8
    n_phi = 256
    tracks, hits, h2c = [], [], []
    for t in range(64):
        phi0 = rng.uniform(0, 2 * math.pi)
        qpt = rng.choice([-1.0, 1.0]) * rng.uniform(0.05, 0.9)
        d0 = 0.0 if t % 4 == 0 else rng.uniform(-3.0, 3.0)
        p = helix_hits(phi0, qpt, d0, LAYERS_14, bz)
        if len(p) < 5:
            continue
        tracks.append((phi0, qpt, d0, len(p)))
        hits.append(p)
        h2c += [len(tracks) - 1] * len(p)
    n_t = len(tracks)
    assert n_t > 40
    hits = np.concatenate(hits)
    perm = rng.permutation(len(hits))
    hits, h2c = hits[perm], np.asarray(h2c, np.int32)[perm]
    rec = np.zeros(n_t, dtype=[("event", "<i4"), ("k", "<i4"), ("i", "<i4"), ("j", "<i4"), ("votes", "<i4"),
                               ("phi0", "<f4"), ("qpt", "<f4"), ("d0", "<f4")])
    for c, (phi0, _, _, _) in enumerate(tracks):
        rec[c]["i"] = int(phi0 / (2 * math.pi) * n_phi) % n_phi        # the candidate's column orients the circle
    plan = HoughPlan(n_phi, 128, 1, -1.0, 1.0, -20.0, 20.0, 0, bz, LAYERS_14, max_hits=len(hits), max_events=1)
    cands = alloc_candidates(n_t)
    cands[:n_t].copy_(torch.from_numpy(rec.view(np.uint8).reshape(n_t, 32)))
    coff = torch.tensor([0, n_t], dtype=torch.int32, device="cuda")
    work = torch.empty((n_t, 9), dtype=torch.float64, device="cuda")
    fit = torch.empty((n_t, 4), dtype=torch.float64, device="cuda")
    nfit = torch.empty((n_t,), dtype=torch.int32, device="cuda")
    hough_fit_circles(plan, torch.from_numpy(hits).cuda(), torch.from_numpy(h2c).cuda(), cands, coff, 1, n_t, None, work,
                      fit, nfit)
    torch.cuda.synchronize()
    f, n = fit.cpu().numpy(), nfit.cpu().numpy()
    K = 0.00299792458
    for c, (phi0, qpt, d0, nh) in enumerate(tracks):
        assert n[c] == nh
        assert abs(np.angle(np.exp(1j * (f[c, 0] - phi0)))) < 2e-5, (c, f[c], tracks[c])
        assert abs(f[c, 1] - qpt) < 2e-5 * max(1.0, abs(qpt)) + 2e-5
        assert abs(f[c, 2] - d0) < 2e-4
        assert abs(f[c, 3] - 1.0 / (abs(qpt) * K * bz)) < 2e-5 * f[c, 3] + 1e-3
    plan.close()
