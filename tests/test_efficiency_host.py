"""Host-side pieces of the efficiency / fake-rate report: truth labels, truth parameters, matching."""
import math

import numpy as np

from workloads import generate_events, get_workload, K_GEV_PER_T_CM
from paper_1311_2769_b200.efficiency import efficiency_report, truth_bins, truth_parameters
from oracle import CAND_DTYPE


def test_hit_track_labels_sit_on_their_circles():
    for cfg in (1, 5):
        w = get_workload(cfg)
        b = generate_events(w, want_truth=True)
        t = b.truth[0]
        lab = t["hit_track"]
        assert len(lab) == b.n_hits and (lab >= -1).all() and (lab == -1).sum() == t["n_noise"]
        rho = t["rho"]
        cx = t["start_x"] - np.sin(t["direction"]) / rho
        cy = t["start_y"] + np.cos(t["direction"]) / rho
        sel = lab >= 0
        res = np.hypot(b.hits_xy[sel, 0] - cx[lab[sel]], b.hits_xy[sel, 1] - cy[lab[sel]]) - 1.0 / np.abs(rho[lab[sel]])
        assert np.abs(res).max() < 8 * w.sigma_rphi_cm + 2e-3          # smear along r-phi + fp32 rounding of the coordinates
        # the labels do not disturb the generated hits
        assert np.array_equal(generate_events(w).hits_xy, b.hits_xy)


def test_truth_parameters_recover_the_d1_convention():
    rng = np.random.default_rng(3)
    bz = 3.8
    n = 200
    phi0 = rng.uniform(0, 2 * math.pi, n)
    qpt = rng.uniform(0.05, 1.0, n) * rng.choice([-1.0, 1.0], n)
    d0 = rng.uniform(-15, 15, n)
    rho = -qpt * K_GEV_PER_T_CM * bz
    nx, ny = -np.sin(phi0), np.cos(phi0)
    cx, cy = d0 * nx + nx / rho, d0 * ny + ny / rho                     # centre = PCA + n_hat / rho  (D1)
    alpha = rng.uniform(-0.4, 0.4, n)                                   # start somewhere else on the same circle
    psi = phi0 + alpha
    sx, sy = cx + np.sin(psi) / rho, cy - np.cos(psi) / rho
    q = np.sign(qpt)
    out = truth_parameters(dict(start_x=sx, start_y=sy, direction=psi, charge=q, pt=1.0 / np.abs(qpt)), bz)
    assert np.allclose(out["qpt"], qpt, rtol=1e-12)
    assert np.allclose(np.angle(np.exp(1j * (out["phi0"] - phi0))), 0, atol=1e-9)
    assert np.allclose(out["d0"], d0, atol=1e-8)
    # straight tracks
    out = truth_parameters(dict(start_x=d0 * nx + 3 * np.cos(phi0), start_y=d0 * ny + 3 * np.sin(phi0), direction=phi0,
                                charge=q, pt=np.ones(n)), 0.0)
    assert np.allclose(out["d0"], d0, atol=1e-10) and np.allclose(out["phi0"], phi0)


def test_report_counts_found_fake_duplicate():
    w = get_workload(0)
    bn = w.binning
    truth = dict(start_x=np.zeros(3), start_y=np.zeros(3), direction=np.array([0.3, 2.0, 4.0]), charge=np.array([1., -1., 1.]),
                 pt=np.array([2.0, 4.0, 5.0]), hit_track=np.array([0] * 10 + [1] * 10 + [2] * 4 + [-1] * 6, np.int32))
    tb = truth_bins(truth_parameters(truth, w.bz_tesla), bn)
    rec = np.zeros(5, CAND_DTYPE)
    rec["i"] = [tb["i"][0], tb["i"][0] + 1, tb["i"][1], 100, tb["i"][2]]
    rec["j"] = [tb["j"][0], tb["j"][0], tb["j"][1], 5, tb["j"][2]]
    keep = np.array([1, 1, 1, 1, 0], np.uint8)
    h2c = np.array([0] * 6 + [1] * 4 + [2] * 9 + [3] + [4] * 4 + [3] * 5 + [-1], np.int32)
    r = efficiency_report(bn, w.bz_tesla, truth, rec, keep, h2c, min_hits=8)
    assert r["tracks"] == 3 and r["reconstructable"] == 2 and r["kept"] == 4
    # by hits: candidates 0 and 1 -> track 0 (one duplicate), 2 -> track 1, 3 -> noise (fake)
    assert r["by_hits"] == dict(efficiency=1.0, fake_rate=0.25, duplicate_rate=0.25, tracks_found=2)
    assert r["by_parameters"] == dict(efficiency=1.0, fake_rate=0.25, duplicate_rate=0.25, tracks_found=2)
