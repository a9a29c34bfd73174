"""Track-finding efficiency / fake / duplicate report against generator truth (Fig. 1 caption: "track-finding
efficiency ... approximately 86%").

Host-side evaluation of what the library returned (kept candidates, hit_to_cand) -- plain numpy on a few thousand
records, not part of the hot path.  Two matchings are reported, both standard:

* by hits:  a kept candidate is matched to the truth track that owns the MAJORITY of its assigned hits (purity > 1/2);
* by parameters:  a kept candidate is matched to a truth track whose true (phi0, q/pT, d0) bin lies within
  (dphi, dq, dk) bins of the candidate's bin.

efficiency = reconstructable truth tracks (>= min_hits hits) with at least one matched candidate / reconstructable tracks;
fake rate  = kept candidates matched to no track / kept candidates;
duplicate rate = matched candidates beyond the first of their track / kept candidates.
"""
from __future__ import annotations

import math
from typing import Dict

import numpy as np

K_GEV_PER_T_CM = 0.00299792458


def truth_parameters(truth: dict, bz_tesla: float) -> Dict[str, np.ndarray]:
    """(phi0, qpt, d0) of every generated track at its point of closest approach to the origin, in the convention of
    include/hough.h (D1): signed curvature rho = -(q/pT) K Bz (counter-clockwise positive), phi0 = direction of travel at
    the PCA, d0 = PCA . n_hat(phi0) with n_hat = (-sin phi0, cos phi0).  Straight tracks (Bz = 0): the line itself."""
    x0 = np.asarray(truth["start_x"], np.float64)
    y0 = np.asarray(truth["start_y"], np.float64)
    psi = np.asarray(truth["direction"], np.float64)
    qpt = np.asarray(truth["charge"], np.float64) / np.asarray(truth["pt"], np.float64)
    rho = -qpt * K_GEV_PER_T_CM * bz_tesla
    phi0 = np.mod(psi, 2 * math.pi)
    d0 = -x0 * np.sin(psi) + y0 * np.cos(psi)                       # straight line / prompt track
    curved = np.abs(rho) > 0
    if curved.any():
        r = 1.0 / rho[curved]                                       # signed radius: centre = start + r n_hat(psi)
        cx = x0[curved] - r * np.sin(psi[curved])
        cy = y0[curved] + r * np.cos(psi[curved])
        cn = np.hypot(cx, cy)
        s = np.sign(r)
        # direction of travel at the PCA (the point of the circle nearest the origin, on the ray origin -> centre)
        ok = cn > 1e-12
        tx = np.where(ok, s * cy / np.maximum(cn, 1e-300), np.cos(psi[curved]))
        ty = np.where(ok, -s * cx / np.maximum(cn, 1e-300), np.sin(psi[curved]))
        ph = np.mod(np.arctan2(ty, tx), 2 * math.pi)
        p0x = cx * (1.0 - np.abs(r) / np.maximum(cn, 1e-300))
        p0y = cy * (1.0 - np.abs(r) / np.maximum(cn, 1e-300))
        dd = -p0x * np.sin(ph) + p0y * np.cos(ph)
        phi0 = phi0.copy()
        d0 = d0.copy()
        phi0[curved] = np.where(ok, ph, phi0[curved])
        d0[curved] = np.where(ok, dd, 0.0)
    return dict(phi0=phi0, qpt=qpt, d0=d0)


def truth_bins(params: Dict[str, np.ndarray], binning) -> Dict[str, np.ndarray]:
    """Bin (i, j, k) of the true parameters (floor of the linear map; k = 0 for a one-slice space).  LINE-model
    spaces bin d0 along j."""
    n_phi, n_q, n_d = binning.n_phi, binning.n_qpt, binning.n_d0
    i = np.floor(params["phi0"] / (2 * math.pi) * n_phi).astype(np.int64) % n_phi
    along_j = params["d0"] if getattr(binning, "model", 0) == 1 else params["qpt"]
    j = np.floor((along_j - binning.qpt_min) / (binning.qpt_max - binning.qpt_min) * n_q).astype(np.int64)
    if n_d > 1:
        k = np.floor((params["d0"] - binning.d0_min) / (binning.d0_max - binning.d0_min) * n_d).astype(np.int64)
    else:
        k = np.zeros_like(i)
    return dict(i=i, j=j, k=k)


def efficiency_report(binning, bz_tesla, truth: dict, records: np.ndarray, keep: np.ndarray, hit_to_cand: np.ndarray,
                      min_hits: int, dphi: int = 1, dq: int = 2, dk: int = 1) -> dict:
    """One event.  records: candidate records of the event (fields i, j, k); keep, hit_to_cand: the library's outputs
    with candidate indices local to `records`."""
    keep = np.asarray(keep).astype(bool)
    n_c = len(records)
    track_of = np.asarray(truth["hit_track"], np.int64)
    n_t = len(truth["pt"])
    hits_per_track = np.bincount(track_of[track_of >= 0], minlength=n_t)
    reco = hits_per_track >= min_hits                                  # reconstructable tracks
    kept_idx = np.nonzero(keep)[0]
    # ---- by hits: majority owner of every kept candidate's hits
    h2c = np.asarray(hit_to_cand, np.int64)
    match_hits = np.full(n_c, -1, np.int64)
    purity = np.zeros(n_c)
    sel = h2c >= 0
    if sel.any():
        order = np.argsort(h2c[sel], kind="stable")
        cs, ts = h2c[sel][order], track_of[sel][order]
        starts = np.nonzero(np.r_[True, cs[1:] != cs[:-1]])[0]
        ends = np.r_[starts[1:], len(cs)]
        for a, b in zip(starts, ends):
            c = cs[a]
            t = ts[a:b]
            t = t[t >= 0]
            if len(t):
                ids, cnt = np.unique(t, return_counts=True)
                m = int(np.argmax(cnt))
                purity[c] = cnt[m] / float(b - a)
                if 2 * cnt[m] > (b - a):
                    match_hits[c] = ids[m]
    # ---- by parameters: nearest truth bin inside the window
    tb = truth_bins(truth_parameters(truth, bz_tesla), binning)
    match_par = np.full(n_c, -1, np.int64)
    if n_t:
        for c in kept_idx:
            di = np.abs(((records["i"][c] - tb["i"] + binning.n_phi // 2) % binning.n_phi) - binning.n_phi // 2)
            ok = (di <= dphi) & (np.abs(records["j"][c] - tb["j"]) <= dq) & (np.abs(records["k"][c] - tb["k"]) <= dk)
            if ok.any():
                cand_t = np.nonzero(ok)[0]
                match_par[c] = cand_t[np.argmin(di[cand_t] + np.abs(records["j"][c] - tb["j"][cand_t]))]

    def rates(match):
        m = match[kept_idx]
        found = np.zeros(n_t, bool)
        found[m[m >= 0]] = True
        n_matched = int((m >= 0).sum())
        n_dup = n_matched - int(len(np.unique(m[m >= 0])))
        nk = max(len(kept_idx), 1)
        return dict(efficiency=float(found[reco].sum() / max(int(reco.sum()), 1)),
                    fake_rate=float((len(kept_idx) - n_matched) / nk), duplicate_rate=float(n_dup / nk),
                    tracks_found=int(found[reco].sum()))

    return dict(tracks=int(n_t), reconstructable=int(reco.sum()), candidates=int(n_c), kept=int(len(kept_idx)),
                hits_assigned=int(sel.sum()), hits_total=int(len(h2c)),
                mean_purity=float(purity[kept_idx].mean()) if len(kept_idx) else 0.0,
                by_hits=rates(match_hits), by_parameters=rates(match_par),
                window_bins=dict(dphi=dphi, dq=dq, dk=dk))
