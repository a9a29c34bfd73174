"""Independent double-precision / brute-force restatements used only to pin the oracle."""
from __future__ import annotations

import math

import numpy as np

K = 0.00299792458


def geometric_bins(hits, n_phi, n_qpt, n_d0, qmin, qmax, d0min, d0max, bz, edge_tol=1e-4):
    """Votes from the tangent-chord construction, in double, with trigonometry.

    For a column (phi0, d0): PCA = d0 * n, chord D = p - PCA, alpha = angle from the direction of
    travel t to the chord; the circle tangent to t at the PCA through p has counter-clockwise
    curvature rho = 2 sin(alpha) / |D|; q/pT = -rho / (K Bz); forward iff |alpha| < pi/2.
    Returns a list of (h, k, i, j, safe) where safe says the value is > edge_tol bins from an edge.
    """
    out = []
    wq = (qmax - qmin) / n_qpt
    for h, (x, y) in enumerate(np.asarray(hits, np.float64)):
        for i in range(n_phi):
            th = (i + 0.5) * 2.0 * math.pi / n_phi
            t = (math.cos(th), math.sin(th))
            n = (-math.sin(th), math.cos(th))
            for k in range(n_d0):
                d0 = 0.0 if n_d0 == 1 else d0min + (k + 0.5) * (d0max - d0min) / n_d0
                dx, dy = x - d0 * n[0], y - d0 * n[1]
                along = dx * t[0] + dy * t[1]
                across = dx * n[0] + dy * n[1]
                alpha = math.atan2(across, along)
                fwd_margin = abs(abs(alpha) - math.pi / 2)
                if abs(alpha) >= math.pi / 2:
                    out.append((h, k, i, -1, fwd_margin > 1e-6))
                    continue
                rho = 2.0 * math.sin(alpha) / math.hypot(dx, dy)
                qpt = -rho / (K * bz)
                tt = (qpt - qmin) / wq
                safe = abs(tt - round(tt)) > edge_tol and fwd_margin > 1e-6
                j = int(math.floor(tt)) if 0.0 <= tt < n_qpt else -1
                out.append((h, k, i, j, safe))
    return out


def brute_peaks(acc, threshold):
    """Definition D5/D6 with python loops: acc int [n_d0, n_phi, n_qpt] -> sorted list of (k, i, j)."""
    nd, nphi, nq = acc.shape
    peaks = []
    for k in range(nd):
        for i in range(nphi):
            for j in range(nq):
                a = acc[k, i, j]
                if a < threshold:
                    continue
                ok = True
                for dk in (-1, 0, 1):
                    for di in (-1, 0, 1):
                        for dj in (-1, 0, 1):
                            if (dk, di, dj) == (0, 0, 0):
                                continue
                            kk, jj = k + dk, j + dj
                            if kk < 0 or kk >= nd or jj < 0 or jj >= nq:
                                continue
                            b = acc[kk, (i + di) % nphi, jj]
                            if (dk, di, dj) < (0, 0, 0):
                                ok = ok and a > b
                            else:
                                ok = ok and a >= b
                if ok:
                    peaks.append((k, i, j))
    return peaks
