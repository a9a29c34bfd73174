"""Seeded synthetic event generator (detector + track simulation only).

Recipe (stated again in DESIGN.md, "Input recipe"); G-numbers refer to SURVEY.md section 8(d):

* RNG (G1, our variant): one counter-based ``numpy.random.Philox`` stream per (workload seed, event
  index), consumed as RAW 64-bit words only; uniform ``u = (x >> 11) * 2**-53``; normal by
  Box-Muller; exponential ``-s*ln(1-u)``.  No ``Generator`` distribution method is used, so the
  stream is fixed by the Philox algorithm alone.  Because each event has its own key, event ``e``
  of a workload is the same no matter how many events are generated or which rank generates it.
* Geometry (G2): cylindrical barrel layers at the workload's radii, solenoid field Bz along +z.
* Track model ("only the transverse plane"): a circle of signed
  counter-clockwise curvature ``rho = -(q/pT) * K * Bz`` with ``K = 0.00299792458 GeV/(T cm)``
  (positive charge turns clockwise for Bz > 0).
* Prompt tracks (G3): start at the origin, direction uniform, charge +-1 (p = 0.5).
* Displaced tracks (G4): ceil(n/4) vertices at transverse radius U[1,20] cm, azimuth uniform; tracks
  dealt round-robin; direction at the vertex = vertex azimuth + U(-0.5, 0.5) rad.
* Hits (G5): one per layer with radius > production radius at the FIRST forward crossing of the
  circle with the layer; layers the circle never reaches are skipped; r-phi smear = rotation about
  the origin by N(0, sigma)/r_layer.
* Noise (G6): exactly on a uniformly chosen layer, azimuth uniform.
* Order (G7): hits of an event are shuffled (argsort of raw 64-bit keys).
* Units (G8): cm, GeV, rad; all arithmetic in float64, hits rounded to float32 (x, y) last.

Nothing here knows about accumulators, bins, votes, peaks or assignments.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import List, Optional, Sequence

import numpy as np

from .configs import HoughWorkload

K_GEV_PER_T_CM = 0.00299792458          # pT[GeV] = K * Bz[T] * R[cm]
_TWO_PI = 2.0 * np.pi


class _RawStream:
    """Sequential consumer of one Philox stream, raw words only."""

    def __init__(self, seed: int, event: int):
        self._bg = np.random.Philox(key=np.array([np.uint64(seed), np.uint64(event)], dtype=np.uint64))

    def raw(self, n: int) -> np.ndarray:
        return self._bg.random_raw(int(n)).astype(np.uint64, copy=False) if n > 0 else np.zeros(0, np.uint64)

    def uniform(self, n: int) -> np.ndarray:
        return (self.raw(n) >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)

    def normal(self, n: int) -> np.ndarray:
        u1 = self.uniform(n)
        u2 = self.uniform(n)
        return np.sqrt(-2.0 * np.log1p(-u1)) * np.cos(_TWO_PI * u2)

    def exponential(self, n: int, scale: float) -> np.ndarray:
        return -scale * np.log1p(-self.uniform(n))


def _propagate_to_layers(px, py, psi, rho, radii):
    """First forward crossing of circles with the barrel layers.

    A track starts at (px, py) with direction angle psi and signed counter-clockwise curvature rho.
    Its circle has centre c = p + n/rho with n = (-sin psi, cos psi).  Writing the position after a
    signed turning angle u (= rho * arc length) as c + R(u) a with a = p - c, the crossing with the
    layer |x| = r satisfies  cos(u + beta) = (r^2 - |c|^2 - |a|^2) / (2 |c| |a|),  beta = arg a - arg c.
    The first crossing is the solution with u/rho > 0 of smallest |u|.

    px, py, psi, rho: arrays [T];  radii: array [L].
    Returns x, y arrays [T, L] and a validity mask [T, L] (layer outside the start point, reached).
    """
    px = np.asarray(px, np.float64)[:, None]
    py = np.asarray(py, np.float64)[:, None]
    psi = np.asarray(psi, np.float64)[:, None]
    rho = np.asarray(rho, np.float64)[:, None]
    r = np.asarray(radii, np.float64)[None, :]

    inv_rho = 1.0 / rho
    cx = px - np.sin(psi) * inv_rho
    cy = py + np.cos(psi) * inv_rho
    ax = px - cx
    ay = py - cy
    cc = np.hypot(cx, cy)
    aa = np.hypot(ax, ay)
    with np.errstate(invalid="ignore", divide="ignore"):
        cosarg = (r * r - cc * cc - aa * aa) / (2.0 * cc * aa)
    reach = np.abs(cosarg) <= 1.0
    ac = np.arccos(np.clip(cosarg, -1.0, 1.0))
    beta = np.arctan2(ay, ax) - np.arctan2(cy, cx)
    sgn = np.sign(rho)
    # two solution families; bring sgn*u into (0, 2pi)
    u1 = np.mod(sgn * (ac - beta), _TWO_PI)
    u2 = np.mod(sgn * (-ac - beta), _TWO_PI)
    tiny = 1e-12
    u1 = np.where(u1 < tiny, u1 + _TWO_PI, u1)
    u2 = np.where(u2 < tiny, u2 + _TWO_PI, u2)
    u = sgn * np.minimum(u1, u2)
    cu, su = np.cos(u), np.sin(u)
    x = cx + cu * ax - su * ay
    y = cy + su * ax + cu * ay
    outside = r > np.hypot(px, py)
    return x, y, reach & outside


def _propagate_lines(px, py, psi, radii):
    """Forward crossing of straight lines p + s (cos psi, sin psi), s > 0, with the barrel layers (zero field).

    |p + s t|^2 = r^2  =>  s = -(p.t) + sqrt((p.t)^2 - |p|^2 + r^2); a layer inside the start radius is not crossed going
    forward unless the root is real and positive.  Returns x, y [T, L] and the validity mask."""
    px = np.asarray(px, np.float64)[:, None]
    py = np.asarray(py, np.float64)[:, None]
    psi = np.asarray(psi, np.float64)[:, None]
    r = np.asarray(radii, np.float64)[None, :]
    tx, ty = np.cos(psi), np.sin(psi)
    pt_ = px * tx + py * ty
    disc = pt_ * pt_ - (px * px + py * py) + r * r
    ok = (disc > 0.0) & (r * r > px * px + py * py)
    sq = np.sqrt(np.where(disc > 0.0, disc, 0.0))
    sfwd = -pt_ + sq
    ok = ok & (sfwd > 0.0)
    return px + sfwd * tx, py + sfwd * ty, ok


def line_hits(phi0: float, d0: float, radii: Sequence[float]) -> np.ndarray:
    """Noiseless hits (float32 [n,2]) of ONE straight track: direction phi0, signed impact parameter d0 (SURVEY D1
    convention: closest point = d0 * (-sin phi0, cos phi0)), followed forward from its closest point."""
    x, y, ok = _propagate_lines([-d0 * np.sin(phi0)], [d0 * np.cos(phi0)], [phi0], radii)
    return np.stack([x[0][ok[0]], y[0][ok[0]]], axis=1).astype(np.float32)


def helix_hits(phi0: float, qpt: float, d0: float, radii: Sequence[float], bz_tesla: float) -> np.ndarray:
    """Noiseless hits (float32 [n,2]) of ONE track given at its point of closest approach.

    (phi0, q/pT, d0) in the SURVEY D1 convention: PCA = d0 * (-sin phi0, cos phi0), direction phi0.
    Used by the oracle pins (a helix generated here must peak in its own parameter bin).
    """
    rho = -qpt * K_GEV_PER_T_CM * bz_tesla
    px = -d0 * np.sin(phi0)
    py = d0 * np.cos(phi0)
    x, y, ok = _propagate_to_layers([px], [py], [phi0], [rho], radii)
    return np.stack([x[0][ok[0]], y[0][ok[0]]], axis=1).astype(np.float32)


@dataclass
class EventBatch:
    hits_xy: np.ndarray          # float32 [H, 2], events concatenated
    event_offsets: np.ndarray    # int32 [n_events + 1]
    truth: Optional[List[dict]]  # per event: arrays describing the generated tracks (float64)

    @property
    def n_hits(self) -> int:
        return int(self.hits_xy.shape[0])

    @property
    def n_events(self) -> int:
        return int(self.event_offsets.shape[0] - 1)

    def event(self, e: int) -> np.ndarray:
        return self.hits_xy[self.event_offsets[e]:self.event_offsets[e + 1]]

    def select(self, events: Sequence[int]) -> "EventBatch":
        parts = [self.event(e) for e in events]
        off = np.zeros(len(parts) + 1, np.int32)
        off[1:] = np.cumsum([p.shape[0] for p in parts])
        hits = np.concatenate(parts, axis=0) if parts else np.zeros((0, 2), np.float32)
        truth = [self.truth[e] for e in events] if self.truth is not None else None
        return EventBatch(np.ascontiguousarray(hits), off, truth)


def generate_event(w: HoughWorkload, event: int, want_truth: bool = False):
    """Hits of event `event` of workload `w`: float32 [n, 2] (and the truth dict if asked)."""
    s = _RawStream(w.seed, event)
    radii = np.asarray(w.layers, np.float64)
    n_layers = radii.shape[0]
    kb = K_GEV_PER_T_CM * w.bz_tesla

    def draw_pt(n):
        if w.pt_law == "uniform":
            return w.pt_min + (w.pt_max - w.pt_min) * s.uniform(n)
        return w.pt_min + s.exponential(n, w.pt_exp_scale)

    # prompt tracks (G3)
    n_p = w.n_prompt
    p_dir = _TWO_PI * s.uniform(n_p)
    p_q = np.where(s.uniform(n_p) < 0.5, -1.0, 1.0)
    p_pt = draw_pt(n_p)
    # displaced tracks (G4)
    n_d = w.n_displaced
    n_v = w.n_vertices if w.n_vertices > 0 else (n_d + 3) // 4
    v_r = w.vertex_r_min + (w.vertex_r_max - w.vertex_r_min) * s.uniform(n_v)
    v_az = _TWO_PI * s.uniform(n_v)
    d_vtx = np.arange(n_d) % max(n_v, 1)
    d_dir = (v_az[d_vtx] if n_d else np.zeros(0)) + (s.uniform(n_d) - 0.5)
    d_q = np.where(s.uniform(n_d) < 0.5, -1.0, 1.0)
    d_pt = draw_pt(n_d)

    px = np.concatenate([np.zeros(n_p), (v_r[d_vtx] * np.cos(v_az[d_vtx])) if n_d else np.zeros(0)])
    py = np.concatenate([np.zeros(n_p), (v_r[d_vtx] * np.sin(v_az[d_vtx])) if n_d else np.zeros(0)])
    psi = np.concatenate([p_dir, d_dir])
    q = np.concatenate([p_q, d_q])
    pt = np.concatenate([p_pt, d_pt])
    rho = -(q / pt) * kb

    n_t = n_p + n_d
    if w.bz_tesla == 0.0:                                 # zero field: straight tracks
        x, y, ok = _propagate_lines(px, py, psi, radii)
    else:
        x, y, ok = _propagate_to_layers(px, py, psi, rho, radii)
    # r-phi smear (G5): rotate about the origin by N(0, sigma) / r_layer
    delta = (s.normal(n_t * n_layers).reshape(n_t, n_layers) * w.sigma_rphi_cm) / radii[None, :]
    cd, sd = np.cos(delta), np.sin(delta)
    xs = cd * x - sd * y
    ys = sd * x + cd * y
    tx = xs[ok]
    ty = ys[ok]
    n_track_hits = tx.shape[0]

    # noise (G6)
    n_noise = w.n_noise if w.n_noise >= 0 else int(round(0.05 * n_track_hits))
    lay = np.minimum((s.uniform(n_noise) * n_layers).astype(np.int64), n_layers - 1)
    nphi = _TWO_PI * s.uniform(n_noise)
    nx = radii[lay] * np.cos(nphi)
    ny = radii[lay] * np.sin(nphi)

    hx = np.concatenate([tx, nx])
    hy = np.concatenate([ty, ny])
    # shuffle (G7)
    order = np.argsort(s.raw(hx.shape[0]), kind="stable")
    hits = np.stack([hx[order], hy[order]], axis=1).astype(np.float32)
    if not want_truth:
        return hits, None
    # generating track of every hit (after the shuffle), -1 = noise: for the efficiency / fake-rate report
    track_of = np.concatenate([np.broadcast_to(np.arange(n_t)[:, None], ok.shape)[ok], np.full(n_noise, -1)])[order]
    truth = dict(start_x=px, start_y=py, direction=psi, charge=q, pt=pt, rho=rho,
                 n_track_hits=n_track_hits, n_noise=n_noise, layer_hit_mask=ok, hit_track=track_of.astype(np.int32))
    return hits, truth


def generate_events(w: HoughWorkload, events: Optional[Sequence[int]] = None,
                    want_truth: bool = False) -> EventBatch:
    """Generate the listed events (default: all `w.n_events`) and pack them with int32 offsets."""
    if events is None:
        events = range(w.n_events)
    parts, truths = [], []
    for e in events:
        h, t = generate_event(w, int(e), want_truth)
        parts.append(h)
        truths.append(t)
    off = np.zeros(len(parts) + 1, np.int64)
    if parts:
        off[1:] = np.cumsum([p.shape[0] for p in parts])
    assert off[-1] < 2 ** 31
    hits = np.concatenate(parts, axis=0) if parts else np.zeros((0, 2), np.float32)
    return EventBatch(np.ascontiguousarray(hits, dtype=np.float32), off.astype(np.int32),
                      truths if want_truth else None)
