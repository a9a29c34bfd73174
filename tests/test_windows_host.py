"""Host logic of the CUDA library (no GPU): the radius-class / column-window tables of hough_window_table.

The tables only size work (include/hough.h, S19): the kernels evaluate the exact D3 sequence at every column
of a window.  What must hold is that a window NEVER misses a column the oracle votes in; how tight it is
decides only the speed.  Both are checked here against the oracle's own vote (full scan).
"""
import numpy as np
import pytest

from oracle import Oracle
from paper_1311_2769_b200 import window_table
from workloads import LAYERS_10, LAYERS_14, generate_events, get_workload

BZ = 3.8


def _valid_columns(o: Oracle, hits):
    """valid[h, k, i] = the oracle casts a vote for hit h in column (k, i) (one event per hit)."""
    n = hits.shape[0]
    off = np.arange(n + 1, dtype=np.int32)
    acc, _ = o.vote(hits, off)
    return acc.sum(axis=3) > 0


def _covered_columns(hits, n_phi, edge, lo, steps):
    """What the device does with the table, restated: class from r^2, u from atan2, run of `steps` columns."""
    x = hits[:, 0].astype(np.float32)
    y = hits[:, 1].astype(np.float32)
    r2 = (x * x).astype(np.float32) + (y * y).astype(np.float32)
    cls = np.searchsorted(edge, r2, side="right") - 1
    cls = np.where(np.isnan(r2), len(edge) - 1, np.clip(cls, 0, len(edge) - 1))
    phi = np.arctan2(y, x).astype(np.float32)
    phi = np.where(phi < 0, phi + np.float32(2 * np.pi), phi).astype(np.float32)
    u = (phi * np.float32(n_phi / (2 * np.pi)) - np.float32(0.5)).astype(np.float32)
    n_d0 = lo.shape[1]
    cov = np.zeros((hits.shape[0], n_d0, n_phi), bool)
    for h in range(hits.shape[0]):
        for k in range(n_d0):
            i_lo = int(np.ceil(np.float32(u[h] + lo[cls[h], k])))
            idx = (i_lo + np.arange(steps[cls[h], k])) % n_phi
            cov[h, k, idx] = True
    return cov, cls


def _random_hits(rng, n, layers, r_max=140.0):
    """Half exactly on layers (as the generator places them), half at arbitrary radii incl. tiny and far."""
    n_l = n // 2
    r = np.concatenate([rng.choice(np.asarray(layers), n_l), rng.uniform(0.0, r_max, n - n_l - 4), [1e-3, 0.3, 19.99, 400.0]])
    ph = rng.uniform(0, 2 * np.pi, r.shape[0])
    return np.stack([r * np.cos(ph), r * np.sin(ph)], 1).astype(np.float32)


@pytest.mark.parametrize("shape,layers,qr,dr", [
    ((64, 32, 8), LAYERS_10, (-1.0, 1.0), (-20.0, 20.0)),
    ((128, 64, 1), LAYERS_14, (-1.0, 1.0), (-20.0, 20.0)),
    ((64, 48, 5), (), (-0.5, 2.0), (-30.0, 10.0)),         # no geometry, asymmetric ranges
    ((32, 16, 4), LAYERS_10, (0.1, 0.9), (5.0, 60.0)),     # q range excluding 0, d0 larger than inner layers
    ((256, 128, 3), LAYERS_14, (-3.0, 3.0), (-1.0, 1.0)),  # A r q > 1 on the outer layers: half-circle windows
])
def test_windows_never_miss_a_vote(shape, layers, qr, dr):
    n_phi, n_qpt, n_d0 = shape
    rng = np.random.default_rng(n_phi + n_d0)
    hits = _random_hits(rng, 260, layers or LAYERS_10)
    o = Oracle(n_phi, n_qpt, n_d0, qr[0], qr[1], dr[0], dr[1], bz_tesla=BZ)
    valid = _valid_columns(o, hits)
    edge, lo, steps = window_table(n_phi, n_qpt, n_d0, qr[0], qr[1], dr[0], dr[1], BZ, layers)
    assert edge[0] == 0 and np.all(np.diff(edge) > 0) and len(edge) <= 255
    cov, _ = _covered_columns(hits, n_phi, edge, lo, steps)
    assert not (valid & ~cov).any(), "a window misses a voting column"
    assert steps.max() <= n_phi and steps.min() >= 0


@pytest.mark.parametrize("cfg", [1, 3])
def test_windows_are_tight_on_the_baseline_workloads(cfg):
    """On hits placed on the detector layers the windows waste little: votes / visited columns."""
    w = get_workload(cfg)
    bn = w.binning
    hits = generate_events(w, events=[0]).hits_xy[:160]
    o = Oracle.from_binning(bn, w.bz_tesla)
    valid = _valid_columns(o, hits)
    edge, lo, steps = window_table(bn.n_phi, bn.n_qpt, bn.n_d0, bn.qpt_min, bn.qpt_max, bn.d0_min, bn.d0_max,
                                   w.bz_tesla, w.layers)
    cov, cls = _covered_columns(hits, bn.n_phi, edge, lo, steps)
    assert not (valid & ~cov).any()
    eff = valid.sum() / cov.sum()
    assert eff > 0.80, eff


def test_windows_negative_field_and_zero_field_fall_back_to_the_forward_half():
    for bz in (-3.8, 0.0):
        edge, lo, steps = window_table(64, 32, 4, bz_tesla=bz, layers=LAYERS_10)
        assert (steps == 64 // 2 + 5).all()
    rng = np.random.default_rng(5)
    hits = _random_hits(rng, 60, LAYERS_10)
    o = Oracle(64, 32, 4, bz_tesla=-3.8)
    valid = _valid_columns(o, hits)
    edge, lo, steps = window_table(64, 32, 4, bz_tesla=-3.8, layers=LAYERS_10)
    cov, _ = _covered_columns(hits, 64, edge, lo, steps)
    assert valid.any() and not (valid & ~cov).any()


@pytest.mark.parametrize("shape,layers,dr", [
    ((64, 32), LAYERS_10, (-20.0, 20.0)),
    ((256, 64), LAYERS_14, (-30.0, 5.0)),                  # asymmetric d0 range
    ((128, 16), (), (2.0, 40.0)),                          # no geometry; range excluding 0 and wider than inner radii
])
def test_line_model_windows_never_miss_a_vote(shape, layers, dr):
    """HOUGH_MODEL_LINE (D3L): the windows of the straight-track space (phi0, d0) contain every voting column."""
    n_phi, n_d = shape
    rng = np.random.default_rng(n_phi + n_d)
    hits = _random_hits(rng, 260, layers or LAYERS_10)
    o = Oracle(n_phi, n_d, 1, dr[0], dr[1], bz_tesla=0.0, model=1)
    valid = _valid_columns(o, hits)
    edge, lo, steps = window_table(n_phi, n_d, 1, dr[0], dr[1], bz_tesla=0.0, layers=layers, model=1)
    cov, _ = _covered_columns(hits, n_phi, edge, lo, steps)
    assert valid.any() and not (valid & ~cov).any(), "a window misses a voting column"
    on_layer = np.isin(np.round(np.hypot(hits[:, 0], hits[:, 1]), 3), np.round(np.asarray(layers or LAYERS_10), 3))
    if layers:
        assert cov[on_layer].sum() < 3.0 * valid[on_layer].sum() + 4 * on_layer.sum()      # and they are not wasteful
