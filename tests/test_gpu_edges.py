"""-m gpu: adversarial inputs for the vote walk's fast path (an error-bounded approximate
evaluation decides a bin only when it is further than the bound m from a bin edge; everything else is redone with the
exact D3 sequence).  The bound is a first-order analysis validated empirically, so it is attacked here on purpose:

hits are CONSTRUCTED (in double, from the D1 geometry, not from the kernel's or the oracle's code) so that for a chosen
(layer radius, phi0 column i, d0 slice k) the D3 value t lands at a chosen distance from a chosen bin edge E -- from a few
fp32 ulps (the rounding of the hit coordinates supplies the last-digit scatter) through 1e-4 ... 0.4 bins, i.e. on both
sides of every class's decision limit 1/2 - m, the innermost layers (largest m) included.  Columns are sampled over all
residues, so the targeted column falls on every position of the walk's 32-pair recurrence chunks, the last pair included.
The whole accumulator of the default path must equal the oracle's (PAPER.md:37 vote step; reading D3)."""
import math

import numpy as np
import pytest

from oracle import Oracle
from workloads import get_workload
from workloads.generator import K_GEV_PER_T_CM

pytestmark = pytest.mark.gpu

from gpu_util import oracle_vote_parallel, run_vote  # noqa: E402

OFFSETS = [0.0] + [s * d for d in (1e-5, 1e-4, 1e-3, 1e-2, 0.05, 0.1, 0.2, 0.4) for s in (-1.0, 1.0)]


def _edge_hits(w, n_cols, n_slices, n_edges, seed):
    """Hits whose t at (i, k) is E + offset in exact arithmetic; returns fp32 hits and how close they really come."""
    bn = w.binning
    rng = np.random.default_rng(seed)
    A = 0.5 * K_GEV_PER_T_CM * float(np.float32(w.bz_tesla))
    wq = (bn.qpt_max - bn.qpt_min) / bn.n_qpt
    cols = rng.choice(bn.n_phi, n_cols, replace=False)
    ks = rng.choice(bn.n_d0, min(n_slices, bn.n_d0), replace=False)
    hits, dist = [], []
    for r in w.layers:
        for i in cols:
            th = (i + 0.5) * 2.0 * math.pi / bn.n_phi
            for k in ks:
                d0 = 0.0 if bn.n_d0 == 1 else bn.d0_min + (k + 0.5) * (bn.d0_max - bn.d0_min) / bn.n_d0
                for E in rng.integers(1, bn.n_qpt, n_edges):
                    for off in OFFSETS:
                        v = bn.qpt_min + (E + off) * wq                    # q/pT the hit must solve to in column (i, k)
                        den = 1.0 - 2.0 * v * A * d0
                        if abs(den) < 1e-6:
                            continue
                        wv = (d0 - v * A * (r * r + d0 * d0)) / den        # w = r sin(phi_hit - theta_i)  (D3 solved for w)
                        if abs(wv) > 0.9 * r:
                            continue
                        ph = th + math.asin(wv / r)                        # forward side: cos(phi_hit - theta_i) > 0
                        x, y = np.float32(r * math.cos(ph)), np.float32(r * math.sin(ph))
                        # what the rounded hit gives, in double: distance of t from the edge
                        xd, yd = float(x), float(y)
                        wd = yd * math.cos(th) - xd * math.sin(th)
                        td = ((d0 - wd) / (A * (xd * xd + yd * yd - 2.0 * d0 * wd + d0 * d0)) - bn.qpt_min) / wq
                        hits.append((x, y))
                        dist.append(abs(td - E))
    return np.asarray(hits, np.float32), np.asarray(dist)


def _split(n_hits, per_event):
    off = list(range(0, n_hits, per_event)) + [n_hits]
    return np.asarray(off, np.int32)


@pytest.mark.parametrize("cfg,n_cols,n_slices,n_edges,per_event", [(3, 24, 6, 5, 8192), (4, 12, 4, 4, 1 << 30), (0, 32, 1, 8, 1 << 30)])
def test_hits_constructed_on_bin_edges_vote_like_the_oracle(cfg, n_cols, n_slices, n_edges, per_event):
    w = get_workload(cfg)
    bn = w.binning
    hits, dist = _edge_hits(w, n_cols, n_slices, n_edges, seed=100 + cfg)
    assert len(hits) > 20000
    # the construction works: hits within ~4 fp32 ulps of t of an edge exist (t ~ n_qpt / 2 -> ulp ~ n_qpt * 6e-8), and the
    # wider offsets are populated as well
    ulp_t = bn.n_qpt * 6.0e-8
    assert (dist < 4 * ulp_t).sum() >= 100 and ((dist > 0.04) & (dist < 0.45)).sum() >= 1000
    rng = np.random.default_rng(cfg)
    hits = hits[rng.permutation(len(hits))]
    off = _split(len(hits), per_event)
    got = run_vote(bn, w.bz_tesla, w.layers, hits, off)
    o = Oracle.from_binning(bn, w.bz_tesla)
    if len(off) == 2:
        acc, votes = oracle_vote_parallel(o, hits, off)
    else:
        from concurrent.futures import ThreadPoolExecutor
        from gpu_util import n_threads
        with ThreadPoolExecutor(n_threads()) as ex:
            parts = list(ex.map(lambda e: o.vote(hits[off[e]:off[e + 1]])[0], range(len(off) - 1)))
        acc = np.concatenate(parts, axis=0)
    assert acc.max() <= (65535 if bn.bin_bytes == 2 else 2 ** 31 - 1)
    assert np.array_equal(got.astype(np.int64), acc.astype(np.int64)), "accumulator differs on edge-targeted hits"
