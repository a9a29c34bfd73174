"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA path).

V-numbers follow SURVEY.md section 8(c) "What pins the oracle".  Each pin is chosen so that a
plausible mistake in oracle/hough_oracle.cpp (dropped term, wrong sign, transposed operand, wrong
index order, off-by-one in a neighbourhood) fails at least one of them.
"""
import math
import os

import numpy as np
import pytest

from oracle import Oracle
from workloads import (LAYERS_10, LAYERS_14, generate_events, get_workload, helix_hits)

from helpers import K, brute_peaks, geometric_bins

BZ = 3.8


# ----------------------------------------------------------------------------- golden (textbook)
def _golden_cases(golden_dir):
    rows = []
    with open(os.path.join(golden_dir, "circle_chord_cases.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            n_phi, i, R, a_deg, q, exp = line.split()
            rows.append((int(n_phi), int(i), float(R), float(a_deg), int(q), float(exp)))
    return rows


def test_golden_tangent_chord(golden_dir):
    """tests/golden/circle_chord_cases.txt: pT = 0.3 B R and the tangent-chord theorem."""
    n_qpt = 256
    for n_phi, i, R, a_deg, q, exp in _golden_cases(golden_dir):
        theta = (i + 0.5) * 2.0 * math.pi / n_phi
        a = math.radians(a_deg)
        r = 2.0 * R * math.sin(a)
        ang = theta - q * a
        hit = np.array([[r * math.cos(ang), r * math.sin(ang)]], np.float32)
        o = Oracle(n_phi, n_qpt, 1, -1.0, 1.0, bz_tesla=BZ)
        rows = o.vote_columns(hit, None, [[0, 0, i]])[0]
        if -1.0 <= exp < 1.0:
            j = int(math.floor((exp + 1.0) / (2.0 / n_qpt)))
            assert rows.sum() == 1 and rows[j] == 1, (n_phi, i, R, a_deg, q, exp, np.nonzero(rows))
        else:
            assert rows.sum() == 0
        # mirror column (phi0 + pi) is the backward branch and must not be voted (S4)
        assert o.vote_columns(hit, None, [[0, 0, (i + n_phi // 2) % n_phi]]).sum() == 0


def test_plan_constants():
    """D2: A = K Bz / 2 = 0.005696056702 for 3.8 T, exact table symmetry, exact d0 tables."""
    o = Oracle(256, 128, 64, bz_tesla=BZ)
    t = o.tables()
    # bz enters as fp32 (3.8f = 3.7999999523...), so A_f is the fp32 nearest 0.5*K*(double)3.8f: one ulp
    # below fp32(0.005696056702); R(1 GeV) = 1/(2A) = 87.78 cm
    assert t["A_f"] == np.float32(0.5 * K * float(np.float32(3.8)))
    assert abs(float(t["A_f"]) - 0.005696056702) < 6e-10 and abs(1.0 / (2.0 * float(t["A_f"])) - 87.78) < 0.01
    assert t["inv_wq"] == np.float32(64.0) and t["qmin"] == np.float32(-1.0)
    n = 256
    th = (np.arange(n) + 0.5) * 2 * np.pi / n
    assert np.abs(t["cosT"] - np.cos(th)).max() < 1e-7 and np.abs(t["sinT"] - np.sin(th)).max() < 1e-7
    q = n // 4
    assert np.array_equal(t["cosT"][q:], -t["sinT"][:-q]) and np.array_equal(t["sinT"][q:], t["cosT"][:-q])
    d0 = -20.0 + (np.arange(64) + 0.5) * 40.0 / 64
    assert np.array_equal(t["d0c"].astype(np.float64), d0)           # exactly representable
    assert np.array_equal(t["td0"].astype(np.float64), 2 * d0)
    assert np.array_equal(t["d0sq"].astype(np.float64), d0 * d0)
    t2 = Oracle(64, 32, 1, bz_tesla=BZ).tables()
    assert t2["d0c"][0] == 0 and t2["td0"][0] == 0 and t2["d0sq"][0] == 0


# ----------------------------------------------------------------------------- V1
@pytest.mark.parametrize("seed", [0, 1, 2, 3])
@pytest.mark.parametrize("shape", [(8, 8, 1), (8, 8, 4), (16, 12, 3)])
def test_v1_bruteforce_double_geometry(seed, shape):
    n_phi, n_qpt, n_d0 = shape
    rng = np.random.default_rng(100 + seed)
    r = rng.uniform(4.0, 110.0, 8)
    ph = rng.uniform(0, 2 * np.pi, 8)
    hits = np.stack([r * np.cos(ph), r * np.sin(ph)], 1).astype(np.float32)
    qr = (1.0, 3.0)[seed % 2]          # the wider range makes inner-layer hits vote in many columns
    o = Oracle(n_phi, n_qpt, n_d0, -qr, qr, -20.0, 20.0, BZ)
    n_checked = 0
    for h in range(hits.shape[0]):
        acc, _ = o.vote(hits[h:h + 1])
        for (_, k, i, j, safe) in geometric_bins(hits[h:h + 1], n_phi, n_qpt, n_d0, -qr, qr, -20.0, 20.0, BZ):
            if not safe:
                continue
            col = acc[0, k, i]
            if j < 0:
                assert col.sum() == 0, (h, k, i)
            else:
                assert col.sum() == 1 and col[j] == 1, (h, k, i, j, np.nonzero(col))
            n_checked += 1
    assert n_checked > 0.9 * hits.shape[0] * n_phi * n_d0


# ----------------------------------------------------------------------------- V2
@pytest.mark.parametrize("shape,ijk", [((256, 256, 1), (37, 200, 0)), ((256, 128, 64), (201, 30, 40)),
                                       ((256, 128, 64), (5, 100, 12)), ((1024, 512, 128), (700, 260, 64))])
def test_v2_noiseless_helix_peaks_in_its_own_bin(shape, ijk):
    n_phi, n_qpt, n_d0 = shape
    i, j, k = ijk
    phi0 = (i + 0.5) * 2 * math.pi / n_phi
    qpt = -1.0 + (j + 0.5) * 2.0 / n_qpt
    d0 = 0.0 if n_d0 == 1 else -20.0 + (k + 0.5) * 40.0 / n_d0
    hits = helix_hits(phi0, qpt, d0, LAYERS_10, BZ)
    n = hits.shape[0]
    assert n >= 7            # layers inside |d0| are never crossed
    o = Oracle(n_phi, n_qpt, n_d0, bz_tesla=BZ)
    k_lo, k_hi = max(0, k - 2), min(n_d0, k + 3)
    acc, _ = o.vote(hits, k_range=(k_lo, k_hi))
    assert acc[0, k - k_lo, i, j] == n                       # every hit votes for the true bin
    assert (acc == n).sum() == 1 and acc.max() == n          # and it is the unique maximum
    ko = (max(k_lo, k - 1) if k_lo > 0 else 0, min(k_hi, k + 2) if k_hi < n_d0 else n_d0)
    c = o.find_peaks(acc, n, k_range=(k_lo, k_hi), k_out=ko)
    assert c.total == 1
    rec = c.records[0]
    assert (rec["k"], rec["i"], rec["j"], rec["votes"]) == (k, i, j, n)
    assert abs(rec["qpt"] - qpt) <= 0.5 * 2.0 / n_qpt
    assert abs(rec["phi0"] - phi0) <= 0.5 * 2 * math.pi / n_phi
    if n_d0 > 1:
        assert abs(rec["d0"] - d0) <= 0.5 * 40.0 / n_d0
    if n_d0 <= 64 and n_phi <= 256:
        full, _ = o.vote(hits)
        cf = o.find_peaks(full, n)
        assert cf.total == 1 and cf.records[0] == rec
        h2c, nh, keep = o.assign_brute(hits, None, cf, 1, n)
        assert (h2c == 0).all() and nh[0] == n and keep[0] == 1


# ----------------------------------------------------------------------------- V3
def test_v3_closed_form_vote_count():
    w = get_workload(0)
    b = generate_events(w)
    o = Oracle.from_binning(w.binning, w.bz_tesla)
    acc, votes = o.vote(b.hits_xy, b.event_offsets)
    vph = o.votes_per_hit(b.hits_xy)
    assert votes == int(acc.sum()) == int(vph.sum())
    A = 0.5 * K * w.bz_tesla
    r = np.hypot(b.hits_xy[:, 0].astype(np.float64), b.hits_xy[:, 1].astype(np.float64))
    arg = np.minimum(A * r * 1.0, 1.0)
    expect = w.binning.n_phi * np.arcsin(arg) / np.pi
    assert np.abs(vph - expect).max() <= 1.0
    # every in-range column of a hit gets exactly one vote, never two
    one, _ = o.vote(b.hits_xy[:1])
    assert one.sum(axis=-1).max() == 1


def test_v3_3d_count_matches_counter_and_geometry():
    rng = np.random.default_rng(7)
    r = np.array(LAYERS_10)[rng.integers(0, 10, 24)]
    ph = rng.uniform(0, 2 * np.pi, 24)
    hits = np.stack([r * np.cos(ph), r * np.sin(ph)], 1).astype(np.float32)
    o = Oracle(32, 16, 8, bz_tesla=BZ)
    acc, votes = o.vote(hits)
    assert votes == acc.sum() == o.votes_per_hit(hits).sum()
    g = geometric_bins(hits, 32, 16, 8, -1.0, 1.0, -20.0, 20.0, BZ)
    n_geo = sum(1 for (_, _, _, j, _) in g if j >= 0)
    n_unsafe = sum(1 for (_, _, _, _, s) in g if not s)
    assert abs(n_geo - votes) <= n_unsafe


# ----------------------------------------------------------------------------- V4
def test_v4_linearity_permutation_batching():
    w = get_workload(1)
    b = generate_events(w)
    o = Oracle(64, 32, 8, bz_tesla=BZ)
    hits = b.hits_xy[:400]
    acc, _ = o.vote(hits)
    a1, _ = o.vote(hits[:150])
    a2, _ = o.vote(hits[150:])
    assert np.array_equal(acc, a1 + a2)
    perm = np.random.default_rng(3).permutation(hits.shape[0])
    ap, _ = o.vote(hits[perm])
    assert np.array_equal(acc, ap)
    off = np.array([0, 150, 150, 400], np.int32)          # includes an empty event
    ab, _ = o.vote(hits, off)
    assert np.array_equal(ab[0], a1[0]) and np.array_equal(ab[2], a2[0]) and ab[1].sum() == 0
    # k-range restriction is a pure slice
    ak, _ = o.vote(hits, k_range=(2, 5))
    assert np.array_equal(ak[0], acc[0, 2:5])
    cols = [[0, 3, 17], [0, 0, 63], [0, 7, 0]]
    rows = o.vote_columns(hits, None, cols)
    for s, (_, k, i) in enumerate(cols):
        assert np.array_equal(rows[s], acc[0, k, i])


# ----------------------------------------------------------------------------- V5
def _tables_py(n_phi):
    q = n_phi // 4
    c = np.zeros(n_phi, np.float32)
    s = np.zeros(n_phi, np.float32)
    for i in range(q):
        th = (i + 0.5) * (2.0 * 3.14159265358979323846 / n_phi)
        c[i] = np.float32(math.cos(th))
        s[i] = np.float32(math.sin(th))
    for i in range(n_phi - q):
        c[i + q] = -s[i]
        s[i + q] = c[i]
    return c, s


def _vote_2d_numpy(hits, n_phi, n_qpt, qmin, qmax, bz):
    """Hand-written 2-D special case: v = (0 - w) * (1 / (A r2)), numpy float32 (each op rounded)."""
    f32 = np.float32
    c, s = _tables_py(n_phi)
    A = f32(0.5 * K * bz)
    inv_wq = f32(n_qpt / (float(qmax) - float(qmin)))
    acc = np.zeros((n_phi, n_qpt), np.int32)
    x = hits[:, 0:1].astype(f32)
    y = hits[:, 1:2].astype(f32)
    r2 = x * x + y * y
    w = y * c[None, :] - x * s[None, :]
    f = x * c[None, :] + y * s[None, :]
    with np.errstate(all="ignore"):
        v = (f32(0.0) - w) * (f32(1.0) / (A * r2))
        t = (v - f32(qmin)) * inv_wq
    ok = (f > 0) & (t >= 0) & (t < f32(n_qpt))
    hh, ii = np.nonzero(ok)
    np.add.at(acc, (ii, t[hh, ii].astype(np.int32)), 1)
    return acc


def test_v5_2d_special_case_bit_exact():
    w = get_workload(0)
    b = generate_events(w)
    bn = w.binning
    o2 = Oracle.from_binning(bn, w.bz_tesla)
    acc2, _ = o2.vote(b.hits_xy)
    ref = _vote_2d_numpy(b.hits_xy, bn.n_phi, bn.n_qpt, bn.qpt_min, bn.qpt_max, w.bz_tesla)
    assert np.array_equal(acc2[0, 0], ref)
    # slice with d0 centre exactly 0 of an odd-n_d0 plan == the 2-D accumulator
    o3 = Oracle(bn.n_phi, bn.n_qpt, 5, bn.qpt_min, bn.qpt_max, -20.0, 20.0, w.bz_tesla)
    assert o3.tables()["d0c"][2] == 0.0
    acc3, _ = o3.vote(b.hits_xy, k_range=(2, 3))
    assert np.array_equal(acc3[0, 0], acc2[0, 0])
    # and the other slices differ (d0 really enters)
    accn, _ = o3.vote(b.hits_xy, k_range=(1, 2))
    assert not np.array_equal(accn[0, 0], acc2[0, 0])


# ----------------------------------------------------------------------------- V6
@pytest.mark.parametrize("cfg,shape", [(0, (256, 256, 1)), (1, (64, 32, 8))])
def test_v6_quarter_turn_shifts_accumulator_exactly(cfg, shape):
    w = get_workload(cfg)
    hits = generate_events(w).hits_xy[:300]
    o = Oracle(*shape, bz_tesla=BZ)
    acc, _ = o.vote(hits)
    rot = hits.copy()
    for m in (1, 2, 3):
        rot = np.stack([-rot[:, 1], rot[:, 0]], 1)        # (x, y) -> (-y, x), exact in fp32
        am, _ = o.vote(rot)
        assert np.array_equal(am, np.roll(acc, m * shape[0] // 4, axis=2))


def test_v6_integer_bin_rotation_statistical():
    w = get_workload(0)
    hits = generate_events(w).hits_xy.astype(np.float64)
    o = Oracle(256, 256, 1, bz_tesla=BZ)
    acc, votes = o.vote(hits.astype(np.float32))
    m = 37
    a = m * 2 * np.pi / 256
    rot = np.stack([np.cos(a) * hits[:, 0] - np.sin(a) * hits[:, 1],
                    np.sin(a) * hits[:, 0] + np.cos(a) * hits[:, 1]], 1).astype(np.float32)
    am, _ = o.vote(rot)
    l1 = np.abs(am - np.roll(acc, m, axis=2)).sum()
    assert l1 <= max(8, 4e-3 * votes)      # a handful of edge votes move by one bin; a wrong shift gives ~2*votes
    assert l1 < 0.02 * votes


# ----------------------------------------------------------------------------- V7
def test_v7_single_cell_and_plateaus():
    o = Oracle(8, 6, 4, bz_tesla=BZ)
    T = 5
    acc = np.zeros((1, 4, 8, 6), np.int32)
    acc[0, 2, 3, 4] = T
    c = o.find_peaks(acc, T)
    assert c.total == 1 and tuple(c.records[0][["k", "i", "j", "votes"]]) == (2, 3, 4, T)
    assert c.records[0]["qpt"] == np.float32(-1.0 + 4.5 * (2.0 / 6))       # lone cell: centroid = centre
    assert o.find_peaks(acc, T + 1).total == 0                            # S9: a >= threshold
    # constant volume: every bin has an equal neighbour "before" it (phi wraps) -> no peak
    assert o.find_peaks(np.full((1, 4, 8, 6), 3, np.int32), 1).total == 0
    # two-bin plateaus: exactly one winner, the FIRST in (k, i, j) order
    for d in [(0, 0, 1), (0, 1, 0), (1, 0, 0), (0, 1, -1), (1, -1, 1), (1, 1, -1)]:
        acc = np.zeros((1, 4, 8, 6), np.int32)
        p = (1, 3, 3)
        q = (1 + d[0], 3 + d[1], 3 + d[2])
        acc[0][p] = 4
        acc[0][q] = 4
        c = o.find_peaks(acc, 1)
        assert c.total == 1 and tuple(c.records[0][["k", "i", "j"]]) == min(p, q), d
    # wrap-around in phi0: peak at i = 0 sees i = n_phi-1
    acc = np.zeros((1, 4, 8, 6), np.int32)
    acc[0, 1, 0, 2] = 5
    acc[0, 1, 7, 2] = 6
    c = o.find_peaks(acc, 1)
    assert c.total == 1 and tuple(c.records[0][["k", "i", "j"]]) == (1, 7, 2)
    # centroid wraps into [0, 2pi)
    assert 0.0 <= c.records[0]["phi0"] < 2 * math.pi
    # faces in j and k: no wrap there
    acc = np.zeros((1, 4, 8, 6), np.int32)
    acc[0, 0, 2, 0] = 5
    acc[0, 3, 2, 5] = 5
    acc[0, 0, 5, 5] = 5
    c = o.find_peaks(acc, 1)
    assert c.total == 3
    assert [tuple(r) for r in c.records[["k", "i", "j"]]] == [(0, 2, 0), (0, 5, 5), (3, 2, 5)]   # D6 order


@pytest.mark.parametrize("shape", [(1, 8, 8), (3, 8, 5), (4, 12, 7), (2, 4, 9)])
def test_v7_random_volumes_vs_definition(shape):
    nd, nphi, nq = shape
    o = Oracle(nphi, nq, nd, bz_tesla=BZ)
    rng = np.random.default_rng(nd * 100 + nphi)
    for trial in range(6):
        acc = rng.integers(0, 4 + trial, size=(2, nd, nphi, nq)).astype(np.int32)   # many ties
        thr = 2
        c = o.find_peaks(acc, thr)
        exp = []
        for e in range(2):
            exp += [(e,) + p for p in brute_peaks(acc[e], thr)]
        got = [tuple(int(v) for v in r) for r in c.records[["event", "k", "i", "j"]]]
        assert got == exp
        assert c.offsets[0] == 0 and c.offsets[2] == len(exp) == c.total
        assert c.offsets[1] == sum(1 for p in exp if p[0] == 0)
        for r in c.records:
            assert r["votes"] == acc[r["event"], r["k"], r["i"], r["j"]]
        # capacity truncation keeps true counts (S12)
        if c.total > 2:
            ct = o.find_peaks(acc, thr, capacity=2)
            assert ct.total == c.total and len(ct.records) == 2 and np.array_equal(ct.records, c.records[:2])
            assert np.array_equal(ct.offsets, c.offsets)


def test_v7_centroid_integer_moments():
    o = Oracle(8, 8, 1, bz_tesla=BZ)
    acc = np.zeros((1, 1, 8, 8), np.int32)
    acc[0, 0, 4, 4] = 6
    acc[0, 0, 4, 5] = 2          # +dj
    acc[0, 0, 3, 4] = 1          # -di
    c = o.find_peaks(acc, 6)
    assert c.total == 1
    r = c.records[0]
    S = 9.0
    assert abs(r["qpt"] - (-1.0 + (4.5 + 2.0 / S) * 0.25)) < 1e-6
    assert abs(r["phi0"] - ((4.5 - 1.0 / S) * 2 * math.pi / 8)) < 1e-6
    assert r["d0"] == 0.0


def test_v7_centroid_d0_term_asymmetric_neighbourhood():
    """D7, the d0 offset: a constructed 3-D volume whose three moments differ in sign and size, values by hand.
    centre 6 at (k,i,j) = (1,4,4); 2 at k+1; 1 at k-1; 1 at i-1  ->  S = 10, Sk = +1, Si = -1, Sj = 0."""
    o = Oracle(8, 8, 4, qpt_min=-1.0, qpt_max=1.0, d0_min=-20.0, d0_max=20.0, bz_tesla=BZ)
    acc = np.zeros((1, 4, 8, 8), np.int32)
    acc[0, 1, 4, 4] = 6
    acc[0, 2, 4, 4] = 2          # +dk
    acc[0, 0, 4, 4] = 1          # -dk
    acc[0, 1, 3, 4] = 1          # -di
    c = o.find_peaks(acc, 6)
    assert c.total == 1 and tuple(c.records[0][["k", "i", "j", "votes"]]) == (1, 4, 4, 6)
    r = c.records[0]
    wd, wq, wphi = 10.0, 0.25, 2 * math.pi / 8
    assert abs(r["d0"] - (-20.0 + (1.5 + 1.0 / 10.0) * wd)) < 2e-6          # = -4.0: Sk enters with +, scaled by wd
    assert abs(r["phi0"] - ((4.5 - 1.0 / 10.0) * wphi)) < 1e-6
    assert abs(r["qpt"] - (-1.0 + 4.5 * wq)) < 1e-6
    # the mirrored volume moves d0 the other way (a sign error in Sk cannot satisfy both)
    acc[0, 2, 4, 4], acc[0, 0, 4, 4] = 1, 2
    r = o.find_peaks(acc, 6).records[0]
    assert abs(r["d0"] - (-20.0 + (1.5 - 1.0 / 10.0) * wd)) < 2e-6
    # peak on the k = 0 face: the missing slice contributes nothing (clipped, S10)
    acc = np.zeros((1, 4, 8, 8), np.int32)
    acc[0, 0, 2, 2] = 7
    acc[0, 1, 2, 2] = 3
    r = o.find_peaks(acc, 7).records[0]
    assert abs(r["d0"] - (-20.0 + (0.5 + 3.0 / 10.0) * wd)) < 2e-6


def test_v7_centroid_phi_wrap_both_branches():
    """D7: "phi0 ... wrapped into [0, 2pi) by one +-2pi".  A peak at i = 0 whose weight sits at i = n_phi - 1 has
    (i + 0.5 + Si/S) < 0 and must come back just below 2pi; the mirror case at i = n_phi - 1 comes back just above 0."""
    n = 8
    o = Oracle(n, 8, 1, bz_tesla=BZ)
    wphi = 2 * math.pi / n
    acc = np.zeros((1, 1, n, 8), np.int32)
    acc[0, 0, 0, 4] = 5
    acc[0, 0, n - 1, 3:6] = 4        # three "before" neighbours, each < 5, together heavier than the centre
    c = o.find_peaks(acc, 5)
    assert c.total == 1 and tuple(c.records[0][["i", "j"]]) == (0, 4)
    ti = 0.5 - 12.0 / 17.0           # S = 17, Si = -12
    assert ti < 0
    exp = ti * wphi + 2 * math.pi
    assert 2 * math.pi - wphi <= c.records[0]["phi0"] < np.float32(2 * math.pi)
    assert abs(c.records[0]["phi0"] - exp) < 2e-6
    acc = np.zeros((1, 1, n, 8), np.int32)
    acc[0, 0, n - 1, 4] = 5
    acc[0, 0, 0, 3:6] = 4            # three "after" neighbours
    c = o.find_peaks(acc, 5)
    assert c.total == 1 and tuple(c.records[0][["i", "j"]]) == (n - 1, 4)
    ti = n - 0.5 + 12.0 / 17.0
    assert ti > n
    exp = ti * wphi - 2 * math.pi
    assert 0.0 <= c.records[0]["phi0"] < wphi
    assert abs(c.records[0]["phi0"] - exp) < 2e-6


def test_s5_top_edge_is_decided_on_t():
    """S5: the range test is on t itself.  q/pT = 1 - 2^-24 (the fp32 just below q_max = 1) is inside [q_min, q_max)
    mathematically, but (v - q_min) = 2 - 2^-24 rounds to 2.0, t = n_qpt, and the vote is DROPPED; v = 1 - 2^-23
    lands in the last bin.  Hits are searched (seeded) on the column's q/pT = 1 circle; fp32 numpy mirrors D3 only to
    pick which of the candidate hits realise those two values; the assertions are the reading's."""
    n_phi, n_qpt, i = 64, 32, 5
    o = Oracle(n_phi, n_qpt, 1, bz_tesla=BZ)
    t = o.tables()
    c, s, A = np.float32(t["cosT"][i]), np.float32(t["sinT"][i]), np.float32(t["A_f"])
    th = (i + 0.5) * 2 * math.pi / n_phi
    Rc = 1.0 / (K * float(np.float32(BZ)) * 1.0)                 # radius of the q/pT = +1 circle through the origin
    rng = np.random.default_rng(5)
    a = rng.uniform(0.02, 0.6, 400000)                          # tangent-chord angle; hit = chord of length 2 R sin(a)
    r = 2 * Rc * np.sin(a)
    ang = th - a                                                # positive charge bends clockwise (D1)
    x = (r * np.cos(ang)).astype(np.float32)
    y = (r * np.sin(ang)).astype(np.float32)
    r2 = x * x + y * y
    w = y * c - x * s
    v = (np.float32(0.0) - w) * (np.float32(1.0) / (A * r2))
    below1 = np.nextafter(np.float32(1.0), np.float32(0.0))
    below2 = np.nextafter(below1, np.float32(0.0))
    drop = np.nonzero(v == below1)[0][:16]
    keep = np.nonzero(v == below2)[0][:16]
    assert len(drop) >= 4 and len(keep) >= 4
    for h in drop:
        hit = np.array([[x[h], y[h]]], np.float32)
        # in range in exact arithmetic on the fp32 value v = 1 - 2^-24 < q_max ...
        assert float(below1) < 1.0
        # ... yet no vote: t == n_qpt exactly
        assert o.vote_columns(hit, None, [[0, 0, i]]).sum() == 0
    for h in keep:
        hit = np.array([[x[h], y[h]]], np.float32)
        row = o.vote_columns(hit, None, [[0, 0, i]])[0]
        assert row.sum() == 1 and row[n_qpt - 1] == 1


def test_v7_slab_peaks_equal_full_volume():
    w = get_workload(1)
    hits = generate_events(w).hits_xy
    o = Oracle(64, 32, 16, bz_tesla=BZ)
    acc, _ = o.vote(hits)
    full = o.find_peaks(acc, 5)
    sub = full.records[(full.records["k"] >= 4) & (full.records["k"] < 9)]
    slab, _ = o.vote(hits, k_range=(3, 10))
    part = o.find_peaks(slab, 5, k_range=(3, 10), k_out=(4, 9))
    assert part.total == len(sub) and np.array_equal(part.records, sub)


# ----------------------------------------------------------------------------- V8
@pytest.mark.parametrize("cfg", [0, 1])
def test_v8_assignment_bruteforce_vs_indexed_and_invariants(cfg):
    w = get_workload(cfg)
    b = generate_events(w)
    o = Oracle.from_binning(w.binning, w.bz_tesla)
    acc, _ = o.vote(b.hits_xy, b.event_offsets)
    c = o.find_peaks(acc, w.threshold)
    raw_b, _, _ = o.assign_brute(b.hits_xy, b.event_offsets, c, 1, w.min_hits, apply_dedup=False)
    raw_i, _, _ = o.assign_indexed(b.hits_xy, b.event_offsets, c, 1, w.min_hits, apply_dedup=False)
    assert np.array_equal(raw_b, raw_i)
    h2c_b, nh_b, keep_b = o.assign_brute(b.hits_xy, b.event_offsets, c, 1, w.min_hits)
    h2c_i, nh_i, keep_i = o.assign_indexed(b.hits_xy, b.event_offsets, c, 1, w.min_hits)
    assert np.array_equal(h2c_b, h2c_i) and np.array_equal(nh_b, nh_i) and np.array_equal(keep_b, keep_i)
    # invariants
    assert nh_b.sum() == (raw_b >= 0).sum()
    assert np.array_equal(nh_b, np.bincount(raw_b[raw_b >= 0], minlength=c.total))
    assert np.array_equal(keep_b.astype(bool), nh_b >= w.min_hits)
    assert np.array_equal(h2c_b, np.where((raw_b >= 0) & keep_b.astype(bool)[np.maximum(raw_b, 0)], raw_b, -1))
    # every assigned hit is compatible with its candidate: its own vote column holds a bin within dj
    for h in np.nonzero(raw_b >= 0)[0][:200]:
        r = c.records[raw_b[h]]
        col = o.vote_columns(b.hits_xy[h:h + 1], None, [[0, r["k"], r["i"]]])[0]
        jh = np.nonzero(col)[0]
        assert len(jh) == 1 and abs(int(jh[0]) - int(r["j"])) <= 1


def test_v8_best_candidate_key_order():
    """D8: more votes wins; then smaller |dj|; then the smaller index."""
    w = get_workload(0)
    o = Oracle(256, 256, 1, bz_tesla=BZ)
    i = 40
    phi0 = (i + 0.5) * 2 * math.pi / 256
    qpt = -1.0 + 100.5 * 2.0 / 256
    hits = helix_hits(phi0, qpt, 0.0, LAYERS_10, BZ)[:1]
    from oracle import CAND_DTYPE, OracleCandidates

    def cands(lst):
        rec = np.zeros(len(lst), CAND_DTYPE)
        for n, (ii, jj, vv) in enumerate(lst):
            rec[n]["i"], rec[n]["j"], rec[n]["votes"] = ii, jj, vv
        return OracleCandidates(rec, np.array([0, len(lst)], np.int32), len(lst))

    def best(lst, dj=1):
        return int(o.assign_brute(hits, None, cands(lst), dj, 0, apply_dedup=False)[0][0])

    assert best([(i, 100, 5)]) == 0
    assert best([(i, 102, 9)]) == -1 and best([(i, 102, 9)], dj=2) == 0
    assert best([(i, 101, 5), (i, 100, 5)]) == 1            # smaller |dj| wins at equal votes
    assert best([(i, 101, 6), (i, 100, 5)]) == 0            # votes dominate |dj|
    assert best([(i, 99, 5), (i, 101, 5)]) == 0             # equal key -> smaller index
    assert best([((i + 128) % 256, 100, 50)]) == -1         # backward column is never compatible
    for lst in ([(i, 101, 5), (i, 100, 5)], [(i, 99, 5), (i, 101, 5)], [(i, 101, 6), (i, 100, 5)]):
        assert best(lst) == int(o.assign_indexed(hits, None, cands(lst), 1, 0, apply_dedup=False)[0][0])


def test_v8_capacity_limits_participants():
    w = get_workload(1)
    b = generate_events(w)
    o = Oracle.from_binning(w.binning, w.bz_tesla)
    acc, _ = o.vote(b.hits_xy)
    c = o.find_peaks(acc, w.threshold)
    cap = c.total // 2
    ct = o.find_peaks(acc, w.threshold, capacity=cap)
    h_b, nh_b, _ = o.assign_brute(b.hits_xy, None, ct, 1, w.min_hits, capacity=cap)
    h_i, nh_i, _ = o.assign_indexed(b.hits_xy, None, ct, 1, w.min_hits, capacity=cap)
    assert np.array_equal(h_b, h_i) and np.array_equal(nh_b, nh_i) and h_b.max() < cap and len(nh_b) == cap


# ----------------------------------------------------------------------------- V12 (D12: re-assignment rounds)
def _hit_bins(o, hits, k, i):
    """q/pT bin of every hit in column (k, i), -1 = no vote: one single-hit accumulator column per hit (D3, pinned by V1-V6)."""
    out = np.full(len(hits), -1, np.int64)
    for h in range(len(hits)):
        nz = np.nonzero(o.vote_columns(hits[h:h + 1], None, [[0, k, i]])[0])[0]
        assert len(nz) <= 1
        if len(nz):
            out[h] = nz[0]
    return out


def _rounds_python(jh, votes, cj, dj, min_hits, max_rounds):
    """D12 written out in numpy from its definition.  jh[h, c] = bin of hit h in candidate c's column."""
    n_h, n_c = jh.shape
    alive = np.ones(n_c, bool)
    nh = np.zeros(n_c, np.int64)
    rounds = 0
    while True:
        rounds += 1
        h2c = np.full(n_h, -1, np.int64)
        for h in range(n_h):
            best = None
            for c in range(n_c):
                if not alive[c] or jh[h, c] < 0 or abs(jh[h, c] - cj[c]) > dj:
                    continue
                key = (votes[c], -abs(jh[h, c] - cj[c]), -c)
                if best is None or key > best[0]:
                    best = (key, c)
            if best is not None:
                h2c[h] = best[1]
        cnt = np.bincount(h2c[h2c >= 0], minlength=n_c)
        nh[alive] = cnt[alive]
        drop = alive & (cnt < min_hits)
        alive &= ~drop
        if not drop.any() or rounds >= max_rounds:
            break
    h2c[(h2c >= 0) & ~alive[np.maximum(h2c, 0)]] = -1
    return h2c, nh, alive, rounds


def test_v12_shared_hit_case_by_hand():
    """One noiseless helix, its own bin as candidate 0 (10 votes) and a neighbour-column candidate 1 with MORE votes
    that only the outer hits reach.  D9 leaves the outer hits unassigned; the second round hands them to candidate 0."""
    from oracle import CAND_DTYPE, OracleCandidates
    o = Oracle(256, 256, 1, bz_tesla=BZ)
    i, j = 40, 100
    hits = helix_hits((i + 0.5) * 2 * math.pi / 256, -1.0 + (j + 0.5) * 2.0 / 256, 0.0, LAYERS_10, BZ)
    own = _hit_bins(o, hits, 0, i)
    assert (own == j).all()                                       # V2: every hit votes in the helix's own bin
    nb = _hit_bins(o, hits, 0, i + 1)
    j1 = int(nb[-1])                                              # where the outermost hit lands one column on
    reach = np.abs(nb - j1) <= 1
    n1 = int(reach.sum())
    assert 1 <= n1 <= 4 and reach[-1] and not reach[0]            # only a few outer hits are compatible with candidate 1
    rec = np.zeros(2, CAND_DTYPE)
    rec[0]["i"], rec[0]["j"], rec[0]["votes"] = i, j, 10
    rec[1]["i"], rec[1]["j"], rec[1]["votes"] = i + 1, j1, 12
    c = OracleCandidates(rec, np.array([0, 2], np.int32), 2)
    # D8 + D9: the outer hits prefer candidate 1 (12 votes), which then fails min_hits = 5 and strands them
    h9, nh9, keep9 = o.assign_brute(hits, None, c, 1, 5)
    assert np.array_equal(h9, np.where(reach, -1, 0)) and list(nh9) == [10 - n1, n1] and list(keep9) == [1, 0]
    h1, nh1, keep1, r1 = o.assign_rounds(hits, None, c, 1, 5, max_rounds=1)
    assert r1 == 1 and np.array_equal(h1, h9) and np.array_equal(nh1, nh9) and np.array_equal(keep1, keep9)
    # D12: round 2 re-associates them with the surviving candidate
    h2, nh2, keep2, r2 = o.assign_rounds(hits, None, c, 1, 5, max_rounds=8)
    assert r2 == 2 and (h2 == 0).all() and list(nh2) == [10, n1] and list(keep2) == [1, 0]
    # min_hits above what either can reach: both die in round 1, nothing to re-assign
    h3, nh3, keep3, r3 = o.assign_rounds(hits, None, c, 1, 11, max_rounds=8)
    assert r3 == 2 and (h3 == -1).all() and list(nh3) == [10 - n1, n1] and list(keep3) == [0, 0]


@pytest.mark.parametrize("min_hits,dj", [(3, 1), (6, 1), (8, 2), (1, 0)])
def test_v12_rounds_vs_python_bruteforce(min_hits, dj):
    """Config 0 with its real candidate list plus decoys: every output and the round count against the definition
    written out in numpy on top of the (pinned) per-hit vote bins."""
    from oracle import OracleCandidates
    w = get_workload(0)
    b = generate_events(w)
    o = Oracle.from_binning(w.binning, w.bz_tesla)
    acc, _ = o.vote(b.hits_xy)
    c = o.find_peaks(acc, 6)                                       # lower threshold: more (and more dubious) candidates
    rec = c.records[:60].copy()
    cands = OracleCandidates(rec, np.array([0, len(rec)], np.int32), len(rec))
    hits = b.hits_xy[:120]
    jh = np.stack([_hit_bins(o, hits, int(r["k"]), int(r["i"])) for r in rec], axis=1)
    for max_rounds in (1, 2, 5):
        exp = _rounds_python(jh, rec["votes"].astype(np.int64), rec["j"].astype(np.int64), dj, min_hits, max_rounds)
        got = o.assign_rounds(hits, None, cands, dj, min_hits, max_rounds=max_rounds)
        assert np.array_equal(got[0], exp[0]) and np.array_equal(got[1], exp[1])
        assert np.array_equal(got[2].astype(bool), exp[2]) and got[3] == exp[3]


@pytest.mark.parametrize("cfg", [0, 1, 5])
def test_v12_fixed_point_properties(cfg):
    """What must hold whatever the input: max_rounds = 1 is D9; the kept set is D9's kept set (a kept candidate only gains
    hits); two rounds reach the fixed point; the result equals a brute-force D8 over the kept candidates alone."""
    from oracle import OracleCandidates
    w = get_workload(cfg)
    b = generate_events(w)
    o = Oracle.from_binning(w.binning, w.bz_tesla)
    acc, _ = o.vote(b.hits_xy, b.event_offsets)
    c = o.find_peaks(acc, w.threshold)
    h9, nh9, keep9 = o.assign_indexed(b.hits_xy, b.event_offsets, c, w.assoc_dj, w.min_hits)
    h1, nh1, keep1, r1 = o.assign_rounds(b.hits_xy, b.event_offsets, c, w.assoc_dj, w.min_hits, max_rounds=1)
    assert r1 == 1 and np.array_equal(h1, h9) and np.array_equal(nh1, nh9) and np.array_equal(keep1, keep9)
    hr, nhr, keepr, rr = o.assign_rounds(b.hits_xy, b.event_offsets, c, w.assoc_dj, w.min_hits, max_rounds=8)
    assert rr <= 2 and np.array_equal(keepr, keep9)
    kept = keep9.astype(bool)
    assert (nhr[kept] >= nh9[kept]).all() and np.array_equal(nhr[~kept], nh9[~kept])
    assert np.array_equal(hr[h9 >= 0], h9[h9 >= 0])               # hits that had a kept candidate keep it
    assert np.array_equal(nhr[kept], np.bincount(hr[hr >= 0], minlength=c.total)[kept])
    # brute-force D8 over the kept candidates alone, indices mapped back
    idx = np.nonzero(kept)[0]
    sub = OracleCandidates(c.records[idx].copy(), np.array([0, len(idx)], np.int32), len(idx))
    hs, _, _ = o.assign_brute(b.hits_xy, b.event_offsets, sub, w.assoc_dj, 0, apply_dedup=False)
    assert np.array_equal(hr, np.where(hs >= 0, idx[np.maximum(hs, 0)], -1))
    assert (hr >= 0).sum() > (h9 >= 0).sum() or cfg == 0          # the rounds do recover hits on the busy workloads


# ----------------------------------------------------------------------------- workload sanity
def test_workload_shapes_match_baseline():
    """Hit counts of the generated configs sit where BASELINE.json says ("about 210", "about 33k" ...)."""
    exp = {0: (205, 215), 1: (1900, 2010), 2: (32000, 34000), 4: (155000, 170000)}
    for cfg, (lo, hi) in exp.items():
        w = get_workload(cfg)
        b = generate_events(w)
        assert lo <= b.n_hits <= hi, (cfg, b.n_hits)
        r = np.hypot(b.hits_xy[:, 0].astype(np.float64), b.hits_xy[:, 1])
        lay = np.array(w.layers)
        assert np.abs(r[:, None] - lay[None, :]).min(axis=1).max() < 1e-4     # every hit sits on a layer
    w3 = get_workload(3)
    b3 = generate_events(w3, events=range(4))
    per = np.diff(b3.event_offsets)
    assert ((per > 8000) & (per < 9100)).all()
    # event e is the same whether generated alone or in a batch (per-event Philox key)
    assert np.array_equal(generate_events(w3, events=[2]).hits_xy, b3.event(2))
    assert len(LAYERS_14) == 14


def test_paper_toy_workload_shape_and_physics_sanity():
    """PAPER.md:39 (Fig. 1): beampipe 3.0 cm, ten evenly spaced layers out to 110.0 cm, 500 curved prompt tracks.
    Not a parity pin: the found-track fraction depends on the (unstated) binning; it only has to be sane."""
    import math
    from workloads import LAYERS_PAPER_TOY
    w = get_workload(5)
    assert len(w.layers) == 10 and abs(w.layers[-1] - 110.0) < 1e-9 and abs(w.layers[0] - 13.7) < 1e-9
    assert np.allclose(np.diff((3.0,) + tuple(LAYERS_PAPER_TOY)), 10.7)
    assert w.n_prompt == 500 and w.n_displaced == 0 and w.binning.n_d0 == 1 and abs(w.sigma_rphi_cm - 0.04) < 1e-12
    batch = generate_events(w, want_truth=True)
    r = np.hypot(batch.hits_xy[:, 0], batch.hits_xy[:, 1])
    assert batch.n_hits == 5000 and np.allclose(np.sort(np.unique(np.round(r, 3))), np.round(LAYERS_PAPER_TOY, 3), atol=2e-3)
    o = Oracle.from_binning(w.binning, w.bz_tesla)
    acc, votes = o.vote(batch.hits_xy, batch.event_offsets)
    ref = o.find_peaks(acc, w.threshold)
    h2c, nh, keep = o.assign_indexed(batch.hits_xy, batch.event_offsets, ref, w.assoc_dj, w.min_hits)
    rec = ref.records[keep.astype(bool)]
    t = batch.truth[0]
    bn = w.binning
    ti = np.floor(np.mod(t["direction"], 2 * math.pi) / (2 * math.pi) * bn.n_phi).astype(int)
    tj = np.floor((t["charge"] / t["pt"] - bn.qpt_min) / (bn.qpt_max - bn.qpt_min) * bn.n_qpt).astype(int)
    found = 0
    for a, c in zip(ti, tj):
        d = np.abs(((rec["i"] - a + bn.n_phi // 2) % bn.n_phi) - bn.n_phi // 2)
        found += bool(np.any((d <= 1) & (np.abs(rec["j"] - c) <= 2)))
    assert 0.25 < found / 500 < 1.0 and len(rec) < 500


# ---- D3L: straight displaced tracks, two-parameter space (phi0, d0) ----------------
def _line_oracle(n_phi, n_d, dmin, dmax):
    return Oracle(n_phi, n_d, 1, dmin, dmax, model=1)


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_v1l_line_bruteforce_double_geometry(seed):
    """Brute force in double from the definition: a line of direction theta_i through p has impact parameter
    d0 = p . n_hat; forward iff p . t_hat > 0.  Compared wherever the double value is away from a bin edge."""
    rng = np.random.default_rng(seed)
    n_phi, n_d, dmin, dmax = 16, 12, -9.0, 7.0
    hits = rng.uniform(-40, 40, (9, 2)).astype(np.float32)
    acc, votes = _line_oracle(n_phi, n_d, dmin, dmax).vote(hits)
    exp = np.zeros((n_phi, n_d), np.int64)
    unsafe = np.zeros((n_phi, n_d), bool)
    for x, y in hits.astype(np.float64):
        for i in range(n_phi):
            th = (i + 0.5) * 2 * math.pi / n_phi
            f = x * math.cos(th) + y * math.sin(th)
            d0 = -x * math.sin(th) + y * math.cos(th)
            t = (d0 - dmin) / ((dmax - dmin) / n_d)
            near = abs(t - round(t)) < 1e-4 or abs(f) < 1e-5
            j = int(math.floor(t))
            if near:
                for jj in (j - 1, j, j + 1):
                    if 0 <= jj < n_d:
                        unsafe[i, jj] = True
            if f > 0 and 0 <= t < n_d:
                exp[i, j] += 1
    got = acc[0, 0].astype(np.int64)
    assert votes == got.sum() and np.array_equal(got[~unsafe], exp[~unsafe]) and (~unsafe).mean() > 0.9


@pytest.mark.parametrize("shape,ij", [((256, 128), (37, 100)), ((512, 256), (300, 17)), ((64, 32), (0, 31))])
def test_v2l_noiseless_line_peaks_in_its_own_bin(shape, ij):
    from workloads import LAYERS_PAPER_TOY, line_hits
    n_phi, n_d = shape
    dmin, dmax = -12.0, 12.0
    i, j = ij
    phi0 = (i + 0.5) * 2 * math.pi / n_phi
    d0 = dmin + (j + 0.5) * (dmax - dmin) / n_d
    hits = line_hits(phi0, d0, LAYERS_PAPER_TOY)
    assert hits.shape[0] == 10
    o = _line_oracle(n_phi, n_d, dmin, dmax)
    acc, _ = o.vote(hits)
    a = acc[0, 0]
    assert a[i, j] == 10 and (a == 10).sum() == 1                     # every hit votes the true bin, nothing else reaches 10
    ref = o.find_peaks(acc, 10)
    assert ref.total == 1 and (ref.records["i"][0], ref.records["j"][0], ref.records["votes"][0]) == (i, j, 10)
    h2c, nh, keep = o.assign_indexed(hits, None, ref, 1, 10)
    assert (h2c == 0).all() and nh[0] == 10 and keep[0] == 1
    # centroid: the `qpt` field carries d0 [cm] in this model; within one bin of the truth
    assert abs(ref.records["qpt"][0] - d0) <= (dmax - dmin) / n_d and abs(ref.records["phi0"][0] - phi0) <= 2 * math.pi / n_phi


def test_v3l_line_closed_form_vote_count_and_sinusoid():
    """A hit at radius r votes in the columns with dmin <= r sin(phi - theta) < dmax on the forward half: their number is
    n_phi (asin(min(dmax/r, 1)) - asin(max(dmin/r, -1))) / 2pi within +-1; the voted bins trace the sinusoid
    d0 = -x sin(theta) + y cos(theta)."""
    n_phi, n_d, dmin, dmax = 720, 64, -15.0, 10.0
    rng = np.random.default_rng(5)
    r = rng.uniform(3.0, 120.0, 40)
    ph = rng.uniform(0, 2 * math.pi, 40)
    hits = np.stack([r * np.cos(ph), r * np.sin(ph)], 1).astype(np.float32)
    o = _line_oracle(n_phi, n_d, dmin, dmax)
    per_hit = o.votes_per_hit(hits)
    exp = n_phi * (np.arcsin(np.minimum(dmax / r, 1.0)) - np.arcsin(np.maximum(dmin / r, -1.0))) / (2 * math.pi)
    assert np.all(np.abs(per_hit - exp) <= 1.0)
    acc, votes = o.vote(hits[:1])
    ii, jj = np.nonzero(acc[0, 0])
    th = (ii + 0.5) * 2 * math.pi / n_phi
    d0 = -float(hits[0, 0]) * np.sin(th) + float(hits[0, 1]) * np.cos(th)
    assert votes == per_hit[0] and np.all(np.abs(dmin + (jj + 0.5) * (dmax - dmin) / n_d - d0) <= 0.5 * (dmax - dmin) / n_d + 1e-4)


def test_v6l_line_quarter_turn_shifts_accumulator_exactly():
    w = get_workload(6)
    batch = generate_events(w)
    o = Oracle.from_binning(w.binning, w.bz_tesla)
    acc, _ = o.vote(batch.hits_xy, batch.event_offsets)
    rot = np.stack([-batch.hits_xy[:, 1], batch.hits_xy[:, 0]], 1)    # (x, y) -> (-y, x): exact in fp32
    acc_r, _ = o.vote(rot, batch.event_offsets)
    assert np.array_equal(np.roll(acc, w.binning.n_phi // 4, axis=2), acc_r)


def test_line_workload_vertices_show_as_sinusoids():
    """PAPER.md:61 / Fig. 3: tracks from one displaced vertex (xv, yv) lie on d0 = -xv sin(phi0) + yv cos(phi0)."""
    w = get_workload(6)
    batch = generate_events(w, want_truth=True)
    t = batch.truth[0]
    sx, sy, psi = t["start_x"], t["start_y"], t["direction"]
    d0_true = -sx * np.sin(psi) + sy * np.cos(psi)
    assert np.allclose(d0_true[:w.n_prompt], 0.0) and np.abs(d0_true[w.n_prompt:]).max() < 12.0 + 1e-9
    o = Oracle.from_binning(w.binning, w.bz_tesla)
    acc, _ = o.vote(batch.hits_xy, batch.event_offsets)
    ref = o.find_peaks(acc, w.threshold)
    h2c, nh, keep = o.assign_indexed(batch.hits_xy, batch.event_offsets, ref, w.assoc_dj, w.min_hits)
    rec = ref.records[keep.astype(bool)]
    bn = w.binning
    ti = np.floor(np.mod(psi, 2 * math.pi) / (2 * math.pi) * bn.n_phi).astype(int)
    tj = np.floor((d0_true - bn.qpt_min) / (bn.qpt_max - bn.qpt_min) * bn.n_qpt).astype(int)
    found = 0
    for a, c in zip(ti, tj):
        d = np.abs(((rec["i"] - a + bn.n_phi // 2) % bn.n_phi) - bn.n_phi // 2)
        found += bool(np.any((d <= 1) & (np.abs(rec["j"] - c) <= 2)))
    assert found / len(ti) > 0.2                                       # sanity only (binning-dependent)


# ---- D10: second Hough transform, found straight tracks -> displaced vertices --------
def _track_list(cols, bins, keep=None):
    from oracle import CAND_DTYPE, OracleCandidates
    rec = np.zeros(len(cols), CAND_DTYPE)
    rec["i"] = cols
    rec["j"] = bins
    return OracleCandidates(rec, np.array([0, len(rec)], np.int32), len(rec)), (np.ones(len(rec), np.uint8) if keep is None else keep)


def test_d10_bruteforce_double_and_closed_form_count():
    """Definition in double: vertex (R, Phi) is on the line (phi0, d0) iff d0 = R sin(Phi - phi0); one vote per column with
    0 <= R < r_max.  Per track the number of voting columns is n_phi (pi - 2 asin(|d0| / r_max)) / 2pi within +-1."""
    rng = np.random.default_rng(3)
    n_phi, n_d, dmin, dmax, n_r, r_max = 96, 64, -12.0, 12.0, 20, 15.0
    o = _line_oracle(n_phi, n_d, dmin, dmax)
    cols = rng.integers(0, n_phi, 12)
    bins = rng.integers(0, n_d, 12)
    cands, keep = _track_list(cols, bins)
    keep[3] = 0
    vacc, votes = o.vertex_vote(cands, keep, 0.5, n_r, r_max)
    exp = np.zeros((n_phi, n_r), np.int64)
    unsafe = np.zeros((n_phi, n_r), bool)
    per_track = []
    for c, (i, j) in enumerate(zip(cols, bins)):
        d0 = dmin + (j + 0.5) * (dmax - dmin) / n_d
        if not keep[c] or abs(d0) < 0.5:
            continue
        phi0 = (i + 0.5) * 2 * math.pi / n_phi
        n_cols = 0
        for m in range(n_phi):
            sd = math.sin((m + 0.5) * 2 * math.pi / n_phi - phi0)
            if abs(sd) < 1e-9:
                continue
            t = d0 / sd / (r_max / n_r)
            if abs(t - round(t)) < 1e-4:
                for nn in (int(math.floor(t)) - 1, int(math.floor(t)), int(math.floor(t)) + 1):
                    if 0 <= nn < n_r:
                        unsafe[m, nn] = True
            if 0 <= t < n_r:
                exp[m, int(math.floor(t))] += 1
                n_cols += 1
        per_track.append((d0, n_cols))
    got = vacc[0].astype(np.int64)
    assert votes == got.sum() and np.array_equal(got[~unsafe], exp[~unsafe]) and (~unsafe).mean() > 0.95
    for d0, n_cols in per_track:
        assert abs(n_cols - n_phi * (math.pi - 2 * math.asin(abs(d0) / r_max)) / (2 * math.pi)) <= 1.0


def test_d10_lines_through_one_vertex_peak_at_the_vertex():
    n_phi, n_d, dmin, dmax = 720, 1024, -16.0, 16.0
    o = _line_oracle(n_phi, n_d, dmin, dmax)
    r_v, phi_col = 7.3, 100                                 # vertex azimuth at a column centre
    phi_v = (phi_col + 0.5) * 2 * math.pi / n_phi
    xv, yv = r_v * math.cos(phi_v), r_v * math.sin(phi_v)
    cols = np.arange(7, n_phi, 20)
    th = (cols + 0.5) * 2 * math.pi / n_phi
    d_true = -xv * np.sin(th) + yv * np.cos(th)
    bins = np.floor((d_true - dmin) / ((dmax - dmin) / n_d)).astype(np.int32)
    cands, keep = _track_list(cols, bins)
    n_r, r_max = 64, 16.0
    vacc, votes = o.vertex_vote(cands, keep, 0.5, n_r, r_max)
    m_pk, n_pk = np.unravel_index(np.argmax(vacc[0]), vacc[0].shape)
    displaced = int((np.abs(dmin + (bins + 0.5) * (dmax - dmin) / n_d) >= 0.5).sum())
    assert m_pk == phi_col and n_pk == int(r_v / (r_max / n_r))
    assert vacc[0].max() >= 0.8 * displaced
    # quarter turn of every track: the vertex accumulator shifts by n_phi / 4 columns exactly (table symmetry, D2)
    cands_r, _ = _track_list((cols + n_phi // 4) % n_phi, bins)
    vacc_r, _ = o.vertex_vote(cands_r, keep, 0.5, n_r, r_max)
    assert np.array_equal(np.roll(vacc, n_phi // 4, axis=1), vacc_r)


def test_d10_workload_6_vertex_directions():
    """Sanity on the full chain (hits -> tracks -> vertices) of workload 6: the strongest vertex candidates point at true
    vertices.  (Radial resolution is poor for jets that fly radially -- their lines are almost parallel to the vertex's
    position vector -- so only the azimuth is checked; this is physics sanity, not a parity pin.)"""
    w = get_workload(6)
    batch = generate_events(w, want_truth=True)
    t = batch.truth[0]
    verts = np.unique(np.round(np.stack([t["start_x"][w.n_prompt:], t["start_y"][w.n_prompt:]], 1), 9), axis=0)
    assert verts.shape == (4, 2)
    o = Oracle.from_binning(w.binning, w.bz_tesla)
    acc, _ = o.vote(batch.hits_xy, batch.event_offsets)
    ref = o.find_peaks(acc, w.threshold)
    h2c, nh, keep = o.assign_indexed(batch.hits_xy, batch.event_offsets, ref, w.assoc_dj, w.min_hits)
    vacc, votes = o.vertex_vote(ref, keep, 0.6, 32, 16.0)
    assert votes > 1000
    vs = Oracle(w.binning.n_phi, 32, 1, 0.0, 16.0, bz_tesla=0.0, model=1)
    vref = vs.find_peaks(vacc[:, None], 6)
    rec = vref.records[np.argsort(-vref.records["votes"])[:6]]
    az_true = np.arctan2(verts[:, 1], verts[:, 0])
    for ph in rec["phi0"]:
        dphi = np.abs(np.angle(np.exp(1j * (az_true - float(ph)))))
        assert dphi.min() < math.radians(20.0)


# ---- D11: circle fit of the assigned hits ("obtain the best measurement of the track parameters"; f4) ------
@pytest.mark.parametrize("seed", [0, 1, 2, 3, 4, 5])
def test_d11_circle_fit_recovers_noiseless_helices(seed):
    """Noiseless hits of a helix (phi0, q/pT, d0) generated from the D1 geometry: the fit returns the parameters."""
    from oracle import CAND_DTYPE, OracleCandidates
    rng = np.random.default_rng(seed)
    n_phi = 256
    o = Oracle(n_phi, 128, 64)
    phi0 = rng.uniform(0, 2 * math.pi)
    qpt = rng.uniform(0.1, 0.9) * rng.choice([-1.0, 1.0])
    d0 = rng.uniform(-8.0, 8.0)
    hits = helix_hits(phi0, qpt, d0, LAYERS_14, 3.8)
    assert hits.shape[0] >= 5
    rec = np.zeros(2, CAND_DTYPE)
    rec["i"][1] = int(phi0 / (2 * math.pi) * n_phi)         # the candidate's column orients the fitted circle
    cands = OracleCandidates(rec, np.array([0, 2], np.int32), 2)
    h2c = np.ones(hits.shape[0], np.int32)                  # every hit assigned to candidate 1, none to candidate 0
    fit, nfit = o.fit_circles(hits, h2c, cands, np.array([1, 1], np.uint8))
    assert nfit[0] == 0 and nfit[1] == hits.shape[0]
    f = fit[1]
    assert abs(np.angle(np.exp(1j * (f[0] - phi0)))) < 2e-5 and abs(f[1] - qpt) < 2e-5 * max(1.0, abs(qpt)) and abs(f[2] - d0) < 2e-4
    assert abs(f[3] - 1.0 / abs(qpt * K * 3.8)) < 1e-3 * f[3]


def test_d11_fit_flags_and_textbook_circle():
    from oracle import CAND_DTYPE, OracleCandidates
    o = Oracle(64, 32, 1)
    # 8 exact points on the circle centre (3, -4), R = 10 (contains the origin side: |centre| = 5 < R)
    ang = np.linspace(0.1, 5.9, 8)
    pts = np.stack([3 + 10 * np.cos(ang), -4 + 10 * np.sin(ang)], 1).astype(np.float32)
    two = pts[:2]
    hits = np.concatenate([pts, two])
    rec = np.zeros(3, CAND_DTYPE)
    cands = OracleCandidates(rec, np.array([0, 3], np.int32), 3)
    h2c = np.array([0] * 8 + [1, 1], np.int32)
    fit, nfit = o.fit_circles(hits, h2c, cands, np.array([1, 1, 0], np.uint8))
    assert list(nfit) == [8, -2, 0]                          # ok; too few hits; dropped candidate
    assert abs(fit[0, 3] - 10.0) < 1e-5 and abs(abs(fit[0, 2]) - 5.0) < 1e-5      # R and |d0| = | |centre| - R |
