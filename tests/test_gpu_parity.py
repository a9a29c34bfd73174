"""-m gpu: the CUDA path through the C ABI vs the CPU oracle, element by element, on the same seeded inputs.

Bar (B:L5): accumulators, peak lists and hit assignments bit-exact; centroids within 1e-5 relative.
"""
import numpy as np
import pytest
import torch

from oracle import Oracle
from workloads import HoughBinning, generate_events, get_workload, helix_hits, LAYERS_10
from workloads.configs import ACC_I32, ACC_U16

pytestmark = pytest.mark.gpu

from gpu_util import (assert_centroids_close, oracle_peaks_parallel, oracle_vote_parallel, run_assign, run_cuda, run_vote)  # noqa: E402


def _narrow(acc_i32, binning):
    if binning.accum_dtype == ACC_U16:
        assert acc_i32.max() <= 65535          # U16 precondition, asserted on the oracle's int32 counts (D4)
        return acc_i32.astype(np.uint16)
    return acc_i32


def _compare_all(w, batch, binning=None, capacity=None, fullscan=False, oracle_parallel=False, options=()):
    bn = binning or w.binning
    o = Oracle.from_binning(bn, w.bz_tesla)
    if oracle_parallel:
        acc, votes = oracle_vote_parallel(o, batch.hits_xy, batch.event_offsets)
        ref = oracle_peaks_parallel(o, acc, w.threshold)
    else:
        acc, votes = o.vote(batch.hits_xy, batch.event_offsets)
        ref = o.find_peaks(acc, w.threshold)
    cap = ref.total + 7 if capacity is None else capacity
    got = run_cuda(bn, w.bz_tesla, w.layers, batch.hits_xy, batch.event_offsets, w.threshold, w.assoc_dj, w.min_hits,
                   cap, fullscan=fullscan, options=options)
    assert np.array_equal(got.accum, _narrow(acc, bn)), "accumulator differs"
    assert int(got.accum.astype(np.int64).sum()) == votes
    assert got.total == ref.total and np.array_equal(got.offsets, ref.offsets)
    n_c = min(cap, ref.total)
    for f in ("event", "k", "i", "j", "votes"):
        assert np.array_equal(got.records[f], ref.records[f][:n_c]), f
    assert_centroids_close(got.records, ref.records[:n_c], bn)
    ref_c = ref if n_c == ref.total else o.find_peaks(acc, w.threshold, capacity=cap)
    h2c, nh, keep = o.assign_indexed(batch.hits_xy, batch.event_offsets, ref_c, w.assoc_dj, w.min_hits, capacity=cap)
    assert np.array_equal(got.hit_to_cand, h2c), "hit_to_cand differs"
    assert np.array_equal(got.cand_nhits[:n_c], nh) and np.array_equal(got.cand_keep[:n_c], keep)
    assert not got.cand_nhits[n_c:].any() and not got.cand_keep[n_c:].any()
    return got, ref


@pytest.mark.parametrize("fullscan", [False, True])
@pytest.mark.parametrize("cfg", [0, 1])
def test_config_0_1_bit_exact(cfg, fullscan):
    w = get_workload(cfg)
    got, ref = _compare_all(w, generate_events(w), fullscan=fullscan)
    assert ref.total > 0


@pytest.mark.parametrize("cfg", [0, 1])
def test_config_0_1_exact_walk_and_tiled_peaks(cfg):
    """The bisecting options: D3 at every window column (no fast path) and the halo-tile peak kernels."""
    w = get_workload(cfg)
    _compare_all(w, generate_events(w), options=("exact_walk", "peaks_tiled"))
    _compare_all(w, generate_events(w), options=("assign_candidates",))


def test_paper_toy_workload_bit_exact():
    """the paper's own scenario (10 evenly spaced layers 3 -> 110 cm, 0.4 mm, 500 tracks)."""
    w = get_workload(5)
    got, ref = _compare_all(w, generate_events(w))
    assert ref.total > 100
    w2 = w.with_tracks(3000)                              # Fig. 2-style: more tracks, same detector
    _compare_all(w2, generate_events(w2))


def test_config_2_bit_exact():
    w = get_workload(2)
    _compare_all(w, generate_events(w), oracle_parallel=True)


def test_config_3_subset_of_events_bit_exact():
    w = get_workload(3)
    batch = generate_events(w, events=[0, 1, 513, 1023, 7])
    _compare_all(w, batch)
    _compare_all(w, batch, options=("assign_candidates",))


def test_config_3_fullscan_matches_tiled_on_more_events():
    """Both CUDA code paths agree with the oracle on a ragged 3-event batch (different hit counts)."""
    w = get_workload(3)
    batch = generate_events(w, events=[11, 12, 13])
    _compare_all(w, batch, fullscan=True)


def test_config_4_reduced_bins_bit_exact():
    """Config-4 hits (162k) into a reduced accumulator the oracle finishes in seconds: many tiles + ragged tail."""
    w = get_workload(4)
    batch = generate_events(w)
    bn = HoughBinning(128, 64, 16, accum_dtype=ACC_U16)
    o = Oracle.from_binning(bn, w.bz_tesla)
    acc, votes = oracle_vote_parallel(o, batch.hits_xy, batch.event_offsets)
    assert acc.max() <= 65535
    got = run_cuda(bn, w.bz_tesla, w.layers, batch.hits_xy, batch.event_offsets, 10 ** 6, 1, 1, 16)
    assert np.array_equal(got.accum, acc.astype(np.uint16))
    assert got.total == 0 and (got.hit_to_cand == -1).all()


def test_config_4_full_size_sampled_columns_and_slab_peaks():
    """Full config-4 size in the launch configuration bench.py uses; outputs the oracle computes one by one."""
    w = get_workload(4)
    bn = w.binning
    batch = generate_events(w)
    o = Oracle.from_binning(bn, w.bz_tesla)
    cap = bn.n_bins // 16
    got = run_cuda(bn, w.bz_tesla, w.layers, batch.hits_xy, batch.event_offsets, w.threshold, w.assoc_dj, w.min_hits, cap)
    rng = np.random.default_rng(4)
    cols = np.stack([np.zeros(48, np.int64), rng.integers(0, bn.n_d0, 48), rng.integers(0, bn.n_phi, 48)], 1)
    cols[0] = (0, 0, 0)
    cols[1] = (0, bn.n_d0 - 1, bn.n_phi - 1)
    rows = o.vote_columns(batch.hits_xy, batch.event_offsets, cols)
    for s, (_, k, i) in enumerate(cols):
        assert np.array_equal(got.accum[0, k, i].astype(np.int32), rows[s]), (k, i)
    # peaks in a d0 slab: the oracle votes slices 61..66 and reports peaks of slices 62..64
    slab, _ = o.vote(batch.hits_xy, batch.event_offsets, k_range=(61, 66))
    assert np.array_equal(got.accum[0, 61:66].astype(np.int32), slab[0])
    part = o.find_peaks(slab, w.threshold, k_range=(61, 66), k_out=(62, 65))
    sel = (got.records["k"] >= 62) & (got.records["k"] < 65)
    assert got.total <= cap
    sub = got.records[sel]
    assert len(sub) == part.total
    for f in ("event", "k", "i", "j", "votes"):
        assert np.array_equal(sub[f], part.records[f]), f
    assert_centroids_close(sub, part.records, bn)
    # properties that hold at any size
    lin = (got.records["k"].astype(np.int64) * bn.n_phi + got.records["i"]) * bn.n_qpt + got.records["j"]
    assert np.all(np.diff(lin) > 0)                                   # D6 order, no duplicates
    assert np.array_equal(got.records["votes"],
                          got.accum[0][got.records["k"], got.records["i"], got.records["j"]].astype(np.int32))
    assert got.records["votes"].min() >= w.threshold
    raw_assigned = got.cand_nhits[:got.total].sum()
    assert np.array_equal(got.cand_keep[:got.total].astype(bool), got.cand_nhits[:got.total] >= w.min_hits)
    kept_hits = np.bincount(got.hit_to_cand[got.hit_to_cand >= 0], minlength=got.total)
    assert np.array_equal(kept_hits, np.where(got.cand_keep[:got.total] > 0, got.cand_nhits[:got.total], 0))
    assert raw_assigned <= batch.n_hits


# ----------------------------------------------------------------------------- every tile variant of the vote
def _mixed_hits(seed, n, layers):
    """Hits on the layers (as generated) and at arbitrary radii (generic radius classes), several events."""
    rng = np.random.default_rng(seed)
    r = np.concatenate([rng.choice(np.asarray(layers), n // 2), rng.uniform(0.0, 150.0, n - n // 2 - 3), [1e-3, 19.99, 500.0]])
    ph = rng.uniform(0, 2 * np.pi, r.shape[0])
    hits = np.stack([r * np.cos(ph), r * np.sin(ph)], 1).astype(np.float32)
    cuts = np.sort(rng.integers(0, n, 2))
    off = np.array([0, cuts[0], cuts[0], cuts[1], n], np.int32)         # 4 events, one empty
    return hits, off


@pytest.mark.parametrize("shape,dtype,max_hits,layers,misalign", [
    ((256, 128, 4), ACC_U16, None, LAYERS_10, False),      # full-phi tile, packed, u16 out
    ((256, 128, 4), ACC_I32, None, LAYERS_10, True),       # full-phi tile, packed, i32 out, 8-byte aligned hits
    ((256, 128, 4), ACC_I32, 70000, LAYERS_10, False),     # 32-bit tile (a call may hold > 65535 hits)
    ((512, 256, 3), ACC_I32, None, LAYERS_10, False),      # phi slabs, packed, i32 out
    ((512, 256, 3), ACC_U16, None, (), True),              # phi slabs, u16 out, no geometry (uniform classes)
    ((1024, 512, 2), ACC_U16, None, LAYERS_10, False),     # config-4 row length, 16+ slabs
    ((100, 37, 3), ACC_U16, None, LAYERS_10, False),       # odd n_qpt: scalar flush, ragged last slab
    ((100, 37, 3), ACC_I32, 70000, LAYERS_10, True),
    ((64, 20000, 1), ACC_I32, None, LAYERS_10, False),     # a row larger than the small-tile budget
    ((8, 300000, 1), ACC_I32, 70000, LAYERS_10, False),    # a row that fits no tile: full-scan fallback
])
def test_vote_tile_variants_bit_exact(shape, dtype, max_hits, layers, misalign):
    bn = HoughBinning(*shape, accum_dtype=dtype)
    hits, off = _mixed_hits(shape[0] + shape[1], 3000, LAYERS_10)
    o = Oracle.from_binning(bn, 3.8)
    acc, votes = oracle_vote_parallel(o, hits, off)
    got = run_vote(bn, 3.8, layers, hits, off, max_hits=max_hits, misalign=misalign)
    assert votes > 0 and np.array_equal(got.astype(np.int32), acc)
    got = run_vote(bn, 3.8, layers, hits, off, max_hits=max_hits, misalign=misalign, options=("exact_walk",))
    assert np.array_equal(got.astype(np.int32), acc)


@pytest.mark.parametrize("seed", list(range(40)))
def test_random_configurations_bit_exact(seed):
    """Differential test over randomly drawn binnings (asymmetric and one-sided q/pT ranges, off-centre d0 ranges,
    odd sizes, both dtypes, several fields, with and without layer geometry): the fast path's error bound, windows and
    tile variants must never change a result."""
    rng = np.random.default_rng(1000 + seed)
    n_phi = 4 * int(rng.integers(2, 160))
    n_qpt = int(rng.choice([8, 24, 37, 64, 128, 200, 256, 333]))
    n_d0 = int(rng.choice([1, 2, 3, 5, 8]))
    model = 1 if seed % 5 == 3 else 0                      # straight-track space (phi0, d0): range in cm, one slice
    if model:
        n_d0 = 1
    qa, qb = sorted(rng.uniform(-1.5, 1.5, 2) * (25.0 if model else 1.0))
    if seed % 4 == 0:
        qa = 0.0                                           # one-sided range: c0 = 0
    if qb - qa < 0.2 * (25.0 if model else 1.0):
        qb = qa + 0.2 * (25.0 if model else 1.0)
    da, db = sorted(rng.uniform(-25.0, 25.0, 2))
    if db - da < 2.0:
        db = da + 2.0
    dtype = ACC_U16 if seed % 2 else ACC_I32
    bz = float(rng.choice([3.8, 2.0, -3.8, 1.0]))
    layers = LAYERS_10 if seed % 3 else ()
    bn = HoughBinning(n_phi, n_qpt, n_d0, float(np.float32(qa)), float(np.float32(qb)), float(np.float32(da)),
                      float(np.float32(db)), dtype, model)
    hits, off = _mixed_hits(5000 + seed, 2500, LAYERS_10)
    o = Oracle.from_binning(bn, bz)
    acc, votes = o.vote(hits, off)
    thr = 3
    dj = int(rng.integers(0, 4))
    ref = o.find_peaks(acc, thr)
    cap = ref.total + 5
    got = run_cuda(bn, bz, layers, hits, off, thr, dj, 2, cap)
    assert np.array_equal(got.accum.astype(np.int32), acc), "accumulator differs"
    assert got.total == ref.total and np.array_equal(got.offsets, ref.offsets)
    for f in ("event", "k", "i", "j", "votes"):
        assert np.array_equal(got.records[f], ref.records[f]), f
    assert_centroids_close(got.records, ref.records, bn)
    h2c, nh, keep = o.assign_indexed(hits, off, ref, dj, 2, capacity=cap)
    assert np.array_equal(got.hit_to_cand, h2c), "hit_to_cand differs"
    assert np.array_equal(got.cand_nhits[:ref.total], nh) and np.array_equal(got.cand_keep[:ref.total], keep)
    got_w = run_assign(bn, bz, layers, hits, off, ref.records, ref.offsets, cap, dj, 2, options=("assign_candidates",))
    assert np.array_equal(got_w[0], h2c), "hit_to_cand differs (candidate-centric path)"
    assert votes > 0 or seed % 4 != 1


def test_vote_half_circle_windows_and_negative_field():
    """A r q > 1 on the outer layers (windows = the whole forward half, wrap-around in every tile) and Bz < 0."""
    hits, off = _mixed_hits(9, 2000, LAYERS_10)
    for bz, q in ((3.8, 3.0), (-3.8, 1.0), (0.0, 1.0)):
        bn = HoughBinning(256, 64, 3, qpt_min=-q, qpt_max=q, d0_min=-1.0, d0_max=1.0)
        o = Oracle.from_binning(bn, bz)
        acc, votes = o.vote(hits, off)
        got = run_vote(bn, bz, LAYERS_10, hits, off)
        assert np.array_equal(got, acc), (bz, q)


@pytest.mark.parametrize("shape,dtype,max_hits,dj", [
    ((256, 128, 4), ACC_U16, None, 1),        # full-phi tiles, 16-bit entries
    ((256, 128, 4), ACC_I32, 70000, 2),       # 32-bit entries
    ((512, 256, 3), ACC_I32, None, 0),        # phi slabs, exact-bin association only
    ((512, 256, 3), ACC_U16, None, 3),        # phi slabs, wide association window
    ((100, 37, 3), ACC_U16, None, 1),         # ragged last slab, odd n_qpt
])
def test_assign_tile_variants_bit_exact(shape, dtype, max_hits, dj):
    """vote -> peaks -> assign through every tile variant of the association walk, vs the oracle's brute force."""
    bn = HoughBinning(*shape, accum_dtype=dtype)
    hits, off = _mixed_hits(shape[0] + dj, 3000, LAYERS_10)
    o = Oracle.from_binning(bn, 3.8)
    acc, _ = o.vote(hits, off)
    thr = 3
    ref = o.find_peaks(acc, thr)
    assert ref.total > 50
    h2c, nh, keep = o.assign_brute(hits, off, ref, dj, 2)
    for options in ((), ("exact_walk",), ("assign_candidates",)):     # the column walk (default) and the candidate-centric path
        got = run_assign(bn, 3.8, LAYERS_10, hits, off, ref.records, ref.offsets, ref.total + 5, dj, 2, max_hits=max_hits,
                         options=options)
        assert np.array_equal(got[0], h2c), options
        assert np.array_equal(got[1][:ref.total], nh) and np.array_equal(got[2][:ref.total], keep), options
    assert (h2c >= 0).sum() > 100


@pytest.mark.parametrize("shape,dtype,fullscan,tiled", [
    ((100, 37, 3), ACC_U16, False, False),      # odd rows: halo tiles; peak blocks that span two d0 slices
    ((100, 37, 3), ACC_I32, True, False),       # generic per-bin path
    ((64, 4096, 2), ACC_I32, False, False),     # slice walk, one row per peak block
    ((64, 4096, 2), ACC_I32, False, True),      # halo tiles, one row per peak block
    ((16, 20000, 2), ACC_U16, False, False),    # slice walk, long rows
    ((16, 20000, 2), ACC_U16, False, True),     # rows too long for the halo tile
    ((512, 256, 3), ACC_I32, False, False),
    ((512, 256, 3), ACC_I32, False, True),
    ((256, 128, 1), ACC_U16, False, False),     # 2-D: no neighbour slices at all
    ((256, 128, 1), ACC_U16, False, True),
    ((64, 64, 40), ACC_U16, False, False),      # slice walk cut into several slice runs
    ((32, 8, 5), ACC_I32, False, False),        # slice walk, one 16-byte chunk pair per row
    ((64, 64, 40), ACC_U16, False, "scalar"),   # 16-bit bins through the unpacked slice walk
    ((64, 64, 40), ACC_U16, False, "regs"),     # packed walk with register-held rows (no cp.async ring)
    ((256, 128, 1), ACC_U16, False, "regs"),
    ((512, 1024, 3), ACC_U16, False, False),    # cp.async ring: two rows per CTA (128 chunks per row)
    ((512, 2048, 3), ACC_U16, False, False),    # rows too long for the ring: packed register walk (peak_kwalk16)
    ((32, 8, 5), ACC_U16, False, False),        # packed slice walk, one chunk per row (both q/pT faces in one thread)
])
def test_peaks_tile_variants_bit_exact(shape, dtype, fullscan, tiled):
    bn = HoughBinning(*shape, accum_dtype=dtype)
    hits, off = _mixed_hits(shape[1], 2500, LAYERS_10)
    hits = np.concatenate([hits, hits[::3]])                      # duplicated hits -> plateaus
    off = np.array([0, 700, 700, hits.shape[0]], np.int32)
    o = Oracle.from_binning(bn, 3.8)
    acc, _ = o.vote(hits, off)
    thr = 2
    ref = o.find_peaks(acc, thr)
    assert ref.total > 20
    for cap in (ref.total + 3, ref.total // 2):
        got = run_cuda(bn, 3.8, LAYERS_10, hits, off, thr, 1, 2, cap, fullscan=fullscan,
                       options=("peaks_scalar",) if tiled == "scalar" else (("peaks_regs",) if tiled == "regs" else
                                                                              (("peaks_tiled",) if tiled else ())))
        assert got.total == ref.total and np.array_equal(got.offsets, ref.offsets)
        n_c = min(cap, ref.total)
        for f in ("event", "k", "i", "j", "votes"):
            assert np.array_equal(got.records[f], ref.records[f][:n_c]), f
        assert_centroids_close(got.records, ref.records[:n_c], bn)


def test_assign_saturated_votes_and_truncated_list():
    """Candidate votes at and beyond the 16-bit tile entry (exact through the record lookup) and capacity < total."""
    w = get_workload(1)
    bn = w.binning
    batch = generate_events(w)
    o = Oracle.from_binning(bn, w.bz_tesla)
    acc, _ = o.vote(batch.hits_xy)
    ref = o.find_peaks(acc, w.threshold)
    rec = ref.records.copy()
    rng = np.random.default_rng(1)
    sel = rng.choice(len(rec), 40, replace=False)
    rec["votes"][sel] = rng.choice([65533, 65534, 65535, 65536, 70000, 1 << 20], 40)
    from oracle import OracleCandidates
    mod = OracleCandidates(rec, ref.offsets, ref.total)
    for cap in (ref.total, ref.total // 2):
        h2c, nh, keep = o.assign_brute(batch.hits_xy, batch.event_offsets, mod, 1, 3, capacity=cap)
        for options in ((), ("assign_candidates",)):
            got = run_assign(bn, w.bz_tesla, w.layers, batch.hits_xy, batch.event_offsets, rec, ref.offsets, cap, 1, 3,
                             options=options)
            assert np.array_equal(got[0], h2c), (cap, options)
            assert np.array_equal(got[1][:cap], nh) and np.array_equal(got[2][:cap], keep)


# ----------------------------------------------------------------------------- edge cases
def test_empty_inputs_and_empty_events():
    w = get_workload(1)
    bn = HoughBinning(64, 32, 8)
    # no hits at all
    got = run_cuda(bn, w.bz_tesla, w.layers, np.zeros((0, 2), np.float32), np.array([0, 0], np.int32), 1, 1, 1, 8)
    assert got.accum.sum() == 0 and got.total == 0 and list(got.offsets) == [0, 0]
    # events 0 and 2 empty
    hits = generate_events(w).hits_xy[:300]
    off = np.array([0, 0, 300, 300], np.int32)
    o = Oracle.from_binning(bn, w.bz_tesla)
    acc, _ = o.vote(hits, off)
    ref = o.find_peaks(acc, 3)
    got = run_cuda(bn, w.bz_tesla, w.layers, hits, off, 3, 1, 3, ref.total + 1)
    assert np.array_equal(got.accum, acc) and np.array_equal(got.offsets, ref.offsets)
    h2c, nh, keep = o.assign_brute(hits, off, ref, 1, 3)
    assert np.array_equal(got.hit_to_cand, h2c) and np.array_equal(got.cand_nhits[:ref.total], nh)


def test_degenerate_hits():
    """Hit at the origin (r2 = 0 -> 1/0), hits far outside, denormal coordinates: no vote, no crash, same bits."""
    bn = HoughBinning(32, 16, 4)
    hits = np.array([[0.0, 0.0], [1e-30, -1e-30], [1e6, 1e6], [4.0, 0.0], [0.0, -110.0], [1e-42, 3.0]], np.float32)
    off = np.array([0, hits.shape[0]], np.int32)
    o = Oracle.from_binning(bn, 3.8)
    acc, _ = o.vote(hits, off)
    got = run_cuda(bn, 3.8, LAYERS_10, hits, off, 1, 1, 1, 64)
    assert np.array_equal(got.accum, acc)
    ref = o.find_peaks(acc, 1)
    assert got.total == ref.total and np.array_equal(got.records["j"], ref.records["j"])


@pytest.mark.parametrize("dtype", [ACC_I32, ACC_U16])
def test_capacity_overflow_and_zero_capacity(dtype):
    w = get_workload(1)
    bn = HoughBinning(256, 128, 64, accum_dtype=dtype)
    batch = generate_events(w)
    _compare_all(w, batch, binning=bn, capacity=100)          # fewer slots than peaks (S12)
    o = Oracle.from_binning(bn, w.bz_tesla)
    acc, _ = o.vote(batch.hits_xy)
    ref = o.find_peaks(acc, w.threshold)
    got = run_cuda(bn, w.bz_tesla, w.layers, batch.hits_xy, batch.event_offsets, w.threshold, 1, w.min_hits, 0)
    assert got.total == ref.total and (got.hit_to_cand == -1).all()


def test_plateaus_and_wraparound_via_constructed_hits():
    """Duplicated hits give multi-vote bins and equal-valued neighbours; phi0 near 0/2pi exercises the wrap."""
    bn = HoughBinning(64, 64, 1)
    base = np.concatenate([helix_hits(0.01, 0.3, 0.0, LAYERS_10, 3.8), helix_hits(6.27, -0.3, 0.0, LAYERS_10, 3.8),
                           helix_hits(3.1, 0.8, 0.0, LAYERS_10, 3.8)])
    hits = np.concatenate([base, base, base[::2]])
    off = np.array([0, hits.shape[0]], np.int32)
    o = Oracle.from_binning(bn, 3.8)
    acc, _ = o.vote(hits, off)
    ref = o.find_peaks(acc, 2)
    got = run_cuda(bn, 3.8, LAYERS_10, hits, off, 2, 2, 2, ref.total)
    assert np.array_equal(got.accum, acc) and got.total == ref.total
    for f in ("k", "i", "j", "votes"):
        assert np.array_equal(got.records[f], ref.records[f])
    h2c, nh, keep = o.assign_brute(hits, off, ref, 2, 2)
    assert np.array_equal(got.hit_to_cand, h2c) and np.array_equal(got.cand_keep[:ref.total], keep)


def test_hit_order_does_not_matter_and_vote_overwrites():
    w = get_workload(1)
    batch = generate_events(w)
    bn = w.binning
    a = run_cuda(bn, w.bz_tesla, w.layers, batch.hits_xy, batch.event_offsets, w.threshold, 1, w.min_hits, 4096)
    perm = np.random.default_rng(0).permutation(batch.n_hits)
    b = run_cuda(bn, w.bz_tesla, w.layers, batch.hits_xy[perm], batch.event_offsets, w.threshold, 1, w.min_hits, 4096)
    assert np.array_equal(a.accum, b.accum) and np.array_equal(a.records, b.records)
    assert np.array_equal(a.hit_to_cand[perm], b.hit_to_cand)


def test_invalid_arguments_are_rejected():
    from paper_1311_2769_b200 import HoughPlan, HoughError
    with pytest.raises(HoughError):
        HoughPlan(255, 128, 1)                      # n_phi % 4
    with pytest.raises(HoughError):
        HoughPlan(256, 128, 1, qpt_min=1.0, qpt_max=-1.0)
    plan = HoughPlan(64, 32, 1, max_hits=10, max_events=1)
    hits = torch.zeros((11, 2), dtype=torch.float32, device="cuda")
    off = torch.tensor([0, 11], dtype=torch.int32, device="cuda")
    with pytest.raises(HoughError):
        plan.vote(hits, off, plan.alloc_accum(1))   # n_hits > max_hits
    plan.close()


# ---- HOUGH_MODEL_LINE: straight displaced tracks, two-parameter space (phi0, d0) ----
def test_line_model_workload_bit_exact():
    w = get_workload(6)
    for fullscan, options in ((False, ()), (True, ()), (False, ("exact_walk",))):
        got, ref = _compare_all(w, generate_events(w), fullscan=fullscan, options=options)
        assert ref.total > 100


@pytest.mark.parametrize("shape,dtype,max_hits,drange,layers", [
    ((256, 128, 1), ACC_U16, None, (-20.0, 20.0), LAYERS_10),      # full-phi packed tile
    ((1024, 512, 1), ACC_I32, None, (-30.0, 10.0), LAYERS_10),     # phi slabs, asymmetric range
    ((256, 64, 1), ACC_I32, 70000, (0.0, 25.0), ()),               # 32-bit tile, one-sided range, no geometry
    ((100, 37, 1), ACC_U16, None, (-5.0, 5.0), LAYERS_10),         # odd sizes
])
def test_line_model_variants_bit_exact(shape, dtype, max_hits, drange, layers):
    bn = HoughBinning(shape[0], shape[1], 1, drange[0], drange[1], accum_dtype=dtype, model=1)
    hits, off = _mixed_hits(shape[0] + 7, 3000, LAYERS_10)
    o = Oracle.from_binning(bn, 0.0)
    acc, votes = o.vote(hits, off)
    got = run_vote(bn, 0.0, layers, hits, off, max_hits=max_hits)
    assert votes > 0 and np.array_equal(got.astype(np.int32), acc)
    thr = 3
    ref = o.find_peaks(acc, thr)
    cap = ref.total + 5
    res = run_cuda(bn, 0.0, layers, hits, off, thr, 1, 2, cap)
    assert res.total == ref.total and np.array_equal(res.offsets, ref.offsets)
    for f in ("event", "k", "i", "j", "votes"):
        assert np.array_equal(res.records[f], ref.records[f]), f
    assert_centroids_close(res.records, ref.records, bn)
    h2c, nh, keep = o.assign_indexed(hits, off, ref, 1, 2, capacity=cap)
    assert np.array_equal(res.hit_to_cand, h2c)
    assert np.array_equal(res.cand_nhits[:ref.total], nh) and np.array_equal(res.cand_keep[:ref.total], keep)


def test_line_model_rejects_a_d0_axis():
    from paper_1311_2769_b200 import HoughError, HoughPlan
    with pytest.raises(HoughError):
        HoughPlan(64, 32, 4, -10.0, 10.0, model=1)
