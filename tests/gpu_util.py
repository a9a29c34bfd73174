"""Helpers shared by the -m gpu parity tests: run the CUDA path through the C ABI, run the oracle."""
from __future__ import annotations

import os
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass

import numpy as np
import torch

from oracle import Oracle
from paper_1311_2769_b200 import (HoughPlan, alloc_candidates, candidates_to_numpy)


@dataclass
class CudaResult:
    accum: np.ndarray
    records: np.ndarray
    offsets: np.ndarray
    total: int
    hit_to_cand: np.ndarray
    cand_nhits: np.ndarray
    cand_keep: np.ndarray


def run_cuda(binning, bz, layers, hits_xy, event_offsets, threshold, assoc_dj, min_hits, capacity,
             fullscan=False, want_accum=True, plan=None, options=()) -> CudaResult:
    n_hits = int(hits_xy.shape[0])
    n_events = int(event_offsets.shape[0] - 1)
    own = plan is None
    if own:
        plan = HoughPlan(binning.n_phi, binning.n_qpt, binning.n_d0, binning.qpt_min, binning.qpt_max, binning.d0_min,
                         binning.d0_max, binning.accum_dtype, bz, layers, max_hits=max(n_hits, 1),
                         max_events=max(n_events, 1), model=getattr(binning, "model", 0))
    if fullscan:
        plan.set_option("fullscan", 1)
    for key in options:
        plan.set_option(key, 1)
    dev = "cuda"
    d_hits = torch.from_numpy(np.ascontiguousarray(hits_xy, np.float32).reshape(-1, 2)).to(dev)
    if n_hits == 0:
        d_hits = torch.zeros((1, 2), dtype=torch.float32, device=dev)[:0]
    d_off = torch.from_numpy(np.ascontiguousarray(event_offsets, np.int32)).to(dev)
    accum = plan.alloc_accum(n_events)
    accum.fill_(7)                                   # hough_vote must overwrite (S8)
    cands = alloc_candidates(capacity)
    cand_off = torch.full((n_events + 1,), -5, dtype=torch.int32, device=dev)
    h2c = torch.full((max(n_hits, 1),), -7, dtype=torch.int32, device=dev)
    nh = torch.full((max(capacity, 1),), -3, dtype=torch.int32, device=dev)
    keep = torch.full((max(capacity, 1),), 9, dtype=torch.uint8, device=dev)
    plan.vote(d_hits, d_off, accum)
    plan.find_peaks(accum, n_events, threshold, cands if capacity > 0 else None, capacity, cand_off)
    plan.assign_hits(d_hits, d_off, cands if capacity > 0 else None, cand_off, capacity, assoc_dj, min_hits,
                     h2c, nh if capacity > 0 else None, keep if capacity > 0 else None)
    torch.cuda.synchronize()
    off = cand_off.cpu().numpy()
    total = int(off[-1])
    n_c = min(total, capacity)
    res = CudaResult(accum.cpu().numpy() if want_accum else None, candidates_to_numpy(cands, n_c), off, total,
                     h2c[:n_hits].cpu().numpy(), nh[:capacity].cpu().numpy(), keep[:capacity].cpu().numpy())
    if own:
        plan.close()
    return res


def n_threads() -> int:
    return max(1, min(32, (os.cpu_count() or 2) - 1))


def oracle_vote_parallel(o: Oracle, hits_xy, event_offsets):
    """Full oracle accumulator computed as independent d0 slabs on several host threads (the oracle itself
    stays single-threaded; slabs are disjoint parts of the same definition)."""
    nd = o.n_d0
    nt = min(n_threads(), nd)
    if nt <= 1:
        return o.vote(hits_xy, event_offsets)
    bounds = np.linspace(0, nd, nt + 1).astype(int)
    slabs = [(int(bounds[t]), int(bounds[t + 1])) for t in range(nt) if bounds[t + 1] > bounds[t]]
    with ThreadPoolExecutor(len(slabs)) as ex:
        parts = list(ex.map(lambda kr: o.vote(hits_xy, event_offsets, k_range=kr), slabs))
    acc = np.concatenate([p[0] for p in parts], axis=1)
    return acc, sum(p[1] for p in parts)


def oracle_peaks_parallel(o: Oracle, acc, threshold):
    """Oracle peak list over the full volume, found slab by slab (each slab sees its neighbour slices)."""
    from oracle import OracleCandidates
    nd = o.n_d0
    nt = min(n_threads(), nd)
    n_ev = acc.shape[0]
    if nt <= 1 or n_ev != 1:
        return o.find_peaks(acc, threshold)
    bounds = np.linspace(0, nd, nt + 1).astype(int)

    def work(t):
        ko = (int(bounds[t]), int(bounds[t + 1]))
        kr = (max(0, ko[0] - 1), min(nd, ko[1] + 1))
        return o.find_peaks(np.ascontiguousarray(acc[:, kr[0]:kr[1]]), threshold, k_range=kr, k_out=ko)

    with ThreadPoolExecutor(nt) as ex:
        parts = list(ex.map(work, [t for t in range(nt) if bounds[t + 1] > bounds[t]]))
    rec = np.concatenate([p.records for p in parts])
    total = sum(p.total for p in parts)
    return OracleCandidates(rec, np.array([0, total], np.int32), total)


def assert_centroids_close(got, ref, binning):
    """B:L5 'peak-centroid track parameters must agree within 1e-5 relative'; floor = bin width (S13)."""
    import math
    for name, width in (("qpt", (binning.qpt_max - binning.qpt_min) / binning.n_qpt),
                        ("phi0", 2 * math.pi / binning.n_phi),
                        ("d0", (binning.d0_max - binning.d0_min) / binning.n_d0)):
        g = got[name].astype(np.float64)
        r = ref[name].astype(np.float64)
        tol = 1e-5 * np.maximum(np.abs(r), width)
        assert np.all(np.abs(g - r) <= tol), name


def run_vote(binning, bz, layers, hits_xy, event_offsets, max_hits=None, misalign=False, fullscan=False, options=()):
    """hough_vote alone -> accumulator as numpy.  misalign: the hit pointer is 8- but not 16-byte aligned."""
    n_hits = int(hits_xy.shape[0])
    n_events = int(event_offsets.shape[0] - 1)
    plan = HoughPlan(binning.n_phi, binning.n_qpt, binning.n_d0, binning.qpt_min, binning.qpt_max, binning.d0_min,
                     binning.d0_max, binning.accum_dtype, bz, layers, max_hits=max_hits or max(n_hits, 1),
                     max_events=max(n_events, 1), model=getattr(binning, "model", 0))
    if fullscan:
        plan.set_option("fullscan", 1)
    for key in options:
        plan.set_option(key, 1)
    buf = torch.zeros((n_hits + 2, 2), dtype=torch.float32, device="cuda")
    assert buf.data_ptr() % 16 == 0
    first = 1 if misalign else 0
    d_hits = buf[first:first + n_hits]
    d_hits.copy_(torch.from_numpy(np.ascontiguousarray(hits_xy, np.float32).reshape(-1, 2)))
    d_off = torch.from_numpy(np.ascontiguousarray(event_offsets, np.int32)).cuda()
    accum = plan.alloc_accum(n_events)
    accum.fill_(3)
    plan.vote(d_hits, d_off, accum)
    torch.cuda.synchronize()
    out = accum.cpu().numpy()
    plan.close()
    return out


def run_assign(binning, bz, layers, hits_xy, event_offsets, records, cand_offsets, capacity, assoc_dj, min_hits,
               max_hits=None, fullscan=False, options=()):
    """hough_assign_hits alone on a caller-made candidate list (CAND_DTYPE records, int32 offsets)."""
    n_hits = int(hits_xy.shape[0])
    n_events = int(event_offsets.shape[0] - 1)
    plan = HoughPlan(binning.n_phi, binning.n_qpt, binning.n_d0, binning.qpt_min, binning.qpt_max, binning.d0_min,
                     binning.d0_max, binning.accum_dtype, bz, layers, max_hits=max_hits or max(n_hits, 1),
                     max_events=max(n_events, 1), model=getattr(binning, "model", 0))
    if fullscan:
        plan.set_option("fullscan", 1)
    for key in options:
        plan.set_option(key, 1)
    d_hits = torch.from_numpy(np.ascontiguousarray(hits_xy, np.float32).reshape(-1, 2)).cuda()
    d_off = torch.from_numpy(np.ascontiguousarray(event_offsets, np.int32)).cuda()
    cands = alloc_candidates(capacity)
    n_c = min(capacity, len(records))
    if n_c:
        cands[:n_c].copy_(torch.from_numpy(np.ascontiguousarray(records[:n_c]).view(np.uint8).reshape(n_c, 32)))
    d_coff = torch.from_numpy(np.ascontiguousarray(cand_offsets, np.int32)).cuda()
    h2c = torch.full((max(n_hits, 1),), -7, dtype=torch.int32, device="cuda")
    nh = torch.full((max(capacity, 1),), -3, dtype=torch.int32, device="cuda")
    keep = torch.full((max(capacity, 1),), 9, dtype=torch.uint8, device="cuda")
    plan.assign_hits(d_hits, d_off, cands, d_coff, capacity, assoc_dj, min_hits, h2c, nh, keep)
    torch.cuda.synchronize()
    out = h2c[:n_hits].cpu().numpy(), nh[:capacity].cpu().numpy(), keep[:capacity].cpu().numpy()
    plan.close()
    return out
