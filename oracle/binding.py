"""ctypes/numpy front end of oracle/hough_oracle.cpp (test infrastructure only)."""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass
from typing import Optional, Tuple

import numpy as np

from . import build as _build

CAND_DTYPE = np.dtype([("event", "<i4"), ("k", "<i4"), ("i", "<i4"), ("j", "<i4"), ("votes", "<i4"),
                       ("phi0", "<f4"), ("qpt", "<f4"), ("d0", "<f4")])
assert CAND_DTYPE.itemsize == 32


class _Binning(C.Structure):
    _fields_ = [("n_phi", C.c_int32), ("n_qpt", C.c_int32), ("n_d0", C.c_int32),
                ("qpt_min", C.c_float), ("qpt_max", C.c_float), ("d0_min", C.c_float), ("d0_max", C.c_float),
                ("model", C.c_int32)]


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(_build.build())
        P = C.c_void_p
        lib.orc_tables.restype = C.c_int
        lib.orc_tables.argtypes = [C.POINTER(_Binning), C.c_float, P, P, P, P, P, P]
        lib.orc_vote.restype = C.c_longlong
        lib.orc_vote.argtypes = [C.POINTER(_Binning), C.c_float, P, C.c_int32, P, C.c_int32, C.c_int32, C.c_int32, P]
        lib.orc_vote_columns.restype = C.c_int
        lib.orc_vote_columns.argtypes = [C.POINTER(_Binning), C.c_float, P, C.c_int32, P, C.c_int32, P, C.c_int32, P]
        lib.orc_votes_per_hit.restype = C.c_int
        lib.orc_votes_per_hit.argtypes = [C.POINTER(_Binning), C.c_float, P, C.c_int32, P]
        lib.orc_find_peaks.restype = C.c_longlong
        lib.orc_find_peaks.argtypes = [C.POINTER(_Binning), P, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32,
                                       C.c_int32, P, C.c_longlong, P]
        for name in ("orc_assign_brute", "orc_assign_indexed"):
            f = getattr(lib, name)
            f.restype = C.c_int
            f.argtypes = [C.POINTER(_Binning), C.c_float, P, C.c_int32, P, C.c_int32, P, P, C.c_longlong,
                          C.c_int32, C.c_int32, C.c_int32, P, P, P]
        lib.orc_assign_rounds.restype = C.c_int
        lib.orc_assign_rounds.argtypes = [C.POINTER(_Binning), C.c_float, P, C.c_int32, P, C.c_int32, P, P, C.c_longlong,
                                          C.c_int32, C.c_int32, C.c_int32, P, P, P]
        lib.orc_vertex_vote.restype = C.c_longlong
        lib.orc_vertex_vote.argtypes = [C.POINTER(_Binning), C.c_float, P, P, C.c_int32, C.c_longlong, P, C.c_float, C.c_int32,
                                        C.c_float, P]
        lib.orc_fit_circles.restype = C.c_int
        lib.orc_fit_circles.argtypes = [C.POINTER(_Binning), C.c_float, P, C.c_int32, P, P, C.c_longlong, P, P, P]
        _lib = lib
    return _lib


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


@dataclass
class OracleCandidates:
    records: np.ndarray      # CAND_DTYPE [min(total, capacity)]
    offsets: np.ndarray      # int32 [n_events + 1], true counts
    total: int


class Oracle:
    """One binning + field; methods mirror the C functions."""

    def __init__(self, n_phi, n_qpt, n_d0, qpt_min=-1.0, qpt_max=1.0, d0_min=-20.0, d0_max=20.0, bz_tesla=3.8, model=0):
        """model 0: curved tracks, axis j = q/pT (D3); model 1: straight displaced tracks, axis j = d0 in cm over
        [qpt_min, qpt_max) (D3L; n_d0 must be 1, the field is ignored)."""
        self.b = _Binning(n_phi, n_qpt, n_d0, qpt_min, qpt_max, d0_min, d0_max, int(model))
        self.model = int(model)
        self.bz = float(bz_tesla)
        self.n_phi, self.n_qpt, self.n_d0 = int(n_phi), int(n_qpt), int(n_d0)
        self.lib = _load()

    @classmethod
    def from_binning(cls, binning, bz_tesla=3.8):
        return cls(binning.n_phi, binning.n_qpt, binning.n_d0, binning.qpt_min, binning.qpt_max,
                   binning.d0_min, binning.d0_max, bz_tesla, getattr(binning, "model", 0))

    @staticmethod
    def _hits(hits_xy):
        h = np.ascontiguousarray(hits_xy, dtype=np.float32).reshape(-1, 2)
        return h

    @staticmethod
    def _offsets(event_offsets, n_hits):
        if event_offsets is None:
            return np.array([0, n_hits], np.int32)
        return np.ascontiguousarray(event_offsets, dtype=np.int32)

    def tables(self):
        cosT = np.zeros(self.n_phi, np.float32)
        sinT = np.zeros(self.n_phi, np.float32)
        d0c = np.zeros(self.n_d0, np.float32)
        td0 = np.zeros(self.n_d0, np.float32)
        d0sq = np.zeros(self.n_d0, np.float32)
        consts = np.zeros(3, np.float32)
        rc = self.lib.orc_tables(C.byref(self.b), self.bz, _ptr(cosT), _ptr(sinT), _ptr(d0c), _ptr(td0),
                                 _ptr(d0sq), _ptr(consts))
        assert rc == 0
        return dict(cosT=cosT, sinT=sinT, d0c=d0c, td0=td0, d0sq=d0sq, A_f=consts[0], qmin=consts[1],
                    inv_wq=consts[2])

    def vote(self, hits_xy, event_offsets=None, k_range: Optional[Tuple[int, int]] = None):
        """int32 accumulator [n_events, k_hi-k_lo, n_phi, n_qpt] and the number of votes."""
        h = self._hits(hits_xy)
        off = self._offsets(event_offsets, h.shape[0])
        n_ev = off.shape[0] - 1
        k_lo, k_hi = k_range if k_range is not None else (0, self.n_d0)
        acc = np.empty((n_ev, k_hi - k_lo, self.n_phi, self.n_qpt), np.int32)
        votes = self.lib.orc_vote(C.byref(self.b), self.bz, _ptr(h), h.shape[0], _ptr(off), n_ev, k_lo, k_hi, _ptr(acc))
        assert votes >= 0, "orc_vote: bad arguments"
        return acc, int(votes)

    def vote_columns(self, hits_xy, event_offsets, cols):
        h = self._hits(hits_xy)
        off = self._offsets(event_offsets, h.shape[0])
        cols = np.ascontiguousarray(cols, dtype=np.int32).reshape(-1, 3)
        rows = np.empty((cols.shape[0], self.n_qpt), np.int32)
        rc = self.lib.orc_vote_columns(C.byref(self.b), self.bz, _ptr(h), h.shape[0], _ptr(off), off.shape[0] - 1,
                                       _ptr(cols), cols.shape[0], _ptr(rows))
        assert rc == 0
        return rows

    def votes_per_hit(self, hits_xy):
        h = self._hits(hits_xy)
        out = np.empty(h.shape[0], np.int32)
        rc = self.lib.orc_votes_per_hit(C.byref(self.b), self.bz, _ptr(h), h.shape[0], _ptr(out))
        assert rc == 0
        return out

    def find_peaks(self, accum, threshold, capacity=None, k_range=None, k_out=None) -> OracleCandidates:
        acc = np.ascontiguousarray(accum, dtype=np.int32)
        assert acc.ndim == 4
        n_ev = acc.shape[0]
        k_lo, k_hi = k_range if k_range is not None else (0, self.n_d0)
        ko_lo, ko_hi = k_out if k_out is not None else (k_lo, k_hi)
        assert acc.shape[1:] == (k_hi - k_lo, self.n_phi, self.n_qpt)
        off = np.zeros(n_ev + 1, np.int32)
        if capacity is None:     # count first, then fill
            total = self.lib.orc_find_peaks(C.byref(self.b), _ptr(acc), n_ev, k_lo, k_hi, ko_lo, ko_hi,
                                            int(threshold), None, 0, _ptr(off))
            assert total >= 0, "orc_find_peaks: bad arguments"
            capacity = int(total)
        rec = np.zeros(int(capacity), CAND_DTYPE)
        total = self.lib.orc_find_peaks(C.byref(self.b), _ptr(acc), n_ev, k_lo, k_hi, ko_lo, ko_hi, int(threshold),
                                        _ptr(rec), int(capacity), _ptr(off))
        assert total >= 0, "orc_find_peaks: bad arguments"
        return OracleCandidates(rec[:min(int(total), int(capacity))], off, int(total))

    def _assign(self, fn, hits_xy, event_offsets, cands: OracleCandidates, assoc_dj, min_hits, apply_dedup,
                capacity=None):
        h = self._hits(hits_xy)
        off = self._offsets(event_offsets, h.shape[0])
        rec = np.ascontiguousarray(cands.records)
        cap = int(rec.shape[0]) if capacity is None else int(capacity)
        n_c = min(cap, int(cands.offsets[-1]))
        h2c = np.full(h.shape[0], -2, np.int32)
        nh = np.zeros(max(n_c, 1), np.int32)
        keep = np.zeros(max(n_c, 1), np.uint8)
        rc = fn(C.byref(self.b), self.bz, _ptr(h), h.shape[0], _ptr(off), off.shape[0] - 1, _ptr(rec),
                _ptr(np.ascontiguousarray(cands.offsets, dtype=np.int32)), cap, int(assoc_dj), int(min_hits),
                int(apply_dedup), _ptr(h2c), _ptr(nh), _ptr(keep))
        assert rc == 0
        return h2c, nh[:n_c], keep[:n_c]

    def vertex_vote(self, cands: "OracleCandidates", keep, d_abs_min: float, n_r: int, r_max: float, capacity=None):
        """orc_vertex_vote (D10): int32 [n_events, n_phi, n_r] vertex accumulator (Phi_v x R_v) and the number of votes."""
        rec = np.ascontiguousarray(cands.records)
        off = np.ascontiguousarray(cands.offsets, dtype=np.int32)
        cap = int(rec.shape[0]) if capacity is None else int(capacity)
        keep = None if keep is None else np.ascontiguousarray(keep, dtype=np.uint8)
        vacc = np.empty((off.shape[0] - 1, self.n_phi, int(n_r)), np.int32)
        votes = self.lib.orc_vertex_vote(C.byref(self.b), self.bz, _ptr(rec), _ptr(off), off.shape[0] - 1, cap, _ptr(keep),
                                         float(d_abs_min), int(n_r), float(r_max), _ptr(vacc))
        assert votes >= 0, "orc_vertex_vote: bad arguments"
        return vacc, int(votes)

    def fit_circles(self, hits_xy, hit_to_cand, cands: "OracleCandidates", keep=None):
        """orc_fit_circles (D11): float64 [n_cands, 4] = {phi0, qpt, d0, R} and int32 [n_cands] hits used (< 0: fit not ok)."""
        h = self._hits(hits_xy)
        rec = np.ascontiguousarray(cands.records)
        h2c = np.ascontiguousarray(hit_to_cand, dtype=np.int32)
        keep = None if keep is None else np.ascontiguousarray(keep, dtype=np.uint8)
        fit = np.zeros((max(len(rec), 1), 4), np.float64)
        nfit = np.zeros(max(len(rec), 1), np.int32)
        rc = self.lib.orc_fit_circles(C.byref(self.b), self.bz, _ptr(h), h.shape[0], _ptr(h2c), _ptr(rec), len(rec), _ptr(keep),
                                      _ptr(fit), _ptr(nfit))
        assert rc == 0
        return fit[:len(rec)], nfit[:len(rec)]

    def assign_rounds(self, hits_xy, event_offsets, cands, assoc_dj=1, min_hits=0, max_rounds=8, capacity=None):
        """orc_assign_rounds (D12): (hit_to_cand, cand_nhits, cand_keep, rounds run)."""
        h = self._hits(hits_xy)
        off = self._offsets(event_offsets, h.shape[0])
        rec = np.ascontiguousarray(cands.records)
        cap = int(rec.shape[0]) if capacity is None else int(capacity)
        n_c = min(cap, int(cands.offsets[-1]))
        h2c = np.full(h.shape[0], -2, np.int32)
        nh = np.zeros(max(n_c, 1), np.int32)
        keep = np.zeros(max(n_c, 1), np.uint8)
        rounds = self.lib.orc_assign_rounds(C.byref(self.b), self.bz, _ptr(h), h.shape[0], _ptr(off), off.shape[0] - 1,
                                            _ptr(rec), _ptr(np.ascontiguousarray(cands.offsets, dtype=np.int32)), cap,
                                            int(assoc_dj), int(min_hits), int(max_rounds), _ptr(h2c), _ptr(nh), _ptr(keep))
        assert rounds >= 1, "orc_assign_rounds: bad arguments"
        return h2c, nh[:n_c], keep[:n_c], int(rounds)

    def assign_brute(self, hits_xy, event_offsets, cands, assoc_dj=1, min_hits=0, apply_dedup=True, capacity=None):
        return self._assign(self.lib.orc_assign_brute, hits_xy, event_offsets, cands, assoc_dj, min_hits,
                            apply_dedup, capacity)

    def assign_indexed(self, hits_xy, event_offsets, cands, assoc_dj=1, min_hits=0, apply_dedup=True, capacity=None):
        return self._assign(self.lib.orc_assign_indexed, hits_xy, event_offsets, cands, assoc_dj, min_hits,
                            apply_dedup, capacity)
