"""Thin ctypes binding of libhough_b200 (include/hough.h): argument marshalling only.

PyTorch supplies device memory and streams; every step of the path runs in the library's kernels.
There is no CPU fallback: a missing library or a failing call raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libhough_b200.so")

HOUGH_OK = 0
HOUGH_ACC_I32 = 0
HOUGH_ACC_U16 = 1
HOUGH_MODEL_HELIX = 0
HOUGH_MODEL_LINE = 1

CAND_DTYPE = np.dtype([("event", "<i4"), ("k", "<i4"), ("i", "<i4"), ("j", "<i4"), ("votes", "<i4"),
                       ("phi0", "<f4"), ("qpt", "<f4"), ("d0", "<f4")])


class HoughError(RuntimeError):
    pass


class hough_binning(C.Structure):
    _fields_ = [("n_phi", C.c_int32), ("n_qpt", C.c_int32), ("n_d0", C.c_int32),
                ("qpt_min", C.c_float), ("qpt_max", C.c_float), ("d0_min", C.c_float), ("d0_max", C.c_float),
                ("accum_dtype", C.c_int32), ("model", C.c_int32)]


class hough_geometry(C.Structure):
    _fields_ = [("bz_tesla", C.c_float), ("n_layers", C.c_int32), ("layer_radius_cm", C.POINTER(C.c_float))]


EXPORTS = ["hough_plan_create", "hough_plan_destroy", "hough_accum_bytes", "hough_vote", "hough_find_peaks",
           "hough_assign_hits", "hough_reassign_hits", "hough_event_run", "hough_vertex_vote", "hough_fit_circles", "hough_fit_circles_static", "hough_plan_set_option", "hough_pipeline_create", "hough_pipeline_destroy",
           "hough_pipeline_run_host", "hough_pipeline_set_option", "hough_window_table", "hough_microbench", "hough_kernel_launches", "hough_status_string",
           "hough_version"]

_lib = None


def load_library() -> C.CDLL:
    """Load libhough_b200.so (built in-tree by paper_1311_2769_b200.build).  Fails loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise HoughError(f"{LIB_PATH} not found: run `python -m paper_1311_2769_b200.build` "
                         "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    P, I = C.c_void_p, C.c_int32
    lib.hough_plan_create.restype = C.c_int
    lib.hough_plan_create.argtypes = [C.POINTER(hough_binning), C.POINTER(hough_geometry), I, I, C.POINTER(P)]
    lib.hough_plan_destroy.restype = C.c_int
    lib.hough_plan_destroy.argtypes = [P]
    lib.hough_accum_bytes.restype = C.c_size_t
    lib.hough_accum_bytes.argtypes = [P, I]
    lib.hough_vote.restype = C.c_int
    lib.hough_vote.argtypes = [P, P, I, P, I, P, P]
    lib.hough_find_peaks.restype = C.c_int
    lib.hough_find_peaks.argtypes = [P, P, I, I, P, I, P, P]
    lib.hough_assign_hits.restype = C.c_int
    lib.hough_assign_hits.argtypes = [P, P, I, P, I, P, P, I, I, I, P, P, P, P]
    lib.hough_event_run.restype = C.c_int
    lib.hough_event_run.argtypes = [P, P, I, P, P, I, P, I, P, I, I, P, P, P, P]
    lib.hough_reassign_hits.restype = C.c_int
    lib.hough_reassign_hits.argtypes = [P, P, I, P, I, P, P, I, I, I, P, P, P, P]
    lib.hough_vertex_vote.restype = C.c_int
    lib.hough_vertex_vote.argtypes = [P, P, P, I, I, P, C.c_float, I, C.c_float, P, P]
    lib.hough_fit_circles.restype = C.c_int
    lib.hough_fit_circles.argtypes = [P, P, I, P, P, P, I, I, P, P, P, P, P]
    lib.hough_fit_circles_static.restype = C.c_int
    lib.hough_fit_circles_static.argtypes = [I, C.c_float, P, I, P, P, P, I, I, P, P, P, P]
    lib.hough_plan_set_option.restype = C.c_int
    lib.hough_plan_set_option.argtypes = [P, C.c_char_p, I]
    lib.hough_pipeline_create.restype = C.c_int
    lib.hough_pipeline_create.argtypes = [C.POINTER(hough_binning), C.POINTER(hough_geometry), I, I, I, I, C.POINTER(P)]
    lib.hough_pipeline_destroy.restype = C.c_int
    lib.hough_pipeline_destroy.argtypes = [P]
    lib.hough_pipeline_set_option.restype = C.c_int
    lib.hough_pipeline_set_option.argtypes = [P, C.c_char_p, I]
    lib.hough_pipeline_run_host.restype = C.c_int
    lib.hough_pipeline_run_host.argtypes = [P, P, I, P, I, I, I, I, P, P, P, I, P, P, P]
    lib.hough_window_table.restype = C.c_int
    lib.hough_window_table.argtypes = [C.POINTER(hough_binning), C.POINTER(hough_geometry), C.POINTER(I), P, P, P]
    lib.hough_microbench.restype = C.c_int
    lib.hough_microbench.argtypes = [I, C.c_size_t, I, C.POINTER(C.c_double), P]
    lib.hough_kernel_launches.restype = C.c_int64
    lib.hough_kernel_launches.argtypes = []
    lib.hough_status_string.restype = C.c_char_p
    lib.hough_status_string.argtypes = [C.c_int]
    lib.hough_version.restype = C.c_char_p
    lib.hough_version.argtypes = []
    _lib = lib
    return lib


def _check(status: int, what: str):
    if status != HOUGH_OK:
        msg = load_library().hough_status_string(status).decode()
        raise HoughError(f"{what} failed: status {status} ({msg})")


def _stream_ptr(stream: Optional[torch.cuda.Stream]) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


def _dptr(t: Optional[torch.Tensor]) -> Optional[int]:
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous(), "device-resident contiguous tensor required"
    return t.data_ptr()


def make_structs(n_phi, n_qpt, n_d0, qpt_min, qpt_max, d0_min, d0_max, accum_dtype, bz_tesla, layers, model=0):
    b = hough_binning(n_phi, n_qpt, n_d0, qpt_min, qpt_max, d0_min, d0_max, accum_dtype, int(model))
    arr = (C.c_float * max(len(layers), 1))(*[float(r) for r in layers])
    g = hough_geometry(float(bz_tesla), len(layers), C.cast(arr, C.POINTER(C.c_float)))
    return b, g, arr


class HoughPlan:
    """hough_plan_create / hough_vote / hough_find_peaks / hough_assign_hits on torch CUDA tensors."""

    def __init__(self, n_phi: int, n_qpt: int, n_d0: int, qpt_min: float = -1.0, qpt_max: float = 1.0,
                 d0_min: float = -20.0, d0_max: float = 20.0, accum_dtype: int = HOUGH_ACC_I32,
                 bz_tesla: float = 3.8, layers: Sequence[float] = (), max_hits: int = 1 << 20,
                 max_events: int = 1, model: int = HOUGH_MODEL_HELIX):
        self.lib = load_library()
        if not torch.cuda.is_available():
            raise HoughError("no CUDA device: libhough_b200 has no CPU fallback")
        self.n_phi, self.n_qpt, self.n_d0 = int(n_phi), int(n_qpt), int(n_d0)
        self.accum_dtype = int(accum_dtype)
        self.max_hits, self.max_events = int(max_hits), int(max_events)
        b, g, self._keep = make_structs(n_phi, n_qpt, n_d0, qpt_min, qpt_max, d0_min, d0_max, accum_dtype,
                                        bz_tesla, layers, model)
        h = C.c_void_p()
        _check(self.lib.hough_plan_create(C.byref(b), C.byref(g), self.max_hits, self.max_events, C.byref(h)),
               "hough_plan_create")
        self._h = h

    @classmethod
    def from_workload(cls, w, max_hits: int, max_events: Optional[int] = None):
        bn = w.binning
        return cls(bn.n_phi, bn.n_qpt, bn.n_d0, bn.qpt_min, bn.qpt_max, bn.d0_min, bn.d0_max, bn.accum_dtype,
                   w.bz_tesla, w.layers, max_hits=max_hits, max_events=max_events or w.n_events,
                   model=getattr(bn, "model", 0))

    def close(self):
        if getattr(self, "_h", None):
            self.lib.hough_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- helpers ---------------------------------------------------------------------------------
    @property
    def torch_accum_dtype(self):
        return torch.int32 if self.accum_dtype == HOUGH_ACC_I32 else torch.uint16

    def accum_bytes(self, n_events: int) -> int:
        return int(self.lib.hough_accum_bytes(self._h, n_events))

    def alloc_accum(self, n_events: int, device="cuda") -> torch.Tensor:
        return torch.empty((n_events, self.n_d0, self.n_phi, self.n_qpt), dtype=self.torch_accum_dtype, device=device)

    def set_option(self, key: str, value: int):
        _check(self.lib.hough_plan_set_option(self._h, key.encode(), int(value)), "hough_plan_set_option")

    # -- the four calls --------------------------------------------------------------------------
    def vote(self, hits_xy: torch.Tensor, event_offsets: torch.Tensor, accum: torch.Tensor, stream=None):
        n_hits = int(hits_xy.shape[0])
        n_events = int(event_offsets.shape[0]) - 1
        assert hits_xy.dtype == torch.float32 and event_offsets.dtype == torch.int32
        _check(self.lib.hough_vote(self._h, _dptr(hits_xy), n_hits, _dptr(event_offsets), n_events, _dptr(accum),
                                   _stream_ptr(stream)), "hough_vote")

    def find_peaks(self, accum: torch.Tensor, n_events: int, threshold: int, cands: Optional[torch.Tensor],
                   capacity: int, cand_offsets: torch.Tensor, stream=None):
        """cands: uint8 tensor [capacity, 32] (hough_candidate records) or None when capacity == 0."""
        assert cand_offsets.dtype == torch.int32 and cand_offsets.numel() >= n_events + 1
        _check(self.lib.hough_find_peaks(self._h, _dptr(accum), n_events, int(threshold), _dptr(cands), int(capacity),
                                         _dptr(cand_offsets), _stream_ptr(stream)), "hough_find_peaks")

    def assign_hits(self, hits_xy, event_offsets, cands, cand_offsets, capacity, assoc_dj, min_hits, hit_to_cand,
                    cand_nhits, cand_keep, stream=None):
        n_hits = int(hits_xy.shape[0])
        n_events = int(event_offsets.shape[0]) - 1
        _check(self.lib.hough_assign_hits(self._h, _dptr(hits_xy), n_hits, _dptr(event_offsets), n_events,
                                          _dptr(cands), _dptr(cand_offsets), int(capacity), int(assoc_dj),
                                          int(min_hits), _dptr(hit_to_cand), _dptr(cand_nhits), _dptr(cand_keep),
                                          _stream_ptr(stream)), "hough_assign_hits")

    def event_run(self, hits_xy, event_offsets, accum, threshold, cands, capacity, cand_offsets, assoc_dj, min_hits,
                  hit_to_cand, cand_nhits, cand_keep, stream=None):
        """include/hough.h hough_event_run: vote + find_peaks + assign_hits of ONE event, in one launch when it fits."""
        assert int(event_offsets.shape[0]) == 2
        _check(self.lib.hough_event_run(self._h, _dptr(hits_xy), int(hits_xy.shape[0]), _dptr(event_offsets), _dptr(accum),
                                        int(threshold), _dptr(cands), int(capacity), _dptr(cand_offsets), int(assoc_dj),
                                        int(min_hits), _dptr(hit_to_cand), _dptr(cand_nhits), _dptr(cand_keep),
                                        _stream_ptr(stream)), "hough_event_run")

    def reassign_hits(self, hits_xy, event_offsets, cands, cand_offsets, capacity, assoc_dj, max_rounds, hit_to_cand,
                      cand_nhits, cand_keep, stream=None):
        n_hits = int(hits_xy.shape[0])
        n_events = int(event_offsets.shape[0]) - 1
        _check(self.lib.hough_reassign_hits(self._h, _dptr(hits_xy), n_hits, _dptr(event_offsets), n_events,
                                            _dptr(cands), _dptr(cand_offsets), int(capacity), int(assoc_dj),
                                            int(max_rounds), _dptr(hit_to_cand), _dptr(cand_nhits), _dptr(cand_keep),
                                            _stream_ptr(stream)), "hough_reassign_hits")


class HoughPipeline:
    """hough_pipeline_create / hough_pipeline_run_host: the batched multi-event path over HOST buffers (pinned
    torch CPU tensors in and out; event tiles on n_streams CUDA streams, each tile's sequence replayed as a CUDA graph)."""

    def __init__(self, n_phi, n_qpt, n_d0, qpt_min=-1.0, qpt_max=1.0, d0_min=-20.0, d0_max=20.0,
                 accum_dtype=HOUGH_ACC_I32, bz_tesla=3.8, layers=(), tile_events=64, max_hits_per_tile=1 << 20,
                 tile_cand_capacity=1 << 20, n_streams=4, model=HOUGH_MODEL_HELIX):
        self.lib = load_library()
        if not torch.cuda.is_available():
            raise HoughError("no CUDA device: libhough_b200 has no CPU fallback")
        b, g, self._keep = make_structs(n_phi, n_qpt, n_d0, qpt_min, qpt_max, d0_min, d0_max, accum_dtype,
                                        bz_tesla, layers, model)
        h = C.c_void_p()
        _check(self.lib.hough_pipeline_create(C.byref(b), C.byref(g), int(tile_events), int(max_hits_per_tile),
                                              int(tile_cand_capacity), int(n_streams), C.byref(h)),
               "hough_pipeline_create")
        self._h = h

    @classmethod
    def from_workload(cls, w, tile_events, max_hits_per_tile, tile_cand_capacity, n_streams=4):
        bn = w.binning
        return cls(bn.n_phi, bn.n_qpt, bn.n_d0, bn.qpt_min, bn.qpt_max, bn.d0_min, bn.d0_max, bn.accum_dtype,
                   w.bz_tesla, w.layers, tile_events, max_hits_per_tile, tile_cand_capacity, n_streams,
                   model=getattr(bn, "model", 0))

    def close(self):
        if getattr(self, "_h", None):
            self.lib.hough_pipeline_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_option(self, key: str, value: int):
        _check(self.lib.hough_pipeline_set_option(self._h, key.encode(), int(value)), "hough_pipeline_set_option")

    def run_host(self, hits_xy, event_offsets, threshold, assoc_dj, min_hits, hit_to_cand, cand_offsets, cands,
                 cand_capacity, cand_nhits, cand_keep) -> bool:
        """All tensors are HOST (CPU, ideally pinned) and contiguous: hits_xy float32 [n_hits, 2], event_offsets int32
        [n_events + 1]; outputs hit_to_cand int32 [n_hits], cand_offsets int32 [n_events + 1], cands uint8
        [cand_capacity, 32], cand_nhits int32 [cand_capacity], cand_keep uint8 [cand_capacity].  Blocks until the
        results are in the host buffers.  Returns True if a candidate capacity was exceeded."""
        for t in (hits_xy, event_offsets, hit_to_cand, cand_offsets, cands, cand_nhits, cand_keep):
            assert (not t.is_cuda) and t.is_contiguous(), "host-resident contiguous tensor required"
        assert hits_xy.dtype == torch.float32 and event_offsets.dtype == torch.int32
        n_hits, n_events = int(hits_xy.shape[0]), int(event_offsets.shape[0]) - 1
        over = C.c_int32(0)
        _check(self.lib.hough_pipeline_run_host(self._h, hits_xy.data_ptr(), n_hits, event_offsets.data_ptr(), n_events,
                                                int(threshold), int(assoc_dj), int(min_hits), hit_to_cand.data_ptr(),
                                                cand_offsets.data_ptr(), cands.data_ptr(), int(cand_capacity),
                                                cand_nhits.data_ptr(), cand_keep.data_ptr(), C.byref(over)),
               "hough_pipeline_run_host")
        return bool(over.value)


def hough_vertex_vote(plan: "HoughPlan", cands, cand_offsets, n_events, capacity, cand_keep, d0_abs_min, n_r, r_max,
                      vertex_accum, stream=None):
    """include/hough.h hough_vertex_vote: vertex_accum int32 [n_events, n_phi, n_r] on the device (overwritten)."""
    assert vertex_accum.dtype == torch.int32 and vertex_accum.numel() >= n_events * plan.n_phi * n_r
    _check(plan.lib.hough_vertex_vote(plan._h, _dptr(cands), _dptr(cand_offsets), int(n_events), int(capacity),
                                      _dptr(cand_keep), float(d0_abs_min), int(n_r), float(r_max), _dptr(vertex_accum),
                                      _stream_ptr(stream)), "hough_vertex_vote")


def hough_fit_circles(plan: "HoughPlan", hits_xy, hit_to_cand, cands, cand_offsets, n_events, capacity, cand_keep, work, fit,
                      n_fit, stream=None):
    """include/hough.h hough_fit_circles: work float64 [capacity, 9], fit float64 [capacity, 4], n_fit int32 [capacity]."""
    assert capacity == 0 or (work.dtype == torch.float64 and fit.dtype == torch.float64 and n_fit.dtype == torch.int32)
    _check(plan.lib.hough_fit_circles(plan._h, _dptr(hits_xy), int(hits_xy.shape[0]), _dptr(hit_to_cand), _dptr(cands),
                                      _dptr(cand_offsets), int(n_events), int(capacity), _dptr(cand_keep), _dptr(work),
                                      _dptr(fit), _dptr(n_fit), _stream_ptr(stream)), "hough_fit_circles")


FIT_STATIC_MAX_CANDIDATES = 65536   # include/hough.h HOUGH_FIT_STATIC_MAX_CANDIDATES


def hough_fit_circles_static(n_phi, bz_tesla, hits_xy, hit_to_cand, cands, cand_offsets, n_events, capacity, cand_keep, fit,
                             n_fit, stream=None):
    """include/hough.h hough_fit_circles_static: the circle fit for callers that may not allocate device memory (a
    fixed-latency event loop, a plug-in whose host application owns all GPU memory).  No plan and no work buffer: the moment
    sums use a fixed per-GPU array inside the library, so capacity <= FIT_STATIC_MAX_CANDIDATES, calls on one GPU must not
    overlap, and the first call per device (address look-up) belongs to start-up.  fit float64 [capacity, 4], n_fit int32."""
    assert capacity == 0 or (fit.dtype == torch.float64 and n_fit.dtype == torch.int32)
    _check(load_library().hough_fit_circles_static(int(n_phi), float(bz_tesla), _dptr(hits_xy), int(hits_xy.shape[0]),
                                                   _dptr(hit_to_cand), _dptr(cands), _dptr(cand_offsets), int(n_events),
                                                   int(capacity), _dptr(cand_keep), _dptr(fit), _dptr(n_fit),
                                                   _stream_ptr(stream)), "hough_fit_circles_static")


def window_table(n_phi, n_qpt, n_d0, qpt_min=-1.0, qpt_max=1.0, d0_min=-20.0, d0_max=20.0, bz_tesla=3.8, layers=(),
                 model=0):
    """hough_window_table (host only): (edge_r2 [n_class], lo_off [n_class, n_d0], steps [n_class, n_d0])."""
    lib = load_library()
    b, g, _keep = make_structs(n_phi, n_qpt, n_d0, qpt_min, qpt_max, d0_min, d0_max, HOUGH_ACC_I32, bz_tesla, layers, model)
    n = C.c_int32(0)
    edge = np.zeros(256, np.float32)
    lo = np.zeros(256 * n_d0, np.float32)
    steps = np.zeros(256 * n_d0, np.int32)
    _check(lib.hough_window_table(C.byref(b), C.byref(g), C.byref(n), edge.ctypes.data_as(C.c_void_p),
                                  lo.ctypes.data_as(C.c_void_p), steps.ctypes.data_as(C.c_void_p)),
           "hough_window_table")
    nc = int(n.value)
    return edge[:nc].copy(), lo[:nc * n_d0].reshape(nc, n_d0).copy(), steps[:nc * n_d0].reshape(nc, n_d0).copy()


def alloc_candidates(capacity: int, device="cuda") -> torch.Tensor:
    return torch.empty((max(int(capacity), 1), 32), dtype=torch.uint8, device=device)


def candidates_to_numpy(cands: torch.Tensor, n: int) -> np.ndarray:
    return cands[:n].cpu().numpy().view(CAND_DTYPE).reshape(-1)


def microbench(kind: int, region_bytes: int = 0, iters: int = 5, stream=None) -> float:
    lib = load_library()
    out = C.c_double(0.0)
    _check(lib.hough_microbench(int(kind), int(region_bytes), int(iters), C.byref(out), _stream_ptr(stream)),
           "hough_microbench")
    return float(out.value)


def kernel_launches() -> int:
    return int(load_library().hough_kernel_launches())


def version() -> str:
    return load_library().hough_version().decode()
