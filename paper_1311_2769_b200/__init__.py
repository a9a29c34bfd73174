"""paper_1311_2769_b200 -- B200-native Hough-transform track finding (arXiv 1311.2769).

The product is `libhough_b200.so` (CUDA, sm_100a; C ABI in include/hough.h).  This package is its thin Python
binding: same names as the C calls, argument marshalling only, PyTorch for device memory and streams.
"""
from .binding import (HoughPlan, HoughPipeline, HoughError, hough_vertex_vote, hough_fit_circles, hough_fit_circles_static, FIT_STATIC_MAX_CANDIDATES, CAND_DTYPE, HOUGH_ACC_I32, HOUGH_ACC_U16, HOUGH_MODEL_HELIX, HOUGH_MODEL_LINE, alloc_candidates,
                      candidates_to_numpy, load_library, microbench, window_table, kernel_launches, version, LIB_PATH, EXPORTS)


def hough_plan_create(binning, bz_tesla=3.8, layers=(), max_hits=1 << 20, max_events=1) -> HoughPlan:
    """include/hough.h: hough_plan_create(binning, detector geometry)."""
    return HoughPlan(binning.n_phi, binning.n_qpt, binning.n_d0, binning.qpt_min, binning.qpt_max, binning.d0_min,
                     binning.d0_max, binning.accum_dtype, bz_tesla, layers, max_hits=max_hits, max_events=max_events,
                     model=getattr(binning, "model", 0))


def hough_vote(plan, hits_xy, event_offsets, accum, stream=None):
    return plan.vote(hits_xy, event_offsets, accum, stream)


def hough_find_peaks(plan, accum, n_events, threshold, cands, capacity, cand_offsets, stream=None):
    return plan.find_peaks(accum, n_events, threshold, cands, capacity, cand_offsets, stream)


def hough_assign_hits(plan, hits_xy, event_offsets, cands, cand_offsets, capacity, assoc_dj, min_hits, hit_to_cand,
                      cand_nhits, cand_keep, stream=None):
    return plan.assign_hits(hits_xy, event_offsets, cands, cand_offsets, capacity, assoc_dj, min_hits, hit_to_cand,
                            cand_nhits, cand_keep, stream)


def hough_plan_destroy(plan):
    plan.close()
