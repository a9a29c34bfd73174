"""Seeded synthetic inputs for the Hough track-finding path (arXiv 1311.2769).

This package serves BOTH the CPU oracle (`oracle/`) and the CUDA library
(`paper_1311_2769_b200/`).  It holds the detector/track simulation and the
workload descriptions only -- none of the Hough method's arithmetic (no
voting formula, no binning of votes, no peak or assignment logic).
"""
from .configs import HoughBinning, HoughWorkload, WORKLOADS, get_workload, LAYERS_10, LAYERS_14, LAYERS_PAPER_TOY
from .generator import (generate_events, generate_event, helix_hits, line_hits, K_GEV_PER_T_CM,
                        EventBatch)

__all__ = ["HoughBinning", "HoughWorkload", "WORKLOADS", "get_workload", "LAYERS_10", "LAYERS_14", "LAYERS_PAPER_TOY",
           "generate_events", "generate_event", "helix_hits", "line_hits", "K_GEV_PER_T_CM", "EventBatch"]
