"""The five workloads of BASELINE.json (`configs[0..4]`), as data.

Citations: B:L7..B:L11 = BASELINE.json configs 0..4; S15 / G1-G8 = SURVEY.md section 8(c)/8(d)
readings that complete what BASELINE.json leaves open (layer radii of the 14-layer barrel, pT law,
vertex kinematics, noise placement).  The paper itself (section 3) only describes a toy
transverse-plane detector; that one is kept as workload "paper_toy".
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Tuple

ACC_I32 = 0
ACC_U16 = 1

# B:L7 -- 10 cylindrical barrel layers [cm]
LAYERS_10: Tuple[float, ...] = (4.0, 7.0, 11.0, 25.0, 34.0, 43.0, 52.0, 61.0, 70.0, 110.0)
# PAPER.md:39 (section 3, Fig. 1): "a beampipe with radius of 3.0 cm, surrounded by ten concentric, evenly-spaced
# tracking layers with an outer radius of 110.0 cm" -- reading: spacing (110 - 3) / 10, first layer one spacing out
LAYERS_PAPER_TOY: Tuple[float, ...] = tuple(3.0 + 10.7 * l for l in range(1, 11))
# B:L9 "14 barrel layers from 4 to 110 cm"; radii per SURVEY S15 (config-0 radii plus 16, 80, 90, 100)
LAYERS_14: Tuple[float, ...] = (4.0, 7.0, 11.0, 16.0, 25.0, 34.0, 43.0, 52.0, 61.0, 70.0, 80.0, 90.0, 100.0, 110.0)


@dataclass(frozen=True)
class HoughBinning:
    n_phi: int
    n_qpt: int
    n_d0: int
    qpt_min: float = -1.0
    qpt_max: float = 1.0
    d0_min: float = -20.0
    d0_max: float = 20.0
    accum_dtype: int = ACC_I32
    model: int = 0               # 0: curved tracks (axis j = q/pT); 1: straight displaced tracks (axis j = d0 [cm] over
                                 # [qpt_min, qpt_max), n_d0 = 1) -- PAPER.md:45

    @property
    def n_bins(self) -> int:
        return self.n_phi * self.n_qpt * self.n_d0

    @property
    def bin_bytes(self) -> int:
        return 4 if self.accum_dtype == ACC_I32 else 2


@dataclass(frozen=True)
class HoughWorkload:
    name: str
    seed: int
    n_events: int
    layers: Tuple[float, ...]
    n_prompt: int
    n_displaced: int
    n_noise: int                 # -1: 5 % of the track hits, rounded (B:L7)
    pt_law: str                  # "uniform" (B:L7) | "exp" (B:L8: pT = pt_min + Exp(scale 2 GeV))
    pt_min: float
    pt_max: float                # used by "uniform" only
    binning: HoughBinning
    threshold: int
    bz_tesla: float = 3.8
    sigma_rphi_cm: float = 20.0e-4   # 20 um (B:L7)
    vertex_r_min: float = 1.0        # B:L8
    vertex_r_max: float = 20.0
    pt_exp_scale: float = 2.0
    assoc_dj: int = 1
    n_vertices: int = 0              # displaced vertices; 0: ceil(n_displaced / 4) (G4)
    cite: str = ""

    @property
    def min_hits(self) -> int:       # SURVEY D9 default
        return self.threshold

    def scaled(self, n_events: int) -> "HoughWorkload":
        """Same generation law, different number of events (event e is identical in both)."""
        return replace(self, n_events=n_events)

    def with_tracks(self, n_prompt: int) -> "HoughWorkload":
        """Same detector and binning, another number of prompt tracks (Fig. 2-style sweeps)."""
        return replace(self, n_prompt=n_prompt, name=f"{self.name}_{n_prompt}trk")


WORKLOADS = {
    0: HoughWorkload(name="cfg0_single_prompt_2d", seed=1, n_events=1, layers=LAYERS_10,
                     n_prompt=20, n_displaced=0, n_noise=-1, pt_law="uniform", pt_min=1.0, pt_max=10.0,
                     binning=HoughBinning(256, 256, 1, accum_dtype=ACC_I32), threshold=8, cite="B:L7"),
    1: HoughWorkload(name="cfg1_single_displaced_3d", seed=2, n_events=1, layers=LAYERS_10,
                     n_prompt=80, n_displaced=20, n_noise=1000, pt_law="exp", pt_min=1.0, pt_max=0.0,
                     binning=HoughBinning(256, 128, 64, accum_dtype=ACC_I32), threshold=7, cite="B:L8"),
    2: HoughWorkload(name="cfg2_pileup_3d", seed=3, n_events=1, layers=LAYERS_14,
                     n_prompt=2000, n_displaced=12, n_noise=5000, pt_law="exp", pt_min=0.9, pt_max=0.0,
                     binning=HoughBinning(512, 256, 64, accum_dtype=ACC_I32), threshold=10, cite="B:L9"),
    3: HoughWorkload(name="cfg3_batched_1024ev", seed=4, n_events=1024, layers=LAYERS_14,
                     n_prompt=500, n_displaced=5, n_noise=1500, pt_law="exp", pt_min=0.9, pt_max=0.0,
                     binning=HoughBinning(256, 128, 32, accum_dtype=ACC_U16), threshold=10, cite="B:L10"),
    4: HoughWorkload(name="cfg4_fine_binned", seed=5, n_events=1, layers=LAYERS_14,
                     n_prompt=10000, n_displaced=200, n_noise=20000, pt_law="exp", pt_min=0.9, pt_max=0.0,
                     binning=HoughBinning(1024, 512, 128, accum_dtype=ACC_U16), threshold=11, cite="B:L11"),
    # the paper's own toy scenario (Fig. 1): transverse plane, 10 evenly spaced layers
    # 3 -> 110 cm, 0.4 mm hit resolution, 500 curved prompt tracks, two-parameter space.  The paper states
    # neither field, pT spectrum, binning nor threshold: 3.8 T, pT = 1 GeV + Exp(2 GeV), 512 x 256 bins and threshold 8
    # (of 10 layers) are this build's choices.
    5: HoughWorkload(name="paper_toy_2d", seed=6, n_events=1, layers=LAYERS_PAPER_TOY,
                     n_prompt=500, n_displaced=0, n_noise=0, pt_law="exp", pt_min=1.0, pt_max=0.0,
                     binning=HoughBinning(512, 256, 1, accum_dtype=ACC_I32), threshold=8,
                     sigma_rphi_cm=0.04, cite="P:L39"),
    # straight displaced tracks in the two-parameter space (phi0, d0) ("or straight
    # displaced tracks"; Fig. 3: "four displaced jets").  The paper's toy detector with the field off:
    # 40 prompt tracks plus 160 tracks from 4 displaced vertices (round-robin, G4), 200 noise hits.  Binning (512 phi0 x
    # 256 d0 bins over [-30, 30) cm) and threshold are this build's choices.
    6: HoughWorkload(name="paper_toy_straight_displaced", seed=7, n_events=1, layers=LAYERS_PAPER_TOY,
                     n_prompt=40, n_displaced=160, n_noise=200, pt_law="exp", pt_min=1.0, pt_max=0.0,
                     binning=HoughBinning(512, 256, 1, qpt_min=-30.0, qpt_max=30.0, accum_dtype=ACC_I32, model=1),
                     threshold=8, bz_tesla=0.0, sigma_rphi_cm=0.04, vertex_r_min=2.0, vertex_r_max=12.0, n_vertices=4,
                     cite="P:L45, P:L61"),
}


def get_workload(idx: int) -> HoughWorkload:
    return WORKLOADS[idx]
