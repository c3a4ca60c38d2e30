"""Seeded synthetic CBCT workloads C0..C4 (inputs only).

This package generates the *inputs* both the CPU oracle (``oracle/``) and the
CUDA path (``paper_1204_6367_b200/``) consume.  It holds none of the
projector's arithmetic: no ray geometry, no clipping, no interpolation, no
energy sum.  It imports neither ``oracle`` nor ``paper_1204_6367_b200``.

The paper measures on a Catphan 600 CT, a
head-and-neck patient CT, a Boone-Seibert spectrum and a measured detector
response; none of that is available, so these seeded phantoms and smooth
analytic curves stand in for them with the same shapes (SURVEY.md section 8(d),
DESIGN.md "Input recipe").
"""
from .prng import SplitMix64
from .configs import Workload, make_workload, WORKLOAD_NAMES, PHANTOMS, pure_cell_fraction, with_tissue_classes, shard_projections

__all__ = ["SplitMix64", "Workload", "make_workload", "WORKLOAD_NAMES", "PHANTOMS", "pure_cell_fraction", "with_tissue_classes",
           "shard_projections"]
