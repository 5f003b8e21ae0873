"""Seeded synthetic inputs for the closed-shell (T) energy path.

This package is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA
path (`paper_2502_17963_b200/`).  It holds no arithmetic of the (T) method —
only the random / closed-form *input* recipes (SURVEY.md §8(c) G12 and P2,
BASELINE.json `configs`).
"""
from .generator import (CONFIGS, TInputs, make_inputs, make_config,
                        worked_example, sample_triplets)

__all__ = ["CONFIGS", "TInputs", "make_inputs", "make_config",
           "worked_example", "sample_triplets"]
