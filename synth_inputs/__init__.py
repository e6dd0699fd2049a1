"""Seeded synthetic inputs for the real-space AMOEBA polarization hot path.

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA
product (``paper_2011_01207_b200/``).  It draws random numbers and places atoms;
it contains none of the method's arithmetic (no Ewald, Thole, field, T, PCG).

The recipes follow BASELINE.json ``configs`` and SURVEY.md section 8(d)
("Synthetic inputs"); they stand in for the paper's DHFR / Mpro-Puddle / STMV
systems, which are not available offline.
"""
from .generator import (System, CONFIGS, make_config, water_box, tiny_cluster,
                        beta_for_cutoff)

__all__ = ["System", "CONFIGS", "make_config", "water_box", "tiny_cluster",
           "beta_for_cutoff"]
