"""Seeded synthetic inputs for the VMAT beamlet-price path (BASELINE.json `configs`).

This module is the ONE thing the CPU oracle (`oracle/`) and the CUDA library
(`paper_1503_01721_b200/`) share: it produces the input arrays (COO triplets of
the dose-deposition-coefficient matrix D, the angle / leaf-row column offsets,
structure ids, objective parameters, fluence vectors x).  It holds none of the
method's arithmetic (no D.x, no gradient, no D^T.g, no leaf selection) and it
imports neither side.

The synthetic phantoms stand in for the paper's private patient DDC matrices
(Table 3): angle-blocked columns (L119), one
cylinder-shaped footprint per beamlet with a lateral cutoff like the paper's
cone radius gamma (L147), FP32 values + int32 indices (Table 2).
The recipe (readings D1-D7 of SURVEY.md section 8(d)) is restated in DESIGN.md.

Everything is written with torch ops on a caller-chosen device so the same code
generates config 0 on the CPU in milliseconds and config 3 (3e9 nnz) on the GPU
in seconds.  The arrays are generated ONCE and fed to both sides; they are never
regenerated separately (exp() differs in ulps between devices).
"""
from .phantom import (  # noqa: F401
    PhantomSpec, Phantom, Sphere, ZCylinder, Arc,
    config_spec, generate, draw_x, hash_uniform, CONFIG_NAMES,
)
