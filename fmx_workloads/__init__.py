"""Seeded synthetic workloads for the mixed-task vFM forward (configs of BASELINE.json).

This module is the ONLY code shared by the oracle side (tests, bench cpu_baseline) and the
CUDA side.  It holds no arithmetic of the method: it draws seeded random tensors, rounds
them once to bf16 bit patterns, and describes shapes.  Recipes follow SURVEY.md §8(d1) and
the readings listed in DESIGN.md §3.
"""
from .bf16 import f32_to_bf16_bits, bf16_bits_to_f32, bf16_bits_to_f64
from .spec import (BackboneSpec, AdapterSpec, TaskSpec, Workload, make_workload,
                   TARGETS, target_dims, config_names)

__all__ = ["f32_to_bf16_bits", "bf16_bits_to_f32", "bf16_bits_to_f64", "BackboneSpec",
           "AdapterSpec", "TaskSpec", "Workload", "make_workload", "TARGETS", "target_dims",
           "config_names"]
