"""Seeded synthetic workloads: shapes and raw-byte generators.

This package is the ONLY code shared by the CUDA path (``paper_2511_11617_b200``)
and the CPU oracle (``oracle/``).  It holds *no arithmetic of the method*: no
partition formula, no planner, no slot addressing, no page-table rule.  It only
describes the inputs (model shapes, tensor inventory, scenario parameters from
BASELINE.json ``configs``) and produces deterministic bytes for them.
"""
from .configs import (  # noqa: F401
    CONFIGS, Config, ModelShape, KVShape, Scenario, TensorSpec,
    tensor_inventory, get_config,
)
from .gen import fill_bytes, fill_normal16, hash64, SEED0  # noqa: F401
