"""Seeded synthetic inputs shared by the CPU oracle and the CUDA path.

This package holds NO arithmetic of the MLPF method: only random draws of
events (PF-element feature rows + event offsets) and of weight tensors, with
the shapes and distributions BASELINE.json's five configs name.  The recipe is
stated in DESIGN.md ("Input recipe").  Both `oracle/` and the product package
consume these arrays; neither imports the other.
"""
from .configs import (ModelCfg, CONFIGS, BASE_SEED, N_FEAT, N_TYPES, N_CLASSES,
                      REG_DIMS, N_REG, model_cfg, weight_names, param_count, stack_prefix)
from .events import make_events, make_named_events
from .weights import make_weights, sharpen

__all__ = ["ModelCfg", "CONFIGS", "BASE_SEED", "N_FEAT", "N_TYPES", "N_CLASSES",
           "REG_DIMS", "N_REG", "model_cfg", "weight_names", "param_count", "stack_prefix",
           "make_events", "make_named_events", "make_weights", "sharpen"]
