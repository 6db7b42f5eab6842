"""Seeded synthetic inputs for the PVFinder hot path (events + weights).

This package serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_2602_19959_b200/``) and therefore holds none of the method's arithmetic:
no interval assignment, no FC, no convolution, no peak finding.  It only draws the
random numbers the configs in BASELINE.json describe and lays them out as the
boundary expects (SoA track arrays + event offsets, PyTorch-layout weight tensors).

Recipe and citations: DESIGN.md "Input recipe"; BASELINE.json configs 0-4;
PAPER.md:11,17 (5.6 PVs per event), PAPER.md:27 (nine features per track).
"""
from .events import EventBatch, make_events, CONFIG_EVENT_MODELS, shard_events, select_events
from .weights import (PVFWeights, make_weights, unet_layer_shapes, fc_layer_shapes,
                      CONV_NAMES)

__all__ = [
    "EventBatch", "make_events", "CONFIG_EVENT_MODELS", "shard_events", "select_events",
    "PVFWeights", "make_weights", "unet_layer_shapes", "fc_layer_shapes", "CONV_NAMES",
]
