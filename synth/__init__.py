"""Seeded synthetic inputs (jets and weight blobs) shared by the oracle tests and the CUDA harness.

This package holds NO arithmetic of the method (no kNN, no EdgeConv, no pooling): it only draws
random numbers in the normative order of DESIGN.md "Input recipe" and lays them out as flat fp32
arrays.  Both `oracle/` (test infrastructure) and `paper_2312_06838_b200/` (the CUDA product) are fed
from here; neither imports the other.
"""
from .arch import Arch, ARCHS, weight_count          # noqa: F401
from .weights import make_weights                    # noqa: F401
from .jets import (make_tiny, make_particlenet_batch, make_ragged_batch, make_sweep_batch,  # noqa: F401
                   make_client_pool, make_edge_case_batch, pad_batch, JetBatch, make_paper_f5_batch, to_channel_first)
from .bdt import make_bdt, make_bdt_events           # noqa: F401
