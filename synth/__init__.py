"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic: only shapes, seeds, distributions and dtype
casts (torch's own bf16 cast).  The five workloads are the `configs` of /root/repo/BASELINE.json;
they stand in for the paper's Video-MME segments / screenshots (none of that data is here or
needed): K, V ~ N(0,1), U ~ N(0,1), W ~ N(0, w_std), offsets uniform, block tables random
permutations.  The recipe is restated in DESIGN.md ("Input recipe").
"""
from .configs import CONFIGS, Config            # noqa: F401
from .gen import (make_chunk, make_block_table, make_offsets, make_query, torch_dtype,  # noqa: F401
                  randn_device)
