"""CPU oracle for HyperVAttention's clustered sparse-attention operator.

TEST INFRASTRUCTURE ONLY.  Plain, slow, fp64 numpy restatement of the paper's Eq. 1-10,
Alg. 1 and Alg. 2, in the paper's order and notation.  It shares no code with the CUDA
path (`paper_2607_03012_b200/csrc`, `paper_2607_03012_b200/binding.py`) and neither imports
the other.  Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` /
`--impl reference` legs may import this package.

Parity status of each function is stated in its module header.  Every function has a pin that does
not come from the oracle itself (hand fixtures, brute force, closed forms, invariants:
tests/test_oracle_*.py); the hybrid intermediate update follows reading R-H3 / R-H3' of DESIGN.md and
is pinned by the invariant "incremental update == recomputation from the labels" (see oracle/hybrid.py).
"""
from .grid import grid_dims, clip_window, window_start, centre_token, home_cell, window_ids  # noqa: F401
from .cluster import local_window_kmeans, lowe_ratio  # noqa: F401
from .mask import build_mask  # noqa: F401
from .merge import merge_clusters, side_hash, tile_cost  # noqa: F401
from .plan import build_plan  # noqa: F401
from .attention import masked_attention_rows, token_key_mask  # noqa: F401
from .hybrid import select_subset, subset_update  # noqa: F401
from .forward import forward_head  # noqa: F401
