"""CPU oracle package - TEST INFRASTRUCTURE (see oracle/lsa_oracle.py header)."""
from .lsa_oracle import (  # noqa: F401
    EPS_NORM, LsaOracle, PoolExhausted, ResidencyOracle, attention, chunk_scores,
    merge_partials, partial_attention, query_tower, topk_select, trigger_fires,
    validate_selection, widen,
)
from . import l1_oracle  # noqa: F401,E402  (paper-exact Level-1 indexer, NEXT-1)
from . import l2_oracle  # noqa: F401,E402  (Level-2 in-window Top-k, NEXT-2)
