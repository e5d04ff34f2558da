"""ORACLE -- test infrastructure only (see vicostream_oracle.py header).  Never imported by the
product path `paper_2606_19849_b200/`."""
from .vicostream_oracle import *  # noqa: F401,F403
from .vicostream_oracle import (  # noqa: F401
    cosine_similarity, pairwise_similarity, drop_predicate, temporal_keep_mask, compact,
    temporal_drop, grid_positions, next_position_base, text_positions, mrope_rotate, PagedKV,
    bounded_attention, merge_partial_attention, eq4_visible, eq4_mask, masked_attention_dense,
    mean_query, retrieval_scores, retrieve_topk, retrieve_threshold, fps_max,
)
from .stream import OracleStream  # noqa: F401
