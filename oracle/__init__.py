"""ORACLE package -- test infrastructure, not the product.

Plain CPU restatement of the causal-set action path of arXiv:1805.04463
(see oracle/causet_oracle.c for the citations).  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package; the product (paper_1805_04463_b200) never does.
"""
from .oracle import (  # noqa: F401
    GEOM_MINK2_LIGHTCONE,
    GEOM_MINK_CONE,
    GEOM_DS2_SLAB,
    GEOM_FLRW_POLAR,
    GEOM_DS4_SPHERICAL,
    build,
    row_stride_words,
    relation,
    causal_matrix_bytes,
    causal_matrix_bits,
    transpose_bits,
    degrees,
    pack_bytes,
    unpack_bits,
    interval_hist_alg19,
    interval_hist_alg20,
    count_relations,
    bd_action,
    chain_pair,
    chain_heights,
    greedy_antichain,
    smear_f,
    smeared_action,
    max_threads,
    action_pipeline,
)
