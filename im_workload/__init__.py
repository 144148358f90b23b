"""Seeded synthetic input generators shared by the oracle tests and the CUDA path.

This module holds NONE of the method's arithmetic (no Philox, no tick semantics, no MLP,
no GAE): it only materialises the workloads of BASELINE.json `configs[0..4]` as plain
integer tables / numpy arrays, which each side then marshals
into its own C struct.
"""
from .workload import (  # noqa: F401
    CONFIGS,
    PoolSpec,
    make_pool_spec,
    make_policy_blob,
    poisson_cdf_row,
    lognormal_table,
    blob_views,
    TOK_PER_QUERY_NOMINAL,
)
