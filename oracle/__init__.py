"""TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes marshalling for oracle/whp_oracle.c (the plain single-threaded CPU restatement of the
hot path). Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package; the product package never does.
"""
from .binding import (  # noqa: F401
    LARGEST_GAP,
    RETURN,
    S_SHAPE,
    argmin,
    batch_largest_gap_distance,
    batch_return_distance,
    batch_distance,
    build,
    decode_neighbour,
    eval_candidate_batches,
    eval_candidates,
    eval_legsum,
    eval_moves,
    eval_routing,
    eval_swaps,
    kmeans_slotting,
    nhatc_loop,
    nhatc_update,
    optimal_route,
    penalty,
    swap_trajectory,
    tour_length,
)
