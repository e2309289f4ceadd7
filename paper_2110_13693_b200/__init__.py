"""whp — B200-native (sm_100a) evaluation of candidate picking plans for warehouse SDO.

`paper_2110_13693_b200.whp` is the thin ctypes binding of the C-ABI library declared in
include/whp.h (built in-tree by `paper_2110_13693_b200.build`); `workloads` holds the seeded
synthetic input generators. Importing the package does not load the CUDA library; the first
call through `whp` does, and fails loudly if it has not been built.
"""
__all__ = ["whp", "workloads", "build"]
