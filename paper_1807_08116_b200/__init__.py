"""B200-native (sm_100a) hot path of Khrapov & Khoperskov (arXiv 1807.08116):
grid-sort neighbour search, SPH density / forces, direct PP gravity, leapfrog update.

The product is the C-ABI library built from csrc/ (declared in include/sph_b200.h);
`binding` is its thin ctypes face.  `workloads` holds the seeded input generators and
is the only module shared with the oracle.  Importing this package does not load CUDA.
"""
__all__ = ["binding", "workloads"]
