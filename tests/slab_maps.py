"""Index maps of the slab decomposition (include/lgf.h lgf_*_sharded; kernels k_slab_scatter / k_slab_gather of
csrc/slab.cuh), as plain integer arithmetic.  No arithmetic of the method is here: these are the owner and position
maps a rank needs to pack what it sends and to place what it receives when the ranks are separate processes
(torch.distributed all_to_all over NCCL between GPUs; over gloo in tests/test_slab_maps.py).  Test infrastructure: it
lives under tests/ because only the tests use it -- the library's sharded context runs its ranks inside one process.

Lattice (L0, L1, L2, L3), site x = x0 + L0 (x1 + L1 (x2 + L2 x3)); P ranks, P | L1 and P | L3.
  slab layout        rank r owns x3 in [r L3/P, (r+1) L3/P): local array [L3/P][L2][L1][L0]       (x0 fastest)
  transposed layout  rank s owns x1 in [s L1/P, (s+1) L1/P): local array [L3][L2][L1/P][L0]
"""
from __future__ import annotations

import numpy as np

__all__ = ["slab_shape", "transposed_shape", "send_blocks", "place_blocks", "send_blocks_back", "place_blocks_back",
           "halo_sources", "traffic_bytes"]


def slab_shape(dims, P):
    L0, L1, L2, L3 = (int(v) for v in dims)
    assert L3 % P == 0 and L1 % P == 0
    return (L3 // P, L2, L1, L0)


def transposed_shape(dims, P):
    L0, L1, L2, L3 = (int(v) for v in dims)
    assert L3 % P == 0 and L1 % P == 0
    return (L3, L2, L1 // P, L0)


def send_blocks(local, dims, P):
    """Forward transpose, sender side: the block of rank r's slab array [..., L3/P, L2, L1, L0] that rank s receives
    is x1 in [s L1/P, (s+1) L1/P).  Returns the list of P contiguous blocks [..., L3/P, L2, L1/P, L0]."""
    L1l = int(dims[1]) // P
    return [np.ascontiguousarray(local[..., s * L1l:(s + 1) * L1l, :]) for s in range(P)]


def place_blocks(blocks, dims, P):
    """Forward transpose, receiver side: the block from rank r holds x3 in [r L3/P, (r+1) L3/P).  Returns rank s's
    transposed array [..., L3, L2, L1/P, L0]."""
    return np.concatenate(blocks, axis=-4)


def send_blocks_back(localT, dims, P):
    """Backward transpose, sender side: of rank s's transposed array, rank r receives x3 in [r L3/P, (r+1) L3/P)."""
    L3l = int(dims[3]) // P
    return [np.ascontiguousarray(localT[..., r * L3l:(r + 1) * L3l, :, :, :]) for r in range(P)]


def place_blocks_back(blocks, dims, P):
    """Backward transpose, receiver side: the block from rank s holds x1 in [s L1/P, (s+1) L1/P)."""
    return np.concatenate(blocks, axis=-2)


def halo_sources(r, P):
    """(rank whose LAST time slice of U_3 rank r needs for S1, rank whose FIRST time slice of X rank r needs for S3)."""
    return (r - 1) % P, (r + 1) % P


def traffic_bytes(dims, P, nc=6, cb=16):
    """Bytes ONE rank sends per iteration: U_3 halo, X halo, the two transposes (the share of its field that changes
    owner, twice).  cb: bytes per complex number."""
    L0, L1, L2, L3 = (int(v) for v in dims)
    S = L0 * L1 * L2
    Vl = S * L3 // P
    return dict(halo_u_bytes=S * nc * cb, halo_x_bytes=S * 4 * cb, transpose_bytes=2 * (Vl * 4 * cb) * (P - 1) // P)
