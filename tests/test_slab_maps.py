"""Host logic of the slab decomposition (tests/slab_maps.py) at world size 2 over gloo on the CPU: the two
all-to-all transposes built from the send/place maps reproduce the global re-distribution, the halo sources are the
periodic neighbours, and the byte counts are those the C library reports (include/lgf.h lgf_sharded_traffic)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import slab_maps as slab


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, dims, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    L0, L1, L2, L3 = dims
    # the global field: value = global site index (+ component * V), so every element says where it came from
    V = L0 * L1 * L2 * L3
    g = (np.arange(V, dtype=np.float64).reshape(L3, L2, L1, L0)[None] + V * np.arange(4, dtype=np.float64)[:, None, None, None, None])
    L3l, L1l = L3 // world, L1 // world
    mine = np.ascontiguousarray(g[:, rank * L3l:(rank + 1) * L3l])                    # slab layout [4][L3/P][L2][L1][L0]
    assert mine.shape[1:] == slab.slab_shape(dims, world)
    # forward transpose: all_to_all of the send blocks, then place
    send = [torch.from_numpy(b) for b in slab.send_blocks(mine, dims, world)]
    recv = [torch.empty_like(send[0]) for _ in range(world)]
    _a2a_gloo(recv, send, rank, world)
    mineT = slab.place_blocks([t.numpy() for t in recv], dims, world)
    assert mineT.shape[1:] == slab.transposed_shape(dims, world)
    okT = np.array_equal(mineT, g[:, :, :, rank * L1l:(rank + 1) * L1l, :])
    # backward transpose brings the slab back
    send = [torch.from_numpy(b) for b in slab.send_blocks_back(mineT, dims, world)]
    recv = [torch.empty_like(send[0]) for _ in range(world)]
    _a2a_gloo(recv, send, rank, world)
    back = slab.place_blocks_back([t.numpy() for t in recv], dims, world)
    ok_back = np.array_equal(back, mine)
    # halos: last slice of the rank below, first slice of the rank above (periodic)
    lo, hi = slab.halo_sources(rank, world)
    last = torch.from_numpy(np.ascontiguousarray(mine[:, -1]))
    first = torch.from_numpy(np.ascontiguousarray(mine[:, 0]))
    got_lo, got_hi = torch.empty_like(last), torch.empty_like(first)
    reqs = [dist.isend(last, (rank + 1) % world), dist.irecv(got_lo, lo)]
    for q in reqs:
        q.wait()
    reqs = [dist.isend(first, (rank - 1) % world), dist.irecv(got_hi, hi)]
    for q in reqs:
        q.wait()
    ok_halo = np.array_equal(got_lo.numpy(), g[:, (rank * L3l - 1) % L3]) and np.array_equal(got_hi.numpy(), g[:, ((rank + 1) * L3l) % L3])
    out[rank] = (okT, ok_back, ok_halo)
    dist.destroy_process_group()


def _a2a_gloo(recv, send, rank, world):
    """all_to_all from point-to-point calls (gloo has no all_to_all): what ncclSend/ncclRecv groups do between GPUs."""
    reqs = []
    for p in range(world):
        if p == rank:
            recv[p].copy_(send[p])
        else:
            reqs.append(dist.isend(send[p], p))
            reqs.append(dist.irecv(recv[p], p))
    for q in reqs:
        q.wait()


@pytest.mark.parametrize("dims", [(4, 4, 2, 4), (8, 4, 4, 8)])
def test_transposes_and_halos_at_world_size_2(dims):
    world = 2
    port = _free_port()
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, port, dims, out), nprocs=world, join=True)
    assert all(all(out[r]) for r in range(world)), dict(out)


def test_traffic_model():
    t = slab.traffic_bytes((64, 64, 64, 64), 8)
    S = 64 ** 3
    assert t["halo_u_bytes"] == S * 96 and t["halo_x_bytes"] == S * 64
    assert t["transpose_bytes"] == 2 * (S * 8 * 64) * 7 // 8          # 7/8 of a rank's 64 B/site field leaves, twice
