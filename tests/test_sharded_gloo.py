"""World-size-2 gloo test (CPU) of the exchange behind the slab-decomposed step:
the communicator's all-to-all over equal blocks in rank order turns x slabs into "locally transposed" y slabs when
every rank sends every peer one (NX/P) x (NY/P) x NZ block, the way back restores the x slabs, and the norm parts add
up.  The CUDA stages around the exchange are covered on one GPU by tests/test_gpu_sharded.py (ranks emulated)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def pack_blocks(slab_x, P):
    """[nxl][ny][w] -> [P][nxl][nyl][w]: block q holds rank q's y range (the layout dgpe_slab_stage_a/c write)."""
    nxl, ny, w = slab_x.shape
    return slab_x.reshape(nxl, P, ny // P, w).permute(1, 0, 2, 3).contiguous()


def unpack_blocks(blocks, P):
    """[P][nxl][nyl][w] -> [nxl][ny][w] (what dgpe_slab_stage_c/e do with what comes back)."""
    _, nxl, nyl, w = blocks.shape
    return blocks.permute(1, 0, 2, 3).reshape(nxl, P * nyl, w).contiguous()


def global_field(nx, ny, w):
    g = torch.arange(nx * ny * w, dtype=torch.float64).reshape(nx, ny, w)
    return torch.complex(g, -0.5 * g)


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    import torch.distributed as dist
    from paper_1610_05329_b200 import sharded
    dist.init_process_group("gloo", rank=rank, world_size=world)
    comm = sharded.DistComm()
    nx, ny, w = 6, 8, 5
    nxl, nyl = nx // world, ny // world
    X = global_field(nx, ny, w)
    mine = X[rank * nxl:(rank + 1) * nxl]                              # my x slab
    send = pack_blocks(mine, world).reshape(-1)
    recv = torch.empty_like(send)
    comm.all_to_all([send], [recv])
    yslab = recv.reshape(nx, nyl, w)                                   # blocks in rank order ARE the y slab
    ok_fwd = bool(torch.equal(yslab, X[:, rank * nyl:(rank + 1) * nyl]))
    back = torch.empty_like(recv)
    comm.all_to_all([recv], [back])                                    # the y slab is the send buffer of the way back
    ok_back = bool(torch.equal(unpack_blocks(back.reshape(world, nxl, nyl, w), world), mine))
    part = torch.tensor([1.0 + rank], dtype=torch.float64)
    comm.all_reduce_sum([part])
    q.put((rank, comm.world, ok_fwd, ok_back, float(part[0]), send.numel() // world))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_exchange_slabs_and_sum_the_norm():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
    from paper_1610_05329_b200 import sharded
    for rank, world, ok_fwd, ok_back, total, blk in res:
        assert world == 2 and ok_fwd and ok_back
        assert total == 3.0                                            # 1 + 2: the norm parts of both ranks
        assert blk == sharded.block_elems(6, 8, 5, 2) == 3 * 4 * 5      # (NX/P) (NY/P) w per peer


def test_local_comm_is_the_same_exchange():
    """The single-process emulation (all ranks on one device) moves the same blocks as the distributed all-to-all."""
    from paper_1610_05329_b200 import sharded
    P, nx, ny, w = 3, 6, 9, 4
    X = global_field(nx, ny, w)
    nxl, nyl = nx // P, ny // P
    send = [pack_blocks(X[p * nxl:(p + 1) * nxl], P).reshape(-1) for p in range(P)]
    recv = [torch.empty_like(s) for s in send]
    comm = sharded.LocalComm(P)
    comm.all_to_all(send, recv)
    for q in range(P):
        assert torch.equal(recv[q].reshape(nx, nyl, w), X[:, q * nyl:(q + 1) * nyl])
    back = [torch.empty_like(s) for s in send]
    comm.all_to_all(recv, back)
    for p in range(P):
        assert torch.equal(unpack_blocks(back[p].reshape(P, nxl, nyl, w), P), X[p * nxl:(p + 1) * nxl])
    parts = [torch.tensor([float(p + 1)], dtype=torch.float64) for p in range(P)]
    comm.all_reduce_sum(parts)
    assert all(float(v[0]) == 6.0 for v in parts)


def test_block_sizes_and_divisibility():
    from paper_1610_05329_b200 import sharded
    assert sharded.block_elems(480, 480, 250, 8) == 60 * 60 * 250     # the paper's Table 3 grid on 8 ranks
    with pytest.raises(ValueError):
        sharded.block_elems(480, 500, 250, 8)
