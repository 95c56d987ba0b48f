"""Worker for test_peer.py / test_peer_gpu.py (world_size 2, gloo).

  cpu   the handle exchange and rank-order bookkeeping with stand-in handle bytes (no CUDA anywhere)
  gpu   two processes on ONE GPU: each owns a buffer on cuda:0, publishes it through a real CUDA IPC handle, maps the
        other's, and runs ra_allreduce_peer / ra_alltoall_peer on its own slice / row.  Ranks are ordered by host
        barriers only (no kernel waits on another rank).  Every rank checks the result against the oracle.
"""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))
import numpy as np  # noqa: E402
import torch  # noqa: E402
import torch.distributed as dist  # noqa: E402

mode = sys.argv[1]
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
from paper_2606_09200_b200 import peer  # noqa: E402

if mode == "cpu":
    # stand-in handles: 80 bytes that encode the owner, so a permuted gather would be seen
    mine = bytes([rank]) * peer.HANDLE_BYTES
    recs = peer.exchange(mine)
    assert len(recs) == world and all(recs[r] == bytes([r]) * peer.HANDLE_BYTES for r in range(world)), recs
    # the slices every rank derives (host-only library call) partition the buffer identically on every rank
    import paper_2606_09200_b200 as ra
    count = 1000003
    sl = [ra.ra_peer_slice(count, world, r) for r in range(world)]
    gathered = [None] * world
    dist.all_gather_object(gathered, sl)
    assert all(g == sl for g in gathered)
    assert sl[0][0] == 0 and sl[-1][1] == count and all(sl[r][1] == sl[r + 1][0] for r in range(world - 1))
    dist.barrier()
    if rank == 0:
        print(f"PEER_CPU_OK world={world}")
else:
    import oracle
    import ra_inputs
    import paper_2606_09200_b200 as ra
    from helpers import to_dev, to_host
    torch.cuda.set_device(0)
    g = peer.PeerGroup()
    # ---- allreduce: count not a multiple of 4*P, so slices are ragged and the scalar tail is rank P-1's
    count = (1 << 20) + 37
    host = [ra_inputs.uniform_f32(count, 4242, ra_inputs.STREAM_AR + r) for r in range(world)]
    mine = to_dev(host[rank])
    bufs = g.share(mine)
    assert bufs[rank] == mine.data_ptr() and len(set(bufs)) == world
    for variant in (0, 1):
        mine.copy_(to_dev(host[rank]))
        g.allreduce(bufs, count, variant=variant)
        ref = [h.copy() for h in host]
        oracle.allreduce(ref)
        assert to_host(mine, np.float32).tobytes() == ref[rank].tobytes(), f"rank {rank} variant {variant}: allreduce differs"
    # ---- alltoall: tagged chunks, rank i owns row i of the P x P chunk matrix
    chunk = 256 * 1024 + 16
    send_all = ra_inputs.tagged_chunks(world, chunk)                        # uint64 words, [P][P][chunk/8]
    want = oracle.alltoall(send_all, world, chunk)
    row = np.ascontiguousarray(send_all.reshape(world, -1)[rank])
    for variant in (0, 1, 2):
        d_send = to_dev(row)
        d_recv = torch.zeros_like(d_send)
        recvs = g.share(d_recv)
        g.alltoall(d_send, recvs, chunk, variant=variant)
        got = to_host(d_recv, np.uint64)
        assert got.tobytes() == np.ascontiguousarray(want.reshape(world, -1)[rank]).tobytes(), f"rank {rank} variant {variant}: alltoall differs"
    g.close()
    dist.barrier()
    if rank == 0:
        print(f"PEER_GPU_OK world={world}")
dist.destroy_process_group()
