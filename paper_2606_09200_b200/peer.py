"""N4 plumbing: one process per GPU, every rank's buffer reachable from every other rank.

Argument marshalling and process-group plumbing only -- the exchange itself runs in the library's kernels
(`ra_allreduce_peer`, `ra_alltoall_peer`, csrc/ra_peer.cu).

    group = PeerGroup()                                   # torch.distributed must be initialised (nccl or gloo)
    bufs = group.share(my_tensor)                         # P device pointers in RANK ORDER, mine at index rank
    group.allreduce(bufs, my_tensor.numel())              # barrier; my slice, fixed rank order; sync; barrier
    recvs = group.share(my_recv)
    group.alltoall(my_send, recvs, chunk_bytes)
    group.close()

`exchange` is the only step that talks to other ranks: an all-gather of fixed-size handle records over the process group
(CPU tensors, so it works on gloo and -- staged through the device -- on nccl).  Rank order is the group's rank order:
index r of every returned list belongs to rank r, which is what fixes the allreduce's summation order.
"""
from __future__ import annotations

HANDLE_BYTES = 80          # sizeof(ra_ipc_handle)


def exchange(local: bytes, group=None) -> list:
    """All-gather one fixed-size record per rank; returns the P records in rank order (index r = rank r's)."""
    import torch
    import torch.distributed as dist
    if not dist.is_initialized():
        raise RuntimeError("peer.exchange: torch.distributed is not initialised")
    world = dist.get_world_size(group)
    mine = torch.frombuffer(bytearray(local), dtype=torch.uint8)
    backend = dist.get_backend(group)
    dev = torch.device("cuda", torch.cuda.current_device()) if backend == "nccl" else torch.device("cpu")
    mine = mine.to(dev)
    out = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(out, mine, group=group)
    recs = [bytes(t.cpu().numpy().tobytes()) for t in out]
    if recs[dist.get_rank(group)] != local:
        raise RuntimeError("peer.exchange: rank order of the gathered records does not match this rank")
    return recs


class PeerGroup:
    """Shares device buffers across the ranks of a process group and runs the peer collectives on them."""

    def __init__(self, group=None):
        import torch.distributed as dist
        if not dist.is_initialized():
            raise RuntimeError("PeerGroup: torch.distributed is not initialised")
        self.group = group
        self.rank = dist.get_rank(group)
        self.world = dist.get_world_size(group)
        self._opened = []

    def share(self, tensor) -> list:
        """Export `tensor`, gather every rank's handle, open the peers'.  Returns P device pointers (int) in rank order."""
        import paper_2606_09200_b200 as ra
        handles = exchange(ra.ra_ipc_export(tensor), self.group)
        ptrs = []
        for r, h in enumerate(handles):
            if r == self.rank:
                ptrs.append(int(tensor.data_ptr()))
            else:
                p = ra.ra_ipc_open(h)
                self._opened.append(p)
                ptrs.append(p)
        return ptrs

    def barrier(self):
        import torch
        import torch.distributed as dist
        torch.cuda.synchronize()
        dist.barrier(group=self.group)

    def allreduce(self, bufs, count, sm_budget=0, variant=0, stream=None):
        """In-place sum over the P shared buffers: this rank reduces its slice (ra_peer_slice) and writes it to all P."""
        import paper_2606_09200_b200 as ra
        self.barrier()                                    # every rank's input is in place
        ra.ra_allreduce_peer(bufs, self.rank, count, sm_budget=sm_budget, variant=variant, stream=stream)
        self.barrier()                                    # every slice has been written everywhere

    def alltoall(self, send, recvs, chunk_bytes, sm_budget=0, variant=0, stream=None):
        """recv_j[rank] = send_rank[j] for every j: this rank pushes its P chunks."""
        import paper_2606_09200_b200 as ra
        self.barrier()
        ra.ra_alltoall_peer(send, recvs, self.rank, chunk_bytes, sm_budget=sm_budget, variant=variant, stream=stream)
        self.barrier()

    def close(self):
        import paper_2606_09200_b200 as ra
        self.barrier()                                    # nobody still reads a mapping that is about to go
        for p in self._opened:
            ra.ra_ipc_close(p)
        self._opened = []
