"""N4 on the one GPU at hand: the peer collectives against the oracle, bit for bit.

(1) P sequential "ranks" on one device: every rank's call gets the same P pointers (rank order) and reduces only its own
    slice / pushes only its own row; after all P calls every buffer must equal the oracle's allreduce / alltoall.  This
    pins the slice arithmetic and the kernels' addressing at real offsets.
(2) Two PROCESSES on the one GPU through real CUDA IPC handles exchanged over gloo (tests/_peer_worker.py): the path a
    multi-GPU node takes, minus NVLink.  Ranks are ordered by host barriers; no kernel waits on another rank.
"""
import numpy as np
import pytest

import oracle
import ra_inputs
from helpers import to_dev, to_host
from test_peer import run_peer_worker

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ra():
    import paper_2606_09200_b200 as m
    return m


@pytest.mark.parametrize("P,count", [(1, 4099), (2, 1 << 20), (4, (1 << 18) + 37), (8, 1 << 21), (3, 5), (16, 70001)])
@pytest.mark.parametrize("variant", [0, 1, 2])
def test_allreduce_peer_sequential_ranks(ra, P, count, variant):
    import torch
    host = [ra_inputs.uniform_f32(count, 900 + P, ra_inputs.STREAM_AR + r) for r in range(P)]
    dev = [to_dev(h) for h in host]
    for r in range(P):
        ra.ra_allreduce_peer(dev, r, count, variant=variant)
        torch.cuda.synchronize()
        # after rank r's call exactly the slices of ranks 0..r hold the sum, everywhere
    ref = [h.copy() for h in host]
    oracle.allreduce(ref)
    for dd, rr in zip(dev, ref):
        assert to_host(dd, np.float32).tobytes() == rr.tobytes()


def test_allreduce_peer_touches_only_its_slice(ra):
    import torch
    P, count = 4, 100003
    host = [ra_inputs.uniform_f32(count, 77, ra_inputs.STREAM_AR + r) for r in range(P)]
    dev = [to_dev(h) for h in host]
    ra.ra_allreduce_peer(dev, 2, count)
    torch.cuda.synchronize()
    b, e = ra.ra_peer_slice(count, P, 2)
    ref = [h.copy() for h in host]
    oracle.allreduce(ref)
    for r in range(P):
        got = to_host(dev[r], np.float32)
        assert got[b:e].tobytes() == ref[r][b:e].tobytes()
        assert got[:b].tobytes() == host[r][:b].tobytes() and got[e:].tobytes() == host[r][e:].tobytes()


@pytest.mark.parametrize("P,chunk", [(1, 4096), (2, 64 * 1024 + 16), (4, 1 << 20), (8, 48), (5, 300 * 1024)])
@pytest.mark.parametrize("variant", [0, 1, 2])
def test_alltoall_peer_sequential_ranks(ra, P, chunk, variant):
    import torch
    send = ra_inputs.tagged_chunks(P, chunk)
    rows = np.ascontiguousarray(send).reshape(P, -1)
    d_send = [to_dev(np.ascontiguousarray(rows[r])) for r in range(P)]
    d_recv = [torch.zeros_like(d_send[r]) for r in range(P)]
    for r in range(P):
        ra.ra_alltoall_peer(d_send[r], d_recv, r, chunk, variant=variant)
    torch.cuda.synchronize()
    want = np.ascontiguousarray(oracle.alltoall(send, P, chunk)).reshape(P, -1)
    for r in range(P):
        assert to_host(d_recv[r], np.uint64).tobytes() == want[r].tobytes()


def test_peer_argument_errors(ra):
    import torch
    a = torch.zeros(1024, dtype=torch.float32, device="cuda")
    b = torch.zeros(1024, dtype=torch.float32, device="cuda")
    for bad in (dict(bufs=[a, b], rank=2), dict(bufs=[a, b], rank=-1), dict(bufs=[a, a], rank=0)):
        with pytest.raises(ra.RaError):
            ra.ra_allreduce_peer(bad["bufs"], bad["rank"], 1024)
    with pytest.raises(ra.RaError):
        ra.ra_alltoall_peer(a, [a, b], 0, 2048)                       # send aliases a receive buffer
    with pytest.raises(ra.RaError):
        ra.ra_alltoall_peer(a, [b], 0, 24)                            # chunk not a multiple of 16 bytes
    with pytest.raises(ra.RaError):
        ra.ra_ipc_close(a.data_ptr())                                 # not an IPC mapping


def test_ipc_export_reports_offset_inside_the_allocation(ra):
    import torch
    big = torch.zeros(1 << 20, dtype=torch.float32, device="cuda")
    h0 = ra.IpcHandle.from_buffer_copy(ra.ra_ipc_export(big))
    h1 = ra.IpcHandle.from_buffer_copy(ra.ra_ipc_export(big[1024:]))
    assert h1.offset == h0.offset + 4096 and h1.bytes == h0.bytes - 4096
    assert bytes(h0.opaque) == bytes(h1.opaque)                       # same allocation, same CUDA handle


def test_two_processes_one_gpu_real_ipc():
    r = run_peer_worker("gpu", timeout=900)
    assert r.returncode == 0, (r.stdout[-2000:], r.stderr[-4000:])
    assert "PEER_GPU_OK world=2" in r.stdout
