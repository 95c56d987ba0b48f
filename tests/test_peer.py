"""N4 host logic on CPU (no GPU): slice bookkeeping of the peer allreduce and the world_size-2 gloo handle exchange.

PAPER.md:30 / :69 -- the collectives run across the GPUs of a node; here every rank reduces its own 1/P slice in the fixed
order 0..P-1 and pushes its own row of chunks, so what must hold on the host side is: the slices partition the buffer the
same way on every rank, and index r of every gathered list is rank r's."""
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def ra():
    import paper_2606_09200_b200 as m
    return m


@pytest.mark.parametrize("count", [0, 1, 3, 4, 5, 37, 1024, 1000003, (1 << 24) + 1])
@pytest.mark.parametrize("P", [1, 2, 3, 4, 8, 16])
def test_slices_partition_the_buffer(ra, count, P):
    sl = [ra.ra_peer_slice(count, P, r) for r in range(P)]
    assert sl[0][0] == 0 and sl[-1][1] == count
    for r in range(P):
        b, e = sl[r]
        assert b <= e and b % 4 == 0 and (e % 4 == 0 or r == P - 1)          # 16-byte vectors; the scalar tail is the last rank's
        if r + 1 < P:
            assert e == sl[r + 1][0]
    # balanced to within one vector per rank (plus the tail)
    sizes = [e - b for b, e in sl]
    assert max(sizes) - min(sizes) <= 4 + 3


def test_slice_argument_errors(ra):
    for P, r in ((0, 0), (17, 0), (4, 4), (4, -1)):
        with pytest.raises(ra.RaError):
            ra.ra_peer_slice(100, P, r)


def test_alltoall_peer_rejects_aliased_buffers(ra):
    """Argument errors are found before any CUDA call (so this runs without a device): two ranks sharing one receive
    buffer, or a receive buffer overlapping the send buffer, is RA_ERR_INVALID_ARG."""
    chunk = 4096
    send, r0, r1 = 0x10000000, 0x20000000, 0x30000000
    for recv in ([r0, r0], [r0, r0 + chunk], [r0, send + chunk]):
        with pytest.raises(ra.RaError) as e:
            ra.ra_alltoall_peer(send, recv, 0, chunk, stream=0)
        assert e.value.status == ra.RA_ERR_INVALID_ARG, recv
    import torch
    if not torch.cuda.is_available():                              # (made-up addresses: never let them reach a real GPU)
        with pytest.raises(ra.RaError) as e:                       # disjoint buffers get past validation ...
            ra.ra_alltoall_peer(send, [r0, r1], 0, chunk, stream=0)
        assert e.value.status in (ra.RA_ERR_CUDA, ra.RA_ERR_ARCH)   # ... and stop at "no device", not at the arguments


def test_peer_calls_fail_loudly_without_device(ra):
    import torch
    if torch.cuda.is_available():
        pytest.skip("needs a CPU-only box")
    with pytest.raises(ra.RaError):
        ra.ra_ipc_export(0x1000)
    with pytest.raises(ra.RaError):
        ra.ra_allreduce_peer([0x1000, 0x2000000], 0, 1024)
    with pytest.raises(ra.RaError):
        ra.ra_ipc_close(0x1000)                       # never opened


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def run_peer_worker(mode, env_extra=None, timeout=600):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join("tests", "_peer_worker.py"), mode]
    env = dict(os.environ, OMP_NUM_THREADS="2")
    env.update(env_extra or {})
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def test_gloo_world2_handle_exchange_and_rank_order():
    r = run_peer_worker("cpu", {"CUDA_VISIBLE_DEVICES": ""})
    assert r.returncode == 0, r.stderr[-3000:]
    assert "PEER_CPU_OK world=2" in r.stdout
