"""Sharded state, host-side design: the top g address bits select the rank.

CPU: for g = 1, 2, 3 and every n the default plan (and the deferred-swaps plan) passes the host proof
(qft_plan_shard_check): per pass the ranks' unit ranges tile the pass, local passes keep every rank on its own shard;
the folded schedule has exactly two passes whose tiles span the ranks (first and last), the mid passes are local, and
the bytes over the links are (1 - 2^-g) of a shard each way for those two.
GPU (one device, no kernel waits on another): every rank's share of every pass enqueued one after the other on the same
buffer must give exactly what qft_execute gives, and the oracle's result.
"""
import numpy as np
import pytest

import paper_2606_18981_b200 as qft


@pytest.mark.parametrize("g", [1, 2, 3])
def test_shard_ranges_pass_the_host_proof(g):
    for n in list(range(18, 35)):
        for flags in (0, qft.QFT_FLAG_DEFER_SWAPS):
            p = qft.Plan(n, n, flags=flags)
            qft.qft_plan_shard_check(p.handle, g)
            shard_bytes = 8 << (n - g)
            spanning = 0
            for ps in range(p.num_passes):
                infos = [qft.qft_plan_shard_info(p.handle, ps, r, g) for r in range(1 << g)]
                gin = infos[0]["rank_bits_in_tile"]
                assert all(i["rank_bits_in_tile"] == gin for i in infos)
                for i in infos:
                    assert i["remote_bytes_each_way"] == shard_bytes - (shard_bytes >> gin)
                spanning += gin > 0
            if flags == 0 and p.num_passes == 3 and n >= 28:
                # first and last pass hold the top address bits, the mid pass is local (at smaller n the mid pass's
                # tile takes every free address bit as a passive extra, the top ones included)
                assert spanning == 2, (n, g)
            p.close()


def test_shard_unsupported_cases():
    p = qft.Plan(12, 12)  # one tile: fewer units than ranks
    with pytest.raises(qft.QftError) as e:
        qft.qft_plan_shard_info(p.handle, 0, 0, 1)
    assert e.value.status == qft.QFT_ERR_UNSUPPORTED
    with pytest.raises(qft.QftError) as e:
        qft.qft_plan_shard_info(p.handle, 0, 2, 1)  # rank out of range
    assert e.value.status == qft.QFT_ERR_INVALID_ARG
    p.close()


@pytest.mark.gpu
@pytest.mark.parametrize("n,g,flags,k", [(20, 1, 0, None), (22, 3, 0, None), (24, 2, 0, 5), (25, 3, 0, None),
                                         (26, 3, 0, None), (26, 2, 32, None), (21, 2, 0, 0)])
def test_ranks_shares_one_after_the_other_equal_the_whole_pass(n, g, flags, k):
    import torch

    import oracle
    import qft_inputs as qi
    from parity_bounds import assert_parity_numpy

    x = qi.gaussian(n, 300 + n)
    kk = n if k is None else k
    plan = qft.Plan(n, kk, flags=flags)
    whole = torch.from_numpy(x).cuda()
    plan.execute(whole)
    parts = torch.from_numpy(x).cuda()
    s = torch.cuda.current_stream().cuda_stream
    order = list(range(1 << g))
    for ps in range(plan.num_passes):
        order = order[1:] + order[:1]  # any order of the ranks within a pass
        for r in order:
            qft.qft_execute_pass_shard(plan.handle, ps, parts.data_ptr(), r, g, s)
    torch.cuda.synchronize()
    assert torch.equal(torch.view_as_real(whole), torch.view_as_real(parts))
    if flags == 0 and n <= 24:
        assert_parity_numpy(parts.cpu().numpy().astype(np.complex128), oracle.qft(x, kk), n, (n, g, kk))
    plan.close()


_FD_WORKER = """
import os, sys, tempfile
sys.path.insert(0, sys.argv[4])
from paper_2606_18981_b200.sharded import exchange_fds
rank, world, job = int(sys.argv[1]), int(sys.argv[2]), sys.argv[3]
f = tempfile.TemporaryFile()
f.write(f"shard of rank {rank}".encode())
f.flush()
fds = exchange_fds(rank, world, f.fileno(), job)
seen = []
for fd in fds:
    # pread: the ranks share each file's offset (one open file description behind every copy of the descriptor)
    seen.append(os.pread(fd, 64, 0).decode())
print("|".join(seen))
"""


@pytest.mark.parametrize("world", [2, 4])
def test_file_descriptor_exchange_between_processes(world):
    """The host side of the multi-process driver (paper_2606_18981_b200/sharded.py): every rank ends up with every
    rank's descriptor (here: of temporary files; on a GPU node: of the shards' cuMemCreate handles)."""
    import os
    import subprocess
    import sys

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    job = f"test{os.getpid()}_{world}"
    procs = [subprocess.Popen([sys.executable, "-c", _FD_WORKER, str(r), str(world), job, root], stdout=subprocess.PIPE,
                              stderr=subprocess.PIPE, text=True) for r in range(world)]
    want = "|".join(f"shard of rank {r}" for r in range(world))
    for r, p in enumerate(procs):
        out, err = p.communicate(timeout=180)
        assert p.returncode == 0, err[-2000:]
        assert out.strip() == want, (r, out)


@pytest.mark.gpu
@pytest.mark.parametrize("n,g,k", [(24, 1, None), (24, 2, None), (26, 3, 7)])
def test_shards_as_separate_allocations_mapped_back_to_back(n, g, k):
    """LocalShards: 2^g physical allocations (cuMemCreate) on this one device, mapped into one virtual range
    (cuMemAddressReserve / cuMemMap / cuMemSetAccess) exactly as the multi-process driver maps its peers' shards; every
    rank's share of every pass, one after the other.  Same result as qft_execute on an ordinary buffer, bit for bit."""
    import torch
    from cuda.bindings import driver as cu

    import qft_inputs as qi
    from paper_2606_18981_b200.sharded import LocalShards

    x = qi.gaussian(n, 500 + n)
    t = torch.from_numpy(x).cuda()
    plan = qft.Plan(n, n if k is None else k)
    ref = t.clone()
    plan.execute(ref)
    torch.cuda.synchronize()
    sh = LocalShards(n, g, device=torch.cuda.current_device(), aqft_cutoff_k=k)
    assert sh.map.world == 1 << g and sh.map.shard_bytes == 8 << (n - g)
    (err,) = cu.cuMemcpy(sh.map.base, t.data_ptr(), 8 << n)
    assert err == cu.CUresult.CUDA_SUCCESS
    sh.execute(torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    out = torch.empty_like(t)
    (err,) = cu.cuMemcpy(out.data_ptr(), sh.map.base, 8 << n)
    assert err == cu.CUresult.CUDA_SUCCESS
    torch.cuda.synchronize()
    assert torch.equal(torch.view_as_real(out), torch.view_as_real(ref))
    sh.close()
    plan.close()


def test_fd_exchange_drops_bogus_senders_and_refuses_a_shared_directory(tmp_path):
    """exchange_fds keeps one descriptor per peer rank and only from a well-formed first message: a sender
    naming a rank out of range, the receiver's own rank, or a rank already heard is dropped and its descriptor closed;
    the socket directory must be private to this user."""
    import array
    import os
    import socket
    import tempfile
    import threading
    import time

    from paper_2606_18981_b200.sharded import _job_dir, exchange_fds

    job = f"bogus{os.getpid()}"
    files = [tempfile.TemporaryFile() for _ in range(3)]
    for i, f in enumerate(files):
        f.write(f"file {i}".encode())
        f.flush()
    res = {}

    def run(rank):
        res[rank] = exchange_fds(rank, 2, files[rank].fileno(), job, sock_dir=str(tmp_path), timeout=60.0)

    t0 = threading.Thread(target=run, args=(0,))
    t0.start()
    sock0 = os.path.join(str(tmp_path), f"qft_shards_{os.getuid()}_{job}", "0.sock")
    for _ in range(2000):
        if os.path.exists(sock0):
            break
        time.sleep(0.005)
    for claimed in (7, 0, 0xFFFFFFFF):  # out of range, the receiver's own rank, garbage
        c = socket.socket(socket.AF_UNIX, socket.SOCK_STREAM)
        c.connect(sock0)
        c.sendmsg([claimed.to_bytes(4, "little")], [(socket.SOL_SOCKET, socket.SCM_RIGHTS, array.array("i", [files[2].fileno()]))])
        c.close()
    t1 = threading.Thread(target=run, args=(1,))
    t1.start()
    t0.join(90)
    t1.join(90)
    assert not t0.is_alive() and not t1.is_alive()
    assert res[0][0] == files[0].fileno() and res[1][1] == files[1].fileno()
    assert os.pread(res[0][1], 64, 0) == b"file 1" and os.pread(res[1][0], 64, 0) == b"file 0"
    os.close(res[0][1])
    os.close(res[1][0])
    assert not os.path.exists(os.path.dirname(sock0))  # the last rank out removed the directory

    shared = tmp_path / f"qft_shards_{os.getuid()}_open"
    shared.mkdir()
    os.chmod(shared, 0o777)
    with pytest.raises(PermissionError):
        _job_dir(str(tmp_path), "open")
    with pytest.raises(ValueError):
        exchange_fds(2, 2, files[0].fileno(), job, sock_dir=str(tmp_path))
