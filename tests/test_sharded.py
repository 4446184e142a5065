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


@pytest.mark.gpu
@pytest.mark.parametrize("n,g,kw", [(28, 1, {}), (27, 2, {"tile_bits": 14, "hub_bits": 6})])
def test_ranks_shares_on_extended_tiles(n, g, kw):
    """The tensor-memory extended-tile kernel's rank-share walk (unit_lo offset plus the half bit as the last tile-index
    bit): default plans have such passes only from n = 28, the tuned n = 27 plan is made of them entirely.
    Every rank's share of every pass, one after the other on one buffer, is qft_execute bit for bit."""
    import torch

    import qft_inputs as qi

    plan = qft.Plan(n, n, **kw)
    kinds = [p["kernel"] for p in plan.describe()["passes"]]
    assert "tma2x" in kinds, kinds
    whole = qi.gaussian_device(n, 700 + n, device="cuda")
    parts = whole.clone()
    plan.execute(whole)
    s = torch.cuda.current_stream().cuda_stream
    order = list(range(1 << g))
    for ps in range(plan.num_passes):
        order = order[1:] + order[:1]
        for r in order:
            qft.qft_execute_pass_shard(plan.handle, ps, parts.data_ptr(), r, g, s)
    torch.cuda.synchronize()
    assert torch.equal(torch.view_as_real(whole), torch.view_as_real(parts))
    plan.close()


_RANK_WORKER = """
import os, sys, time
rank, world, n, job, root, out = int(sys.argv[1]), int(sys.argv[2]), int(sys.argv[3]), sys.argv[4], sys.argv[5], sys.argv[6]
sys.path.insert(0, root)
import numpy as np
from cuda.bindings import driver as cu
import qft_inputs as qi
from paper_2606_18981_b200.sharded import ShardedQft


class FileBarrier:
    # test infrastructure: a barrier over the ranks' processes through files in a directory they share
    def __init__(self):
        self.i = 0

    def __call__(self):
        open(os.path.join(out, f"b{self.i}_{rank}"), "w").close()
        deadline = time.time() + 120
        while not all(os.path.exists(os.path.join(out, f"b{self.i}_{r}")) for r in range(world)):
            if time.time() > deadline:
                raise TimeoutError(f"rank {rank}: barrier {self.i}")
            time.sleep(0.0005)
        self.i += 1


barrier = FileBarrier()
sq = ShardedQft(n, rank, world, 0, barrier, job)   # every rank on device 0: the one GPU there is
S = (1 << n) // world
x = qi.gaussian(n, 900 + n)[rank * S:(rank + 1) * S].copy()
(err,) = cu.cuMemcpyHtoD(sq.shard_ptr, x, x.nbytes)
assert err == cu.CUresult.CUDA_SUCCESS, err
(err,) = cu.cuCtxSynchronize()
assert err == cu.CUresult.CUDA_SUCCESS, err
barrier()                                           # every shard holds its input before any pass reads a peer's
sq.execute(0)
y = np.empty_like(x)
(err,) = cu.cuMemcpyDtoH(y, sq.shard_ptr, y.nbytes)
assert err == cu.CUresult.CUDA_SUCCESS, err
np.save(os.path.join(out, f"shard_{rank}.npy"), y)
info = [sq.map.world, sq.map.shard_bytes, sq.plan.num_passes]
sq.close()
print("ok", *info)
"""


@pytest.mark.gpu
@pytest.mark.parametrize("world", [1, 2, 4])
def test_multi_process_driver_on_one_gpu(world, tmp_path):
    """ShardedQft as it is meant to run - one process per rank - with every rank on the one GPU of this box: each
    process creates its shard (cuMemCreate), exports it as a file descriptor, receives its peers' descriptors over the
    Unix sockets, imports and maps all shards back to back, runs its share of every pass (TMA loads and plain stores
    through the imported mappings) and meets the others at a barrier between passes.  The assembled result equals
    qft_execute on an ordinary buffer bit for bit and the oracle within the parity bounds.  (world = 1: the class at
    g = 0 with nothing to exchange.)  This exercises the cross-process handle exchange and mapping; it says nothing
    about NVLink, and no timing is taken."""
    import os
    import subprocess
    import sys

    import torch

    import oracle
    import qft_inputs as qi
    from parity_bounds import assert_parity_numpy

    n = 24
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    job = f"mp{os.getpid()}_{world}"
    procs = [subprocess.Popen([sys.executable, "-c", _RANK_WORKER, str(r), str(world), str(n), job, root, str(tmp_path)],
                              stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True) for r in range(world)]
    try:
        for r, p in enumerate(procs):
            out, err = p.communicate(timeout=300)
            assert p.returncode == 0, (r, err[-3000:])
            assert out.split() == ["ok", str(world), str((8 << n) // world), "3"], out
    finally:
        for p in procs:
            if p.poll() is None:
                p.kill()
    got = np.concatenate([np.load(os.path.join(str(tmp_path), f"shard_{r}.npy")) for r in range(world)])
    x = qi.gaussian(n, 900 + n)
    t = torch.from_numpy(x).cuda()
    plan = qft.Plan(n, n)
    plan.execute(t)
    torch.cuda.synchronize()
    plan.close()
    assert np.array_equal(got.view(np.float32), t.cpu().numpy().view(np.float32))
    assert_parity_numpy(got.astype(np.complex128), oracle.qft(x), n, ("multi-process", world))
