"""Sharded state across the GPUs of one NVSwitch node ("scale with distributed
simulators").  Host-side driver around the C ABI's sharding calls; DESIGN.md section 9 has the design.

One process per GPU.  The 2^n amplitudes live on 2^g ranks, the top g address bits select the rank.  Every rank
allocates its shard with the virtual-memory-management API (cuMemCreate), exports it as a POSIX file descriptor, and
maps ALL shards back to back into one virtual range of its own (cuMemAddressReserve / cuMemMap / cuMemSetAccess: peer
memory over NVLink), so that every pass is the single-GPU kernel on the same addresses:

    for p in passes:   qft_execute_pass_shard(plan, p, base, rank, g, stream);  stream sync;  barrier over the ranks

A pass whose tiles hold no rank bit touches only the rank's own shard; a pass whose tiles hold the rank bits reads and
writes its peers' shards directly from the kernel (TMA loads, plain stores): the exchange is fused into the pass, there
is no collective on the data path.  The barrier is whatever the caller passes (torch.distributed.barrier with NCCL).

Tested on a single GPU only: `LocalShards` (all shards on one device, the ranks' shares enqueued one after the other),
the file-descriptor exchange between processes on the CPU, and `ShardedQft` itself as 1, 2 and 4 processes that all use
the one GPU (each creates, exports, imports and maps real shards and runs its share of every pass between barriers:
tests/test_sharded.py).  NOT run on more than one GPU: nothing here has seen a peer mapping over NVLink, and no time was
taken.  PyTorch is not needed here; the driver API comes from cuda-python.
"""
from __future__ import annotations

import array
import os
import socket
import time

from . import Plan, qft_execute_pass_shard, qft_plan_shard_check

__all__ = ["ShardMap", "LocalShards", "ShardedQft", "exchange_fds"]


def _cu():
    from cuda.bindings import driver as cu

    return cu


def _check(res, what):
    """cuda-python returns (CUresult, value...) tuples."""
    cu = _cu()
    if res[0] != cu.CUresult.CUDA_SUCCESS:
        raise RuntimeError(f"{what}: {res[0]}")
    return None if len(res) == 1 else (res[1] if len(res) == 2 else res[1:])


def _ensure_context(device: int):
    """The driver API calls below need an initialised driver and the device's primary context current."""
    cu = _cu()
    _check(cu.cuInit(0), "cuInit")
    dev = _check(cu.cuDeviceGet(device), "cuDeviceGet")
    ctx = _check(cu.cuDevicePrimaryCtxRetain(dev), "cuDevicePrimaryCtxRetain")
    _check(cu.cuCtxSetCurrent(ctx), "cuCtxSetCurrent")


def _alloc_prop(device: int):
    cu = _cu()
    prop = cu.CUmemAllocationProp()
    prop.type = cu.CUmemAllocationType.CU_MEM_ALLOCATION_TYPE_PINNED
    prop.location.type = cu.CUmemLocationType.CU_MEM_LOCATION_TYPE_DEVICE
    prop.location.id = device
    prop.requestedHandleTypes = cu.CUmemAllocationHandleType.CU_MEM_HANDLE_TYPE_POSIX_FILE_DESCRIPTOR
    return prop


def granularity(device: int) -> int:
    cu = _cu()
    return int(_check(cu.cuMemGetAllocationGranularity(_alloc_prop(device), cu.CUmemAllocationGranularity_flags.CU_MEM_ALLOC_GRANULARITY_RECOMMENDED),
                      "cuMemGetAllocationGranularity"))


class ShardMap:
    """`world` physical allocations of `shard_bytes` each, mapped back to back into one virtual range that the device
    `device` may read and write.  `handles[r]` is a CUmemGenericAllocationHandle (own shard: created here; peers':
    imported from their file descriptors)."""

    def __init__(self, shard_bytes: int, handles, device: int):
        cu = _cu()
        self.shard_bytes = shard_bytes
        self.world = len(handles)
        self.handles = list(handles)
        total = shard_bytes * self.world
        self.total = total
        self.base = 0
        mapped = 0  # shards mapped so far: what a failure half-way has to undo
        try:
            self.base = int(_check(cu.cuMemAddressReserve(total, granularity(device), 0, 0), "cuMemAddressReserve"))
            for r, h in enumerate(self.handles):
                _check(cu.cuMemMap(self.base + r * shard_bytes, shard_bytes, 0, h, 0), "cuMemMap")
                mapped = r + 1
            acc = cu.CUmemAccessDesc()
            acc.location.type = cu.CUmemLocationType.CU_MEM_LOCATION_TYPE_DEVICE
            acc.location.id = device
            acc.flags = cu.CUmemAccess_flags.CU_MEM_ACCESS_FLAGS_PROT_READWRITE
            _check(cu.cuMemSetAccess(self.base, total, [acc], 1), "cuMemSetAccess")
        except BaseException:
            # the map takes ownership of the handles: release them, the mappings made so far and the reservation
            if self.base:
                if mapped:
                    cu.cuMemUnmap(self.base, mapped * shard_bytes)
                cu.cuMemAddressFree(self.base, total)
                self.base = 0
            for h in self.handles:
                cu.cuMemRelease(h)
            self.handles = []
            raise

    def shard_ptr(self, rank: int) -> int:
        return self.base + rank * self.shard_bytes

    def close(self):
        cu = _cu()
        if self.base:
            cu.cuMemUnmap(self.base, self.total)
            cu.cuMemAddressFree(self.base, self.total)
            for h in self.handles:
                cu.cuMemRelease(h)
            self.base = 0


def create_shard(shard_bytes: int, device: int):
    """One physical allocation on `device`; returns (handle, file descriptor to hand to the peers)."""
    cu = _cu()
    g = granularity(device)
    if shard_bytes % g:
        raise ValueError(f"shard of {shard_bytes} bytes is not a multiple of the allocation granularity {g}")
    h = _check(cu.cuMemCreate(shard_bytes, _alloc_prop(device), 0), "cuMemCreate")
    fd = _check(cu.cuMemExportToShareableHandle(h, cu.CUmemAllocationHandleType.CU_MEM_HANDLE_TYPE_POSIX_FILE_DESCRIPTOR, 0),
                "cuMemExportToShareableHandle")
    return h, int(fd)


def import_shard(fd: int):
    cu = _cu()
    return _check(cu.cuMemImportFromShareableHandle(fd, cu.CUmemAllocationHandleType.CU_MEM_HANDLE_TYPE_POSIX_FILE_DESCRIPTOR),
                  "cuMemImportFromShareableHandle")


def _job_dir(sock_dir: str, job: str) -> str:
    """The directory that holds this job's sockets: <sock_dir>/qft_shards_<uid>_<job>, mode 0700, owned by this user.
    Every rank of the job computes the same name; whoever comes first creates it.  A directory of that name that
    belongs to somebody else, or that others may write to, is refused: descriptors are not handed to strangers."""
    d = os.path.join(sock_dir, f"qft_shards_{os.getuid()}_{job}")
    try:
        os.mkdir(d, 0o700)
    except FileExistsError:
        pass
    st = os.lstat(d)
    import stat as _stat

    if not _stat.S_ISDIR(st.st_mode) or st.st_uid != os.getuid() or (st.st_mode & 0o077):
        raise PermissionError(f"{d} is not a private directory of uid {os.getuid()}")
    return d


def _peer_uid(conn) -> int:
    import struct

    cred = conn.getsockopt(socket.SOL_SOCKET, socket.SO_PEERCRED, struct.calcsize("3i"))
    _pid, uid, _gid = struct.unpack("3i", cred)
    return uid


def exchange_fds(rank: int, world: int, fd: int, job: str, sock_dir: str = "/tmp", timeout: float = 120.0):
    """All-to-all of one file descriptor per rank between the processes of one node, over Unix-domain sockets
    (SCM_RIGHTS).  Returns the list of descriptors indexed by rank (own entry = `fd`).  Pure host code: no CUDA.
    The sockets live in a 0700 directory of this user (_job_dir); a message counts only if its sender runs under this
    user (SO_PEERCRED), names a rank in range other than our own, and is the first from that rank.  Anything else is
    dropped (its descriptors closed) and the wait goes on until every rank has been heard or `timeout` expires."""
    if not (0 <= rank < world):
        raise ValueError(f"rank {rank} outside 0..{world - 1}")
    d = _job_dir(sock_dir, job)
    path = lambda r: os.path.join(d, f"{r}.sock")
    srv = socket.socket(socket.AF_UNIX, socket.SOCK_STREAM)
    try:
        os.unlink(path(rank))
    except FileNotFoundError:
        pass
    srv.bind(path(rank))
    srv.listen(world)
    fds = [None] * world
    fds[rank] = fd
    try:
        # send to everybody (a connection only needs the peer's socket to exist: the message waits in its backlog), then
        # collect one message from everybody
        for peer in range(world):
            if peer == rank:
                continue
            deadline = time.time() + timeout
            while True:
                c = socket.socket(socket.AF_UNIX, socket.SOCK_STREAM)
                try:
                    c.connect(path(peer))
                    break
                except (FileNotFoundError, ConnectionRefusedError):
                    c.close()
                    if time.time() > deadline:
                        raise TimeoutError(f"rank {rank}: peer {peer} did not open its socket")
                    time.sleep(0.01)
            c.sendmsg([rank.to_bytes(4, "little")], [(socket.SOL_SOCKET, socket.SCM_RIGHTS, array.array("i", [fd]))])
            c.close()
        deadline = time.time() + timeout
        while any(f is None for f in fds):
            left = deadline - time.time()
            if left <= 0:
                raise TimeoutError(f"rank {rank}: no descriptor from ranks {[r for r, f in enumerate(fds) if f is None]}")
            srv.settimeout(left)
            try:
                conn, _addr = srv.accept()
            except socket.timeout:
                continue
            try:
                conn.settimeout(max(left, 0.1))
                uid = _peer_uid(conn)
                msg, anc, _flags, _a = conn.recvmsg(4, socket.CMSG_LEN(4))
                got = array.array("i")
                for level, ctype, data in anc:
                    if level == socket.SOL_SOCKET and ctype == socket.SCM_RIGHTS:
                        got.frombytes(data[: len(data) - (len(data) % got.itemsize)])
                src = int.from_bytes(msg, "little") if len(msg) == 4 else -1
                if uid == os.getuid() and 0 <= src < world and src != rank and fds[src] is None and len(got) == 1:
                    fds[src] = int(got[0])
                else:  # a stranger, a duplicate, a malformed message: not ours to keep
                    for g in got:
                        os.close(g)
            except (socket.timeout, OSError):
                pass
            finally:
                conn.close()
    except BaseException:
        for r, f in enumerate(fds):
            if r != rank and f is not None:
                os.close(f)
        raise
    finally:
        srv.close()
        try:
            os.unlink(path(rank))
        except FileNotFoundError:
            pass
        try:
            os.rmdir(d)  # the last rank out removes the directory; the others find it non-empty
        except OSError:
            pass
    return fds


class _Driver:
    """The pass loop shared by the two front ends."""

    def __init__(self, n_qubits: int, log2_ranks: int, **plan_kw):
        self.n = n_qubits
        self.g = log2_ranks
        k = plan_kw.pop("aqft_cutoff_k", None)
        self.plan = Plan(n_qubits, n_qubits if k is None else k, **plan_kw)
        qft_plan_shard_check(self.plan.handle, log2_ranks)  # ranges tile every pass, local passes stay at home


class LocalShards(_Driver):
    """All 2^g shards on ONE device, as separate physical allocations mapped back to back: the sharded path without the
    second GPU.  `execute` enqueues the ranks' shares of every pass one after the other."""

    def __init__(self, n_qubits: int, log2_ranks: int, device: int = 0, **plan_kw):
        super().__init__(n_qubits, log2_ranks, **plan_kw)
        _ensure_context(device)
        shard_bytes = 8 << (n_qubits - log2_ranks)
        handles = []
        for _ in range(1 << log2_ranks):
            h, fd = create_shard(shard_bytes, device)
            os.close(fd)
            handles.append(h)
        self.map = ShardMap(shard_bytes, handles, device)

    def execute(self, stream: int = 0):
        for p in range(self.plan.num_passes):
            for r in range(1 << self.g):
                qft_execute_pass_shard(self.plan.handle, p, self.map.base, r, self.g, stream)

    def close(self):
        self.map.close()
        self.plan.close()


class ShardedQft(_Driver):
    """One rank of the multi-process driver.  `barrier()` must synchronise all ranks (e.g. torch.distributed.barrier);
    `job` names the Unix sockets of this job (e.g. MASTER_PORT)."""

    def __init__(self, n_qubits: int, rank: int, world: int, device: int, barrier, job: str, **plan_kw):
        g = world.bit_length() - 1
        if world != 1 << g:
            raise ValueError("the number of ranks must be a power of two")
        super().__init__(n_qubits, g, **plan_kw)
        self.rank, self.world, self.barrier = rank, world, barrier
        _ensure_context(device)
        shard_bytes = 8 << (n_qubits - g)
        own, fd = create_shard(shard_bytes, device)
        fds = exchange_fds(rank, world, fd, job)
        handles = [own if r == rank else import_shard(fds[r]) for r in range(world)]
        for f in fds:
            os.close(f)
        self.map = ShardMap(shard_bytes, handles, device)
        barrier()

    @property
    def shard_ptr(self) -> int:
        return self.map.shard_ptr(self.rank)

    def execute(self, stream: int = 0):
        cu = _cu()
        for p in range(self.plan.num_passes):
            qft_execute_pass_shard(self.plan.handle, p, self.map.base, self.rank, self.g, stream)
            _check(cu.cuStreamSynchronize(cu.CUstream(stream)), "cuStreamSynchronize")  # this rank's stores are done ...
            self.barrier()                                                  # ... and so are everybody else's

    def close(self):
        self.barrier()
        self.map.close()
        self.plan.close()
