"""Thin Python binding of libqft.so (include/qft.h): argument marshalling only.

Every step of the path (planning, kernels, copies) runs inside the C-ABI
library; PyTorch appears only in callers, for device memory and streams.  There
is no CPU fallback: if libqft.so cannot be loaded (and cannot be built because
nvcc is missing) importing a symbol raises RuntimeError.

Names mirror the C ABI: qft_plan_create, qft_execute, qft_execute_host,
qft_plan_destroy, qft_plan_num_passes, qft_plan_num_launches,
qft_plan_gate_counts, qft_plan_describe, qft_plan_self_check,
qft_status_string.  `Plan` is a small RAII convenience around them.
"""
from __future__ import annotations

import ctypes
import json
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libqft.so")

QFT_OK, QFT_ERR_INVALID_ARG, QFT_ERR_UNSUPPORTED, QFT_ERR_ALLOC, QFT_ERR_CUDA, QFT_ERR_INTERNAL = range(6)
QFT_NORM_UNITARY, QFT_NORM_NONE, QFT_NORM_INV_N = 0, 1, 2
QFT_FLAG_GENERIC_ONLY, QFT_FLAG_UNFOLDED, QFT_FLAG_NO_TMA, QFT_FLAG_NO_EXT_TILE, QFT_FLAG_DEFER_SWAPS = 1, 2, 4, 16, 32
QFT_MAX_QUBITS = 34
QFT_STATIC_MAX_BATCH = 4096  # states per qft_fidelity_batched_static call (its built-in 128 KiB scratch array)

EXPORTS = [
    "qft_plan_create", "qft_plan_create_batched", "qft_plan_create_tuned", "qft_execute", "qft_execute_pass", "qft_execute_host", "qft_plan_destroy",
    "qft_plan_num_passes", "qft_plan_num_launches", "qft_plan_gate_counts", "qft_plan_describe",
    "qft_plan_describe_length", "qft_num_qubits_for", "qft_encode_padded", "qft_execute_oop", "qft_plan_output_order",
    "qft_plan_self_check", "qft_status_string", "qft_last_cuda_error",
    "qft_plan_shard_info", "qft_plan_shard_check", "qft_execute_pass_shard",
    "qft_norm_sq", "qft_encode", "qft_rescale", "qft_fidelity", "qft_leakage",
    "qft_fidelity_batched_static", "qft_static_last_error", "qft_tensor_map_fallbacks",
]

_lib = None


class QftError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = qft_status_string(status)
        detail = qft_last_cuda_error()
        super().__init__(f"{where}: {msg}" + (f" ({detail})" if detail else ""))


def load() -> ctypes.CDLL:
    """Load libqft.so; build it first if it is missing and nvcc is available."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        try:
            from . import build as _build

            _build.build()
        except Exception as exc:  # no nvcc, compile error ...
            raise RuntimeError(
                f"libqft.so is missing at {LIB_PATH} and could not be built ({exc}); "
                "there is no CPU fallback for the QFT path") from exc
    L = ctypes.CDLL(LIB_PATH)
    vp, ci = ctypes.c_void_p, ctypes.c_int
    L.qft_plan_create.argtypes = [ctypes.POINTER(vp), ci, ci, ci, ci, ci]
    L.qft_plan_create.restype = ci
    L.qft_plan_create_batched.argtypes = [ctypes.POINTER(vp), ci, ci, ci, ci, ci, ci]
    L.qft_plan_create_batched.restype = ci
    L.qft_plan_create_tuned.argtypes = [ctypes.POINTER(vp), ci, ci, ci, ci, ci, ci, ci, ctypes.c_uint]
    L.qft_plan_create_tuned.restype = ci
    L.qft_execute.argtypes = [vp, vp, vp]
    L.qft_execute.restype = ci
    L.qft_execute_oop.argtypes = [vp, vp, vp, vp]
    L.qft_execute_oop.restype = ci
    L.qft_plan_output_order.argtypes = [vp, ctypes.POINTER(ci)]
    L.qft_plan_output_order.restype = ci
    L.qft_execute_pass.argtypes = [vp, ci, vp, vp]
    L.qft_execute_pass.restype = ci
    L.qft_plan_shard_info.argtypes = [vp, ci, ci, ci, ctypes.POINTER(ctypes.c_longlong), ctypes.POINTER(ctypes.c_longlong),
                                      ctypes.POINTER(ci), ctypes.POINTER(ctypes.c_longlong)]
    L.qft_plan_shard_info.restype = ci
    L.qft_plan_shard_check.argtypes = [vp, ci]
    L.qft_plan_shard_check.restype = ci
    L.qft_execute_pass_shard.argtypes = [vp, ci, vp, ci, ci, vp]
    L.qft_execute_pass_shard.restype = ci
    L.qft_execute_host.argtypes = [vp, vp, vp]
    L.qft_execute_host.restype = ci
    L.qft_plan_destroy.argtypes = [vp]
    L.qft_plan_destroy.restype = ci
    L.qft_plan_num_passes.argtypes = [vp]
    L.qft_plan_num_passes.restype = ci
    L.qft_plan_num_launches.argtypes = [vp]
    L.qft_plan_num_launches.restype = ci
    llp = ctypes.POINTER(ctypes.c_longlong)
    L.qft_plan_gate_counts.argtypes = [vp, llp, llp, llp]
    L.qft_plan_gate_counts.restype = ci
    L.qft_plan_describe.argtypes = [vp, ctypes.c_char_p, ctypes.c_size_t]
    L.qft_plan_describe.restype = ci
    L.qft_plan_describe_length.argtypes = [vp]
    L.qft_plan_describe_length.restype = ctypes.c_size_t
    L.qft_num_qubits_for.argtypes = [ctypes.c_ulonglong]
    L.qft_num_qubits_for.restype = ci
    L.qft_encode_padded.argtypes = [vp, ci, vp, ctypes.c_ulonglong, ctypes.POINTER(ctypes.c_double), vp]
    L.qft_encode_padded.restype = ci
    L.qft_plan_self_check.argtypes = [vp]
    L.qft_plan_self_check.restype = ci
    L.qft_status_string.argtypes = [ci]
    L.qft_status_string.restype = ctypes.c_char_p
    dp = ctypes.POINTER(ctypes.c_double)
    L.qft_norm_sq.argtypes = [vp, ci, dp, vp]
    L.qft_encode.argtypes = [vp, ci, dp, vp]
    L.qft_rescale.argtypes = [vp, ci, ctypes.c_double, vp]
    L.qft_fidelity.argtypes = [vp, vp, ci, dp, vp]
    L.qft_leakage.argtypes = [vp, ci, ctypes.c_ulonglong, dp, vp]
    for _f in (L.qft_norm_sq, L.qft_encode, L.qft_rescale, L.qft_fidelity, L.qft_leakage):
        _f.restype = ci
    L.qft_last_cuda_error.argtypes = []
    L.qft_last_cuda_error.restype = ctypes.c_char_p
    L.qft_fidelity_batched_static.argtypes = [vp, vp, ci, ci, vp, vp]
    L.qft_fidelity_batched_static.restype = ci
    L.qft_tensor_map_fallbacks.argtypes = []
    L.qft_tensor_map_fallbacks.restype = ctypes.c_ulonglong
    L.qft_static_last_error.argtypes = []
    L.qft_static_last_error.restype = ctypes.c_char_p
    _lib = L
    return L


# ---- one-to-one wrappers (raise QftError on a non-zero status) ---------------------------------

def qft_status_string(status: int) -> str:
    return load().qft_status_string(int(status)).decode()


def qft_last_cuda_error() -> str:
    return load().qft_last_cuda_error().decode()


def qft_plan_create(n_qubits: int, aqft_cutoff_k: int, max_fused_qubits: int = 13, sign: int = -1,
                    normalisation: int = QFT_NORM_UNITARY) -> int:
    h = ctypes.c_void_p()
    st = load().qft_plan_create(ctypes.byref(h), n_qubits, aqft_cutoff_k, max_fused_qubits, sign, normalisation)
    if st != QFT_OK:
        raise QftError(st, "qft_plan_create")
    return h.value


def qft_plan_create_batched(n_qubits: int, log2_batch: int, aqft_cutoff_k: int, max_fused_qubits: int = 13,
                            sign: int = -1, normalisation: int = QFT_NORM_UNITARY) -> int:
    h = ctypes.c_void_p()
    st = load().qft_plan_create_batched(ctypes.byref(h), n_qubits, log2_batch, aqft_cutoff_k, max_fused_qubits, sign,
                                        normalisation)
    if st != QFT_OK:
        raise QftError(st, "qft_plan_create_batched")
    return h.value


def qft_plan_create_tuned(n_qubits: int, aqft_cutoff_k: int, max_fused_qubits: int = 13, sign: int = -1,
                          normalisation: int = QFT_NORM_UNITARY, tile_bits: int = 0, hub_bits: int = 0,
                          flags: int = 0) -> int:
    h = ctypes.c_void_p()
    st = load().qft_plan_create_tuned(ctypes.byref(h), n_qubits, aqft_cutoff_k, max_fused_qubits, sign,
                                      normalisation, tile_bits, hub_bits, flags)
    if st != QFT_OK:
        raise QftError(st, "qft_plan_create_tuned")
    return h.value


def qft_execute(plan: int, device_state_ptr: int, stream: int = 0) -> None:
    st = load().qft_execute(plan, device_state_ptr, stream)
    if st != QFT_OK:
        raise QftError(st, "qft_execute")


def qft_execute_oop(plan: int, device_in_ptr: int, device_out_ptr: int, stream: int = 0) -> None:
    st = load().qft_execute_oop(plan, device_in_ptr, device_out_ptr, stream)
    if st != QFT_OK:
        raise QftError(st, "qft_execute_oop")


def qft_plan_output_order(plan: int, n_qubits: int | None = None):
    """qubit_of_bit[a] for a < n.  The C call writes the plan's own n entries whatever the caller believes n to be,
    so the buffer always has room for QFT_MAX_QUBITS and n is read from the plan; a caller-supplied n_qubits that
    disagrees with the plan is an error, not an overrun."""
    arr = (ctypes.c_int * QFT_MAX_QUBITS)()
    st = load().qft_plan_output_order(plan, arr)
    if st != QFT_OK:
        raise QftError(st, "qft_plan_output_order")
    n = int(qft_plan_describe(plan)["n"])
    if n_qubits is not None and int(n_qubits) != n:
        raise ValueError(f"qft_plan_output_order: the plan has {n} qubits, the caller said {n_qubits}")
    return list(arr)[:n]


def qft_execute_pass(plan: int, pass_index: int, device_state_ptr: int, stream: int = 0) -> None:
    st = load().qft_execute_pass(plan, pass_index, device_state_ptr, stream)
    if st != QFT_OK:
        raise QftError(st, "qft_execute_pass")


def qft_plan_shard_info(plan: int, pass_index: int, rank: int, log2_ranks: int) -> dict:
    lo, cnt, rem, gin = ctypes.c_longlong(), ctypes.c_longlong(), ctypes.c_longlong(), ctypes.c_int()
    st = load().qft_plan_shard_info(plan, pass_index, rank, log2_ranks, ctypes.byref(lo), ctypes.byref(cnt), ctypes.byref(gin),
                                    ctypes.byref(rem))
    if st != QFT_OK:
        raise QftError(st, "qft_plan_shard_info")
    return {"unit_lo": lo.value, "unit_n": cnt.value, "rank_bits_in_tile": gin.value, "remote_bytes_each_way": rem.value}


def qft_plan_shard_check(plan: int, log2_ranks: int) -> None:
    st = load().qft_plan_shard_check(plan, log2_ranks)
    if st != QFT_OK:
        raise QftError(st, "qft_plan_shard_check")


def qft_execute_pass_shard(plan: int, pass_index: int, state_base_ptr: int, rank: int, log2_ranks: int, stream: int = 0) -> None:
    st = load().qft_execute_pass_shard(plan, pass_index, state_base_ptr, rank, log2_ranks, stream)
    if st != QFT_OK:
        raise QftError(st, "qft_execute_pass_shard")


def qft_execute_host(plan: int, host_state_ptr: int, stream: int = 0) -> None:
    st = load().qft_execute_host(plan, host_state_ptr, stream)
    if st != QFT_OK:
        raise QftError(st, "qft_execute_host")


def qft_plan_destroy(plan: int) -> None:
    load().qft_plan_destroy(plan)


def qft_plan_num_passes(plan: int) -> int:
    return int(load().qft_plan_num_passes(plan))


def qft_plan_num_launches(plan: int) -> int:
    return int(load().qft_plan_num_launches(plan))


def qft_plan_gate_counts(plan: int):
    a, b, c = ctypes.c_longlong(), ctypes.c_longlong(), ctypes.c_longlong()
    st = load().qft_plan_gate_counts(plan, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c))
    if st != QFT_OK:
        raise QftError(st, "qft_plan_gate_counts")
    return a.value, b.value, c.value


def qft_plan_describe_length(plan: int) -> int:
    return int(load().qft_plan_describe_length(plan))


def qft_plan_describe(plan: int) -> dict:
    buf = ctypes.create_string_buffer(qft_plan_describe_length(plan))
    st = load().qft_plan_describe(plan, buf, len(buf))
    if st != QFT_OK:
        raise QftError(st, "qft_plan_describe")
    return json.loads(buf.value.decode())


def qft_plan_self_check(plan: int) -> None:
    st = load().qft_plan_self_check(plan)
    if st != QFT_OK:
        raise QftError(st, "qft_plan_self_check")


def _dbl_call(name: str, *args) -> float:
    out = ctypes.c_double()
    fn = getattr(load(), name)
    st = fn(*args[:-1], ctypes.byref(out), args[-1])
    if st != QFT_OK:
        raise QftError(st, name)
    return out.value


def qft_norm_sq(device_state_ptr: int, n_qubits: int, stream: int = 0) -> float:
    return _dbl_call("qft_norm_sq", device_state_ptr, n_qubits, stream)


def qft_encode(device_state_ptr: int, n_qubits: int, stream: int = 0) -> float:
    """Divides the state by its L2 norm in place and returns that norm (scale_in)."""
    return _dbl_call("qft_encode", device_state_ptr, n_qubits, stream)


def qft_num_qubits_for(length: int) -> int:
    return int(load().qft_num_qubits_for(int(length)))


def qft_encode_padded(device_state_ptr: int, n_qubits: int, device_x_ptr: int, length: int, stream: int = 0) -> float:
    """Copies x (length complex64, device) to the front of the 2^n state, zero-fills the rest, normalises; returns scale_in."""
    out = ctypes.c_double()
    st = load().qft_encode_padded(device_state_ptr, n_qubits, device_x_ptr, int(length), ctypes.byref(out), stream)
    if st != QFT_OK:
        raise QftError(st, "qft_encode_padded")
    return out.value


def qft_rescale(device_state_ptr: int, n_qubits: int, factor: float, stream: int = 0) -> None:
    st = load().qft_rescale(device_state_ptr, n_qubits, float(factor), stream)
    if st != QFT_OK:
        raise QftError(st, "qft_rescale")


def qft_fidelity(device_a_ptr: int, device_b_ptr: int, n_qubits: int, stream: int = 0) -> float:
    return _dbl_call("qft_fidelity", device_a_ptr, device_b_ptr, n_qubits, stream)


def qft_leakage(device_state_ptr: int, n_qubits: int, bin_index: int, stream: int = 0) -> float:
    return _dbl_call("qft_leakage", device_state_ptr, n_qubits, int(bin_index), stream)


def qft_tensor_map_fallbacks() -> int:
    """Pass launches of this process that fell back to the generic kernel (tensor map refused); 0 is the expected value."""
    return int(load().qft_tensor_map_fallbacks())


def qft_static_last_error() -> str:
    return load().qft_static_last_error().decode()


def qft_fidelity_batched_static(device_a_ptr: int, device_b_ptr: int, n_qubits: int, batch: int,
                                device_fidelity_out_ptr: int, stream: int = 0) -> None:
    """Fidelity of `batch` pairs of states (complex64[batch * 2^n] each, device) into a device double[batch],
    without any device allocation: for processes whose GPU memory is all spoken for (one big pool, or state
    vectors sized to fill the card) and for loops that cannot take an allocation's stall.  The accumulators are
    a fixed array inside libqft.so, shared by every call on the device: batch <= QFT_STATIC_MAX_BATCH (more
    raises QftError with status QFT_ERR_UNSUPPORTED), and calls that overlap on the GPU race.  Only enqueues;
    the first call on a device also looks the array's address up and should precede any stream capture."""
    st = load().qft_fidelity_batched_static(device_a_ptr, device_b_ptr, int(n_qubits), int(batch),
                                            device_fidelity_out_ptr, stream)
    if st != QFT_OK:
        err = QftError(st, "qft_fidelity_batched_static")
        err.args = (f"{qft_status_string(st)}: {qft_static_last_error()}",)
        raise err


class Plan:
    """RAII wrapper: Plan(n, k).execute(tensor) transforms a CUDA complex64 tensor in place."""

    def __init__(self, n_qubits: int, aqft_cutoff_k: int | None = None, max_fused_qubits: int = 13, sign: int = -1,
                 normalisation: int = QFT_NORM_UNITARY, tile_bits: int = 0, hub_bits: int = 0, flags: int = 0,
                 log2_batch: int = 0):
        if aqft_cutoff_k is None:
            aqft_cutoff_k = n_qubits
        self.n = n_qubits + log2_batch  # address bits of the state this plan transforms
        self.n_qubits = n_qubits
        if log2_batch:
            if tile_bits or hub_bits or flags:
                raise ValueError("the tuning knobs are not available for batched plans")
            self.handle = qft_plan_create_batched(n_qubits, log2_batch, aqft_cutoff_k, max_fused_qubits, sign,
                                                  normalisation)
        else:
            self.handle = qft_plan_create_tuned(n_qubits, aqft_cutoff_k, max_fused_qubits, sign, normalisation,
                                                tile_bits, hub_bits, flags)

    def execute(self, state, stream: int | None = None) -> None:
        """state: torch complex64 CUDA tensor of 2^n elements (contiguous).  In place, asynchronous."""
        import torch

        if state.dtype != torch.complex64 or not state.is_cuda or not state.is_contiguous() or \
                state.numel() != (1 << self.n):
            raise ValueError("state must be a contiguous CUDA complex64 tensor of 2^n elements")
        if stream is None:
            stream = torch.cuda.current_stream(state.device).cuda_stream
        qft_execute(self.handle, state.data_ptr(), stream)

    def execute_oop(self, src, dst, stream: int | None = None) -> None:
        """dst <- transform of src (both CUDA complex64 tensors of 2^n elements); src is left untouched."""
        import torch

        for t in (src, dst):
            if t.dtype != torch.complex64 or not t.is_cuda or not t.is_contiguous() or t.numel() != (1 << self.n):
                raise ValueError("src and dst must be contiguous CUDA complex64 tensors of 2^n elements")
        if stream is None:
            stream = torch.cuda.current_stream(dst.device).cuda_stream
        qft_execute_oop(self.handle, src.data_ptr(), dst.data_ptr(), stream)

    def output_order(self):
        """qubit_of_bit[a] for a < n_qubits (n-1-a unless the plan defers the swaps)."""
        return qft_plan_output_order(self.handle, self.n_qubits)

    def execute_host(self, state, stream: int = 0) -> None:
        """state: numpy complex64 array or CPU torch tensor of 2^n elements; in place, synchronous."""
        if hasattr(state, "data_ptr"):
            ptr, cnt = state.data_ptr(), state.numel()
        else:
            ptr, cnt = state.ctypes.data, state.size
        if cnt != (1 << self.n):
            raise ValueError("state must hold 2^n complex64 elements")
        qft_execute_host(self.handle, ptr, stream)

    @property
    def num_passes(self) -> int:
        return qft_plan_num_passes(self.handle)

    @property
    def num_launches(self) -> int:
        return qft_plan_num_launches(self.handle)

    def gate_counts(self):
        return qft_plan_gate_counts(self.handle)

    def describe(self) -> dict:
        return qft_plan_describe(self.handle)

    def self_check(self) -> None:
        qft_plan_self_check(self.handle)

    def close(self) -> None:
        if getattr(self, "handle", None):
            qft_plan_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
