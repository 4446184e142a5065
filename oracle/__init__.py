"""ctypes front-end of the CPU oracle (oracle/qft_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and the
cpu_baseline / --impl reference legs of bench.py.  Nothing under
paper_2606_18981_b200/ imports this package and this package imports nothing
from it.  See the header of qft_oracle.c for what each routine follows in
PAPER.md and for the parity-pin status (all pinned).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "qft_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

GATE_H, GATE_CR, GATE_SWAP = 0, 1, 2
NORM_UNITARY, NORM_NONE, NORM_INV_N = 0, 1, 2


def build(force: bool = False) -> str:
    """Compile liboracle.so with gcc (plain -O2, OpenMP); returns its path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int32)
        lp = ctypes.POINTER(ctypes.c_int64)
        L.orc_max_threads.restype = ctypes.c_int
        L.orc_apply_h.argtypes = [dp, ctypes.c_int, ctypes.c_int]
        L.orc_apply_cr.argtypes = [dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int]
        L.orc_apply_swap.argtypes = [dp, ctypes.c_int, ctypes.c_int, ctypes.c_int]
        L.orc_gate_count.argtypes = [ctypes.c_int, ctypes.c_int]
        L.orc_gate_count.restype = ctypes.c_int64
        L.orc_gate_list.argtypes = [ctypes.c_int, ctypes.c_int, ip, ctypes.c_int64]
        L.orc_gate_list.restype = ctypes.c_int64
        L.orc_run_gates.argtypes = [dp, ctypes.c_int, ip, ctypes.c_int64, ctypes.c_int]
        L.orc_qft.argtypes = [dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int]
        L.orc_qft.restype = ctypes.c_int
        L.orc_naive_dft.argtypes = [dp, dp, ctypes.c_int, ctypes.c_int, ctypes.c_int]
        L.orc_naive_dft.restype = ctypes.c_int
        L.orc_element_turns.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int64, ctypes.c_int64]
        L.orc_element_turns.restype = ctypes.c_double
        L.orc_outputs_at.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                     ctypes.c_int, lp, ctypes.c_int, dp]
        L.orc_outputs_at.restype = ctypes.c_int
        _lib = L
    return _lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _n_of(x: np.ndarray) -> int:
    n = int(x.shape[0]).bit_length() - 1
    if x.ndim != 1 or (1 << n) != x.shape[0]:
        raise ValueError("state must be a 1-D array of 2^n amplitudes")
    return n


def _state(x) -> np.ndarray:
    """Widen any complex input (the same complex64 the GPU gets) to complex128."""
    return np.ascontiguousarray(np.asarray(x), dtype=np.complex128).copy()


def max_threads() -> int:
    return int(lib().orc_max_threads())


def gate_count(n: int, k: int) -> int:
    return int(lib().orc_gate_count(n, k))


def gate_list(n: int, k: int) -> np.ndarray:
    """(ngates, 4) int32 rows {type, q0, q1, m}; see orc_gate_list."""
    ng = gate_count(n, k)
    out = np.zeros((ng, 4), dtype=np.int32)
    got = lib().orc_gate_list(n, k, out.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), ng)
    assert got == ng
    return out


def apply_h(x, t: int) -> np.ndarray:
    s = _state(x)
    lib().orc_apply_h(_dp(s), _n_of(s), t)
    return s


def apply_cr(x, control: int, target: int, m: int, sign: int = -1) -> np.ndarray:
    s = _state(x)
    lib().orc_apply_cr(_dp(s), _n_of(s), control, target, m, sign)
    return s


def apply_swap(x, a: int, b: int) -> np.ndarray:
    s = _state(x)
    lib().orc_apply_swap(_dp(s), _n_of(s), a, b)
    return s


def apply_gate_inplace(s: np.ndarray, gate, sign: int = -1) -> None:
    """One gate {type, q0, q1, m} on a complex128 state, in place (used to time a bounded
    sample of a circuit that is too long to run whole)."""
    assert s.dtype == np.complex128 and s.flags.c_contiguous
    n = _n_of(s)
    ty, q0, q1, m = (int(v) for v in gate)
    if ty == GATE_H:
        lib().orc_apply_h(_dp(s), n, q0)
    elif ty == GATE_CR:
        lib().orc_apply_cr(_dp(s), n, q0, q1, m, sign)
    else:
        lib().orc_apply_swap(_dp(s), n, q0, q1)


def run_gates(x, gates: np.ndarray, sign: int = -1) -> np.ndarray:
    s = _state(x)
    g = np.ascontiguousarray(gates, dtype=np.int32)
    lib().orc_run_gates(_dp(s), _n_of(s), g.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), g.shape[0], sign)
    return s


def qft(x, k: int | None = None, sign: int = -1, norm: int = NORM_UNITARY) -> np.ndarray:
    """The whole path (circuit, swaps, normalisation) on a copy of x, complex128."""
    s = _state(x)
    n = _n_of(s)
    if k is None:
        k = n
    if lib().orc_qft(_dp(s), n, k, sign, norm) != 0:
        raise ValueError("orc_qft: bad arguments")
    return s


def naive_dft(x, sign: int = -1, norm: int = NORM_UNITARY) -> np.ndarray:
    s = _state(x)
    y = np.empty_like(s)
    if lib().orc_naive_dft(_dp(s), _dp(y), _n_of(s), sign, norm) != 0:
        raise ValueError("orc_naive_dft: bad arguments (n <= 16)")
    return y


def element_turns(n: int, k: int, sign: int, K: int, j: int) -> float:
    return float(lib().orc_element_turns(n, k, sign, K, j))


def outputs_at(x, Ks, k: int | None = None, sign: int = -1, norm: int = NORM_UNITARY) -> np.ndarray:
    """Sampled outputs out[K], K in Ks, as plain sums over the whole input."""
    x = np.ascontiguousarray(x)
    n = _n_of(x)
    if k is None:
        k = n
    if x.dtype == np.complex64:
        is_f32 = 1
    else:
        x = np.ascontiguousarray(x, dtype=np.complex128)
        is_f32 = 0
    Ks = np.ascontiguousarray(Ks, dtype=np.int64)
    out = np.zeros(Ks.shape[0], dtype=np.complex128)
    lib().orc_outputs_at(x.ctypes.data_as(ctypes.c_void_p), is_f32, n, k, sign, norm,
                         Ks.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)), Ks.shape[0], _dp(out))
    return out


# ---- the steps either side of the circuit, written out from their definitions ----

def norm_sq(x) -> float:
    """sum_j |x_j|^2 in float64 (the square of scale_in)."""
    a = np.asarray(x, dtype=np.complex128).ravel()
    return float(np.sum(a.real * a.real + a.imag * a.imag))


def encode(x):
    """amplitude encoding; returns (x / scale_in, scale_in) with scale_in = ||x||_2."""
    a = np.asarray(x, dtype=np.complex128).ravel()
    scale_in = float(np.sqrt(norm_sq(a)))
    return a / scale_in, scale_in


def fidelity(a, b) -> float:
    """F = |<a, b>|^2 / (||a||^2 ||b||^2)."""
    a = np.asarray(a, dtype=np.complex128).ravel()
    b = np.asarray(b, dtype=np.complex128).ravel()
    inner = np.sum(np.conj(a) * b)
    return float((inner.real ** 2 + inner.imag ** 2) / (norm_sq(a) * norm_sq(b)))


def leakage(out, k0: int) -> float:
    """top-bin leakage 1 - |out[k0]|^2 / ||out||^2."""
    o = np.asarray(out, dtype=np.complex128).ravel()
    return float(1.0 - (o[k0].real ** 2 + o[k0].imag ** 2) / norm_sq(o))
