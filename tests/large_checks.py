"""Checkers for states too large for the CPU oracle (n = 30, 33): test infrastructure only.

Everything here is float64 torch arithmetic that runs on whatever device holds the state (the
8-64 GiB inputs live in HBM), written from closed forms that tests/test_oracle_pins.py and
tests/test_large_checks_cpu.py pin against the gate-by-gate oracle at small n on the CPU:

  sampled_outputs()      out[K] = 2^{-n/2} sum_j x[j] exp(2 pi i turns_k(K, j)), the circuit's matrix
                         element (oracle.orc_element_turns) summed over the whole input:
                         turns_k(K, j) = sign * sum_{t : y_t = 1} tr_{k,t}(j) / 2^{t+1},
                         y_t = bit n-1-t of K, tr_{k,t}(j) = (j mod 2^{t+1}) with bits below t-k
                         cleared.  For k >= n-1 this is the DFT phase sign * (j K mod N) / N.  The
                         phase is linear in the bits of j, so it factors into a low-bits and a
                         high-bits table and the sums for all sampled K are two matrix products.
  tones_closed_form()    AQFT_k of a sum of tones, every output, by factorising over input bits:
                         out[K] = sum_i a_i prod_c (1 + exp(2 pi i alpha_c)) / 2,
                         alpha_c = f_i 2^c / N - field_c(K) / 2^{k+1}.
  norm2()                float64 sum of |x|^2 (Parseval).
None of this is used by the product path.
"""
from __future__ import annotations

import math

import torch


def _chunks(n, chunk_bits):
    cb = min(chunk_bits, n)
    return cb, 1 << cb, 1 << (n - cb)


def norm2(x: torch.Tensor, chunk_bits: int = 26) -> float:
    v = torch.view_as_real(x)
    n = int(x.numel()).bit_length() - 1
    cb, C, nc = _chunks(n, chunk_bits)
    acc = torch.zeros((), dtype=torch.float64, device=x.device)
    for c in range(nc):
        blk = v[c * C:(c + 1) * C].to(torch.float64)
        acc += (blk * blk).sum()
    return float(acc.item())


def _phase_coefficients(n: int, Ks, k: int, sign: int) -> torch.Tensor:
    """c[b, s]: the turns that input bit b contributes to the matrix element <Ks[s]| AQFT_k |j>.

    turns_k(K, j) = sign * sum_{t : y_t = 1} tr_{k,t}(j) / 2^{t+1} is linear in the bits of j: bit b belongs to
    tr_{k,t}(j) iff t - k <= b <= t, so c_b = sign * sum_{t = b}^{min(n-1, b+k)} y_t 2^{b-t-1}, y_t = bit n-1-t
    of K.  Every term is a dyadic rational >= 2^-(k+1): sums of them are exact in float64."""
    c = torch.zeros(n, len(Ks), dtype=torch.float64)
    for s, K in enumerate(Ks):
        K = int(K)
        for b in range(n):
            acc = 0.0
            for t in range(b, min(n - 1, b + k) + 1):
                if (K >> (n - 1 - t)) & 1:
                    acc += 2.0 ** (b - t - 1)
            c[b, s] = sign * acc
    return c


def _cis_turns(turns: torch.Tensor) -> torch.Tensor:
    fr = turns - torch.floor(turns)  # exact: the turns are dyadic rationals well inside float64
    ang = fr * (2.0 * math.pi)
    return torch.complex(torch.cos(ang), torch.sin(ang))


def _bits(idx: torch.Tensor, nbits: int) -> torch.Tensor:
    sh = torch.arange(nbits, dtype=torch.int64, device=idx.device)
    return ((idx[:, None] >> sh[None, :]) & 1).to(torch.float64)


def sampled_outputs(x: torch.Tensor, Ks, k: int, sign: int = -1, chunk_bits: int = 24) -> torch.Tensor:
    """Direct float64 sums for the output indices Ks (unitary scaling); x is the INPUT state.

    out[K] = 2^{-n/2} sum_j x[j] exp(2 pi i turns_k(K, j)).  Because turns_k is linear in the bits of j
    (_phase_coefficients), the phase factorises over j = j_hi 2^h + j_lo into W_hi[j_hi] W_lo[j_lo], so the sum is
    W_hi^T (X W_lo) with X the input seen as a 2^(n-h) x 2^h matrix: one complex128 matrix product per chunk of rows
    for all sampled indices at once.  Exact k (k >= n-1) needs no special case: then c_b = sign K 2^b / N mod 1."""
    N = x.numel()
    n = int(N).bit_length() - 1
    cb, C, nc = _chunks(n, chunk_bits)
    h = min(cb, 12)
    dev = x.device
    c = _phase_coefficients(n, Ks, min(k, n), sign).to(dev)
    lo = torch.arange(1 << h, dtype=torch.int64, device=dev)
    W_lo = _cis_turns(_bits(lo, h) @ c[:h]) if h > 0 else torch.ones(1, len(Ks), dtype=torch.complex128, device=dev)
    R = C >> h  # rows per chunk
    rows = torch.arange(R, dtype=torch.int64, device=dev)
    out = torch.zeros(len(Ks), dtype=torch.complex128, device=dev)
    for ci in range(nc):
        X = x[ci * C:(ci + 1) * C].view(R, 1 << h).to(torch.complex128)
        P = X @ W_lo  # [R, S]
        if n > h:
            W_hi = _cis_turns(_bits(rows + ci * R, n - h) @ c[h:])
            out += (P * W_hi).sum(dim=0)
        else:
            out += P.sum(dim=0)
    return out * (2.0 ** (-0.5 * n))


def tones_closed_form_chunk(n: int, k: int, freqs, phases, K: torch.Tensor) -> torch.Tensor:
    """AQFT_k (forward sign, unitary) of the multi_tone() input at the output indices K (int64)."""
    N = 1 << n
    dev = K.device
    amp = 1.0 / math.sqrt(len(freqs))
    acc = torch.zeros(K.shape, dtype=torch.complex128, device=dev)
    kk = min(k, n - 1)
    for f, th in zip(freqs, phases):
        f = int(f)
        re = torch.full(K.shape, math.cos(float(th)) * amp, dtype=torch.float64, device=dev)
        im = torch.full(K.shape, math.sin(float(th)) * amp, dtype=torch.float64, device=dev)
        for c in range(n):
            top = min(n - 1, c + kk)           # highest target t that sees bit c as a control (or itself)
            width = top - c + 1                 # bits y_c .. y_top = bits n-1-c .. n-1-top of K
            field = (K >> (n - 1 - top)) & ((1 << width) - 1)
            # sum_{t=c..top} y_t 2^{c-t-1}: y_c is the field's most significant bit, weight 1/2
            al = (((f << c) % N) / N) - field.to(torch.float64) * (1.0 / float(1 << width))
            ang = al * (2.0 * math.pi)
            fr = 0.5 * (1.0 + torch.cos(ang))
            fi = 0.5 * torch.sin(ang)
            re, im = re * fr - im * fi, re * fi + im * fr
        acc += torch.complex(re, im)
    return acc


def tones_parity(y: torch.Tensor, n: int, k: int, freqs, phases, chunk_bits: int = 22, index_chunks=None):
    """Distance between the device result y and the closed form, over all outputs or over the listed chunks of
    2^chunk_bits consecutive outputs: (relative L2, sum |ref|^2, max |y - ref|, max |ref|)."""
    cb, C, nc = _chunks(n, chunk_bits)
    dev = y.device
    base = torch.arange(C, dtype=torch.int64, device=dev)
    num = torch.zeros((), dtype=torch.float64, device=dev)
    den = torch.zeros((), dtype=torch.float64, device=dev)
    mx = torch.zeros((), dtype=torch.float64, device=dev)
    rmax = torch.zeros((), dtype=torch.float64, device=dev)
    for c in (range(nc) if index_chunks is None else index_chunks):
        K = base + c * C
        ref = tones_closed_form_chunk(n, k, freqs, phases, K)
        d = y[c * C:(c + 1) * C].to(torch.complex128) - ref
        num += (d.real * d.real + d.imag * d.imag).sum()
        den += (ref.real * ref.real + ref.imag * ref.imag).sum()
        mx = torch.maximum(mx, d.abs().max())
        rmax = torch.maximum(rmax, ref.abs().max())
    return math.sqrt(float(num.item()) / float(den.item())), float(den.item()), float(mx.item()), float(rmax.item())


def tones_rel_l2(y: torch.Tensor, n: int, k: int, freqs, phases, chunk_bits: int = 22, index_chunks=None):
    """(relative L2, sum |ref|^2) of tones_parity."""
    rel, den, _, _ = tones_parity(y, n, k, freqs, phases, chunk_bits, index_chunks)
    return rel, den
