"""Seeded synthetic inputs shared by the oracle side and the CUDA side.

This module holds NONE of the method's arithmetic (no butterflies, no
controlled phases, no DFT): only the workload recipes of BASELINE.json /
SURVEY.md section 8(d), so that both sides see bit-identical complex64 inputs.

Recipes (all unit l2 norm, complex64, index j <-> basis state with qubit q =
bit q of j):
  gaussian(n, seed)     re, im ~ N(0,1) from numpy default_rng(seed), normalised
                        in float64, cast to complex64 (configs 1-3).
  tone(n, f)            exp(2 pi i ((f j) mod N) / N) / sqrt(N)  -- the paper's
                        own single-tone correctness input.
  delta(n, idx)         Kronecker delta.
  tone_params(n, seed, ntones)   frequencies / phases of the sparse multi-tone
                        inputs of configs 4-5 (numpy default_rng(seed)).
  multi_tone(n, freqs, phases)   (T N)^{-1/2} sum_i e^{i theta_i} e^{2 pi i f_i j / N}.
Device-side variants (torch, float64 arithmetic on the device, chunked so that
n = 33 fits) are used where the state is too large to generate on the host.
"""
from __future__ import annotations

import math

import numpy as np


def gaussian(n: int, seed: int) -> np.ndarray:
    N = 1 << n
    rng = np.random.default_rng(seed)
    re = rng.standard_normal(N)
    im = rng.standard_normal(N)
    x = re + 1j * im
    x /= np.sqrt(np.sum(re * re + im * im))
    return x.astype(np.complex64)


def tone(n: int, f: int) -> np.ndarray:
    N = 1 << n
    j = np.arange(N, dtype=np.int64)
    p = (j * int(f)) & (N - 1)
    ang = (2.0 * np.pi / N) * p.astype(np.float64)
    return ((np.cos(ang) + 1j * np.sin(ang)) / math.sqrt(N)).astype(np.complex64)


def delta(n: int, idx: int) -> np.ndarray:
    x = np.zeros(1 << n, dtype=np.complex64)
    x[idx] = 1.0
    return x


def tone_params(n: int, seed: int, ntones: int = 5):
    """Distinct uniform frequencies in [0, N) and uniform phases in [0, 2 pi)."""
    rng = np.random.default_rng(seed)
    N = 1 << n
    freqs = []
    while len(freqs) < ntones:
        f = int(rng.integers(0, N))
        if f not in freqs:
            freqs.append(f)
    phases = rng.uniform(0.0, 2.0 * np.pi, size=ntones)
    return np.asarray(freqs, dtype=np.int64), np.asarray(phases, dtype=np.float64)


def multi_tone(n: int, freqs, phases) -> np.ndarray:
    N = 1 << n
    j = np.arange(N, dtype=np.int64)
    acc = np.zeros(N, dtype=np.complex128)
    for f, th in zip(freqs, phases):
        p = (j * int(f)) & (N - 1)
        ang = (2.0 * np.pi / N) * p.astype(np.float64) + float(th)
        acc += np.cos(ang) + 1j * np.sin(ang)
    acc /= math.sqrt(len(freqs) * N)
    return acc.astype(np.complex64)


# ----------------------------------------------------------------------------
# device-side generators (torch); same recipes, float64 arithmetic, chunked.
# ----------------------------------------------------------------------------

def multi_tone_device(n: int, freqs, phases, device="cuda", out=None, chunk_bits: int = 24):
    """multi_tone() generated in place on the device (complex64 result).

    The integer phase (f*j) mod 2^n is exact: int64 multiplication wraps mod
    2^64 and 2^n divides 2^64.
    """
    import torch

    N = 1 << n
    if out is None:
        out = torch.empty(N, dtype=torch.complex64, device=device)
    cb = min(chunk_bits, n)
    C = 1 << cb
    amp = 1.0 / math.sqrt(len(freqs) * N)
    base = torch.arange(C, dtype=torch.int64, device=device)
    view = torch.view_as_real(out)
    for c in range(N >> cb):
        j = base + (c << cb)
        re = torch.zeros(C, dtype=torch.float64, device=device)
        im = torch.zeros(C, dtype=torch.float64, device=device)
        for f, th in zip(freqs, phases):
            p = (j * int(f)) & (N - 1)
            ang = p.to(torch.float64) * (2.0 * math.pi / N) + float(th)
            re += torch.cos(ang)
            im += torch.sin(ang)
        view[c << cb:(c + 1) << cb, 0] = (re * amp).to(torch.float32)
        view[c << cb:(c + 1) << cb, 1] = (im * amp).to(torch.float32)
    return out


def gaussian_device(n: int, seed: int, device="cuda", out=None, chunk_bits: int = 26):
    """Unit-norm complex Gaussian generated on the device from torch's seeded
    Philox generator (used for states too large for the host: n >= 28).  The
    norm is a float64 reduction."""
    import torch

    N = 1 << n
    if out is None:
        out = torch.empty(N, dtype=torch.complex64, device=device)
    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    view = torch.view_as_real(out)
    cb = min(chunk_bits, n)
    C = 1 << cb
    ss = torch.zeros((), dtype=torch.float64, device=device)
    for c in range(N >> cb):
        blk = view[c << cb:(c + 1) << cb]
        blk.normal_(generator=g)
        ss += (blk.to(torch.float64) ** 2).sum()
    scale = float(1.0 / math.sqrt(float(ss.item())))
    for c in range(N >> cb):
        view[c << cb:(c + 1) << cb].mul_(scale)
    return out
