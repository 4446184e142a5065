"""Pins the large-state checkers (tests/large_checks.py) against the CPU oracle at small n, on the
CPU, so that the n = 30 / 33 GPU tests can rely on them."""
import numpy as np
import pytest
import torch

import large_checks as lc
import oracle
import qft_inputs as qi


@pytest.mark.parametrize("k", [0, 3, 7, 11, 12])
def test_sampled_outputs_match_oracle(k):
    n = 12
    x = qi.gaussian(n, 17)
    Ks = [0, 1, 5, 100, 2047, 4095]
    for sign in (-1, 1):
        full = oracle.qft(x, k, sign)
        got = lc.sampled_outputs(torch.from_numpy(x), Ks, k, sign, chunk_bits=10).numpy()
        assert np.max(np.abs(got - full[Ks])) < 1e-12
        assert np.max(np.abs(got - oracle.outputs_at(x, Ks, k, sign))) < 1e-12


@pytest.mark.parametrize("n,k", [(14, 5), (14, 14), (13, 0), (9, 2), (3, 1)])
def test_sampled_outputs_32_indices_both_tables(n, k):
    """Sizes at which both the low-bits and the high-bits phase table are in play (h = 12 or chunk_bits < n),
    32 sampled indices at once as in the n = 30 / 33 GPU tests, against the full oracle output."""
    x = qi.gaussian(n, 40 + n)
    rng = np.random.default_rng(n)
    Ks = sorted({int(v) for v in rng.integers(0, 1 << n, size=64)})[:32]
    full = oracle.qft(x, k)
    for chunk_bits in (24, max(1, n - 3)):
        got = lc.sampled_outputs(torch.from_numpy(x), Ks, k, -1, chunk_bits=chunk_bits).numpy()
        assert np.max(np.abs(got - full[Ks])) < 1e-12


def test_phase_coefficients_reduce_to_the_dft_for_exact_k():
    """Exact k: the linear phase must be K j / N, i.e. c_b = -K 2^b / N modulo one turn."""
    n = 11
    for K in (0, 1, 2, 777, 2047):
        c = lc._phase_coefficients(n, [K], n, -1)[:, 0].numpy()
        for b in range(n):
            want = (-(K << b) / (1 << n)) % 1.0
            assert abs((c[b] % 1.0) - want) < 1e-15


@pytest.mark.parametrize("k", [0, 1, 4, 8, 10, 11, 30])
def test_tones_closed_form_matches_oracle(k):
    n = 11
    fr, ph = qi.tone_params(n, 3, 5)
    N = 1 << n
    j = np.arange(N)
    xd = sum(np.exp(1j * th) * np.exp(2j * np.pi * ((j * int(f)) % N) / N) for f, th in zip(fr, ph)) / np.sqrt(5 * N)
    ref = oracle.qft(xd, k)
    got = lc.tones_closed_form_chunk(n, k, fr, ph, torch.arange(N, dtype=torch.int64)).numpy()
    assert np.max(np.abs(got - ref)) < 1e-12
    y = torch.from_numpy(ref.astype(np.complex64))
    rel, den = lc.tones_rel_l2(y, n, k, fr, ph, chunk_bits=8)
    assert rel < 1e-6 and abs(den - 1.0) < 1e-9
    rel2, _ = lc.tones_rel_l2(y, n, k, fr, ph, chunk_bits=8, index_chunks=[0, 3])
    assert rel2 < 1e-6


def test_device_generators_match_host_recipes():
    n = 12
    fr, ph = qi.tone_params(n, 4, 5)
    a = qi.multi_tone(n, fr, ph)
    b = qi.multi_tone_device(n, fr, ph, device="cpu", chunk_bits=9).numpy()
    assert np.max(np.abs(a - b)) < 1e-7
    g = qi.gaussian_device(n, 2, device="cpu", chunk_bits=10)
    assert abs(lc.norm2(g, chunk_bits=9) - 1.0) < 1e-6
