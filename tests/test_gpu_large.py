"""GPU parity at BASELINE.json's full sizes (configs 3-5), in the launch configuration bench.py times.

n = 26: element by element against the CPU oracle (1 GiB of fp64 state), for every max_fused_qubits of
config 3.  n = 30 and n = 33: beyond the oracle's practical size, so (north_star) closed-form
sparse-tone outputs, Parseval, and float64 direct sums at sampled output indices
(tests/large_checks.py, pinned to the oracle on the CPU by tests/test_large_checks_cpu.py).
"""
import math

import numpy as np
import pytest

import qft_inputs as qi

pytestmark = pytest.mark.gpu

TOL_LARGE = 1e-4  # north_star: relative L2 <= 1e-4 up to n = 33


def _free_gib():
    import torch

    torch.cuda.empty_cache()  # earlier tests' cached blocks count as used otherwise
    free, _ = torch.cuda.mem_get_info()
    return free / 2 ** 30


def test_config3_n26_window_sweep_against_oracle():
    import torch

    import oracle
    import paper_2606_18981_b200 as qft

    n = 26
    x = qi.gaussian(n, 1)
    ref = torch.from_numpy(oracle.qft(x)).cuda()
    refn = float(torch.linalg.vector_norm(ref).item())
    passes = []
    for w in (2, 4, 6, 10, 13):
        plan = qft.Plan(n, n, w)
        t = torch.from_numpy(x).cuda()
        plan.execute(t)
        torch.cuda.synchronize()
        err = float(torch.linalg.vector_norm(t.to(torch.complex128) - ref).item()) / refn
        passes.append(plan.num_passes)
        plan.close()
        assert err <= TOL_LARGE, (w, err)
        del t
    assert passes == sorted(passes, reverse=True) and passes[-1] == 3
    # AQFT at the same size, one cutoff
    refk = torch.from_numpy(oracle.qft(x, 8)).cuda()
    plan = qft.Plan(n, 8)
    t = torch.from_numpy(x).cuda()
    plan.execute(t)
    torch.cuda.synchronize()
    err = float(torch.linalg.vector_norm(t.to(torch.complex128) - refk).item()) / float(
        torch.linalg.vector_norm(refk).item())
    plan.close()
    assert err <= TOL_LARGE


def _sample_indices(n, freqs, seed, count=32):
    rng = np.random.default_rng(seed)
    Ks = [int(f) for f in freqs]
    while len(Ks) < count:
        K = int(rng.integers(0, 1 << n))
        if K not in Ks:
            Ks.append(K)
    return Ks


def test_config4_n30_aqft_sweep_tones_closed_form():
    import torch

    import large_checks as lc
    import paper_2606_18981_b200 as qft

    if _free_gib() < 14:
        pytest.skip("needs 14 GiB of free device memory")
    n = 30
    fr, ph = qi.tone_params(n, 3, 5)
    x = qi.multi_tone_device(n, fr, ph, device="cuda")
    assert abs(lc.norm2(x) - 1.0) < 1e-5
    nchunks = 1 << (n - 22)
    rng = np.random.default_rng(30)
    near = sorted({int(f) >> 22 for f in fr})
    for k in (4, 8, 12, 16, 30):
        y = x.clone()
        plan = qft.Plan(n, k)
        assert plan.num_passes == 3
        plan.execute(y)
        torch.cuda.synchronize()
        plan.close()
        assert abs(lc.norm2(y) - 1.0) < 1e-4  # Parseval: every AQFT_k is unitary
        if k in (4, 30):
            chunks = None  # every output index
        else:  # the chunks around the tone bins (where the energy is) + 24 random chunks
            chunks = sorted(set(near) | {int(c) for c in rng.integers(0, nchunks, size=24)})
        rel, den = lc.tones_rel_l2(y, n, k, fr, ph, chunk_bits=22, index_chunks=chunks)
        assert rel <= TOL_LARGE, (k, rel)
        if chunks is None:
            assert abs(den - 1.0) < 1e-9
        if k == 30:  # exact: five bins of modulus 1/sqrt 5, nothing else
            got = y[torch.as_tensor(fr, device="cuda")].to(torch.complex128).cpu().numpy()
            assert np.max(np.abs(got - np.exp(1j * ph) / math.sqrt(5))) < 1e-4
        del y


def test_config4_n30_gaussian_parseval_and_sampled_sums():
    import torch

    import large_checks as lc
    import paper_2606_18981_b200 as qft

    if _free_gib() < 14:
        pytest.skip("needs 14 GiB of free device memory")
    n = 30
    x = qi.gaussian_device(n, 2, device="cuda")
    fr, _ = qi.tone_params(n, 3, 5)
    for k, count in ((30, 32), (12, 6)):
        Ks = _sample_indices(n, fr, 31, count)
        want = lc.sampled_outputs(x, Ks, k)  # from the actual fp32 device input, BEFORE the transform
        y = x.clone()
        plan = qft.Plan(n, k)
        plan.execute(y)
        torch.cuda.synchronize()
        plan.close()
        assert abs(lc.norm2(y) - 1.0) < 1e-4
        got = y[torch.as_tensor(Ks, device="cuda")].to(torch.complex128)
        # |out[K]| ~ 2^-15 for a unit-norm Gaussian state: compare relative to the samples' norm
        rel = float(torch.linalg.vector_norm(got - want).item() / torch.linalg.vector_norm(want).item())
        assert rel <= TOL_LARGE, (k, rel)
        del y


def test_config5_n33_tones_exact_and_k16():
    import torch

    import large_checks as lc
    import paper_2606_18981_b200 as qft

    if _free_gib() < 70:
        pytest.skip("needs 70 GiB of free device memory")
    n = 33
    fr, ph = qi.tone_params(n, 4, 5)
    x = torch.empty(1 << n, dtype=torch.complex64, device="cuda")
    nchunks = 1 << (n - 22)
    rng = np.random.default_rng(33)
    near = sorted({int(f) >> 22 for f in fr})
    for k, count in ((33, 32), (16, 3)):
        qi.multi_tone_device(n, fr, ph, device="cuda", out=x)
        assert abs(lc.norm2(x) - 1.0) < 1e-5
        Ks = _sample_indices(n, fr, 34, count)
        want = lc.sampled_outputs(x, Ks, k)  # direct fp64 sums over the 2^33 inputs, before the transform
        plan = qft.Plan(n, k)
        assert plan.num_passes == 4
        plan.execute(x)  # in place: 64 GiB, no second copy
        torch.cuda.synchronize()
        plan.close()
        assert abs(lc.norm2(x) - 1.0) < 1e-4
        got = x[torch.as_tensor(Ks, device="cuda")].to(torch.complex128)
        err = float(torch.linalg.vector_norm(got - want).item() / torch.linalg.vector_norm(want).item())
        assert err <= TOL_LARGE, (k, err)
        chunks = sorted(set(near) | {int(c) for c in rng.integers(0, nchunks, size=40)})
        rel, _ = lc.tones_rel_l2(x, n, k, fr, ph, chunk_bits=22, index_chunks=chunks)
        assert rel <= TOL_LARGE, (k, rel)
        if k == 33:
            g5 = x[torch.as_tensor(fr, device="cuda")].to(torch.complex128).cpu().numpy()
            assert np.max(np.abs(g5 - np.exp(1j * ph) / math.sqrt(5))) < 1e-4


def test_max_size_n34_tones_exact():
    """The largest state the ABI accepts (n = 34: 128 GiB in place on a 180 GB B200): five tones against the
    closed form on sampled chunks, Parseval, and direct double-precision sums at sampled outputs."""
    import torch

    import large_checks as lc
    import paper_2606_18981_b200 as qft

    if _free_gib() < 136:
        pytest.skip("needs 136 GiB of free device memory")
    n = 34
    fr, ph = qi.tone_params(n, 5, 5)
    x = torch.empty(1 << n, dtype=torch.complex64, device="cuda")
    qi.multi_tone_device(n, fr, ph, device="cuda", out=x)
    assert abs(lc.norm2(x) - 1.0) < 1e-5
    Ks = _sample_indices(n, fr, 35, 8)
    want = lc.sampled_outputs(x, Ks, n)
    plan = qft.Plan(n, n)
    plan.self_check()
    plan.execute(x)
    torch.cuda.synchronize()
    plan.close()
    assert abs(lc.norm2(x) - 1.0) < 1e-4
    got = x[torch.as_tensor(Ks, device="cuda")].to(torch.complex128)
    err = float(torch.linalg.vector_norm(got - want).item() / torch.linalg.vector_norm(want).item())
    assert err <= TOL_LARGE, err
    rng = np.random.default_rng(34)
    near = sorted({int(f) >> 22 for f in fr})
    chunks = sorted(set(near) | {int(c) for c in rng.integers(0, 1 << (n - 22), size=24)})
    rel, _ = lc.tones_rel_l2(x, n, n, fr, ph, chunk_bits=22, index_chunks=chunks)
    assert rel <= TOL_LARGE, rel
    g5 = x[torch.as_tensor(fr, device="cuda")].to(torch.complex128).cpu().numpy()
    assert np.max(np.abs(g5 - np.exp(1j * ph) / math.sqrt(5))) < 1e-4
