"""GPU parity at BASELINE.json's full sizes (configs 3-5), in the launch configuration bench.py times.

n = 26: element by element against the CPU oracle (1 GiB of fp64 state), for every max_fused_qubits of
config 3.  n = 28 and n = 30 (Gaussian input): element by element against the full oracle as well, so that
the kernel instantiations the headline bench times are compared densely (the oracle needs 4 / 16 GiB of host
memory and one to three minutes).  n = 30 and n = 33 otherwise: beyond the oracle's practical size, so
(north_star) closed-form sparse-tone outputs, Parseval, and float64 direct sums at 32 sampled output indices
(tests/large_checks.py, pinned to the oracle on the CPU by tests/test_large_checks_cpu.py).
Bounds: tests/parity_bounds.py (north_star's relative L2, a regression bound, a max-abs element bound).
"""
import math

import numpy as np
import pytest

import qft_inputs as qi

from parity_bounds import MAXABS_FRAC, REG_L2, TOL_LARGE, ChunkedParity

pytestmark = pytest.mark.gpu

NSAMPLES = 32  # north_star: double-precision direct sums at 32 sampled output indices


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
    passes = []
    for w in (2, 4, 6, 10, 13):
        plan = qft.Plan(n, n, w)
        t = torch.from_numpy(x).cuda()
        plan.execute(t)
        torch.cuda.synchronize()
        cp = ChunkedParity()
        cp.add(t, ref)
        passes.append(plan.num_passes)
        kinds = [p["kernel"] for p in plan.describe()["passes"]]
        plan.close()
        cp.check(n, ("max_fused_qubits", w))
        assert set(kinds) == {"tma2"}, (w, kinds)  # no pass of config 3 falls back to the generic kernel
        del t
    assert passes == [13, 7, 5, 3, 3]
    # AQFT at the same size, one cutoff
    refk = torch.from_numpy(oracle.qft(x, 8)).cuda()
    plan = qft.Plan(n, 8)
    t = torch.from_numpy(x).cuda()
    plan.execute(t)
    torch.cuda.synchronize()
    plan.close()
    cp = ChunkedParity()
    cp.add(t, refk)
    cp.check(n, "k = 8")


def _sample_indices(n, freqs, seed, count=NSAMPLES):
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
        rel, den, mx, rmax = lc.tones_parity(y, n, k, fr, ph, chunk_bits=22, index_chunks=chunks)
        assert rel <= TOL_LARGE and rel <= REG_L2 and mx <= MAXABS_FRAC * rmax, (k, rel, mx, rmax)
        if chunks is None:
            assert abs(den - 1.0) < 1e-9
        if k == 30:  # exact: five bins of modulus 1/sqrt 5, nothing else
            got = y[torch.as_tensor(fr, device="cuda")].to(torch.complex128).cpu().numpy()
            assert np.max(np.abs(got - np.exp(1j * ph) / math.sqrt(5))) < 1e-4
        del y


def _check_samples(got, want, what):
    """Sampled outputs against the double-precision direct sums: the three bounds of parity_bounds on the sample."""
    import torch

    d = got - want
    rel = float(torch.linalg.vector_norm(d).item() / torch.linalg.vector_norm(want).item())
    assert rel <= TOL_LARGE, (what, "north_star tolerance", rel)
    assert rel <= REG_L2, (what, "regression bound", rel)
    assert float(d.abs().max().item()) <= MAXABS_FRAC * float(want.abs().max().item()), (what, "element bound")


def test_config4_n30_gaussian_parseval_and_sampled_sums():
    import torch

    import large_checks as lc
    import paper_2606_18981_b200 as qft

    if _free_gib() < 18:
        pytest.skip("needs 18 GiB of free device memory")
    n = 30
    x = qi.gaussian_device(n, 2, device="cuda")
    fr, _ = qi.tone_params(n, 3, 5)
    Ks = _sample_indices(n, fr, 31)
    assert len(Ks) == NSAMPLES
    for k in (4, 8, 12, 16, 30):  # every cutoff of config 4
        want = lc.sampled_outputs(x, Ks, k)  # from the actual fp32 device input, BEFORE the transform
        y = x.clone()
        plan = qft.Plan(n, k)
        plan.execute(y)
        torch.cuda.synchronize()
        plan.close()
        assert abs(lc.norm2(y) - 1.0) < 1e-4
        got = y[torch.as_tensor(Ks, device="cuda")].to(torch.complex128)
        # |out[K]| ~ 2^-15 for a unit-norm Gaussian state: compare relative to the samples' norm
        _check_samples(got, want, ("n = 30 Gaussian", k))
        del y


def _host_gib():
    try:
        import psutil

        return psutil.virtual_memory().available / 2 ** 30
    except Exception:
        return 0.0


@pytest.mark.parametrize("n,k", [(28, 28), (28, 5), (30, 30), (31, 31)])
def test_dense_full_oracle_at_the_bench_kernels(n, k):
    """Every output element of a Gaussian input against the full CPU oracle at n = 28 and n = 30: the default
    plans here are made of the same kernel instantiations bench.py times (the tensor-memory extended 5+4+1
    passes), which the tone inputs (a handful of non-zero outputs) and 32 samples cannot check densely.
    n = 31 is the smallest state whose default plan contains the 5+5+1 extended pass that the n = 31 ... 33 plans
    (BASELINE config 5) are made of; its oracle run needs 60 GiB of host memory and a few minutes."""
    import torch

    import oracle
    import paper_2606_18981_b200 as qft

    need_host = 28 * (1 << n) / 2 ** 30 + 4  # fp64 oracle state + complex64 input + slack
    if _host_gib() < need_host:
        pytest.skip(f"needs {need_host:.0f} GiB of free host memory for the oracle")
    if _free_gib() < 3 * 8 * (1 << n) / 2 ** 30:
        pytest.skip("not enough free device memory")
    x = qi.gaussian_device(n, 2, device="cuda")
    xh = x.cpu().numpy()
    plan = qft.Plan(n, k)
    bench = qft.Plan(30, 30)  # the headline workload's plan: same kernel, same register steps
    shapes = lambda p: {(q["kernel"], tuple(q["steps"])) for q in p.describe()["passes"]}
    if n == 28:
        assert shapes(bench) <= shapes(plan) | {("tma2x", (5, 4, 1))} and ("tma2x", (5, 4, 1)) in shapes(plan)
    if n == 31:
        big = qft.Plan(33, 33)  # config 5's plan: three passes of this shape
        assert shapes(big) == {("tma2x", (5, 5, 1))} and ("tma2x", (5, 5, 1)) in shapes(plan)
        big.close()
    bench.close()
    plan.execute(x)
    torch.cuda.synchronize()
    plan.close()
    ref = oracle.qft(xh, k)  # gate by gate on the host, complex128
    del xh
    cp = ChunkedParity()
    C = 1 << 24
    for c in range((1 << n) // C):
        cp.add(x[c * C:(c + 1) * C], torch.from_numpy(ref[c * C:(c + 1) * C]).cuda())
    rel, mx = cp.check(n, (n, k))
    print(f"dense parity n={n} k={k}: rel_l2={rel:.3e} max_abs/max_ref={mx:.3e}")


def test_config5_n33_tones_exact_and_k16():
    import torch

    import large_checks as lc
    import paper_2606_18981_b200 as qft

    if _free_gib() < 70:
        pytest.skip("needs 70 GiB of free device memory")
    n = 33
    fr, ph = qi.tone_params(n, 4, 5)
    x = torch.empty(1 << n, dtype=torch.complex64, device="cuda")
    for k in (33, 16):
        qi.multi_tone_device(n, fr, ph, device="cuda", out=x)
        assert abs(lc.norm2(x) - 1.0) < 1e-5
        Ks = _sample_indices(n, fr, 34)
        want = lc.sampled_outputs(x, Ks, k)  # direct fp64 sums over the 2^33 inputs, before the transform
        plan = qft.Plan(n, k)
        assert plan.num_passes == 3  # ceil(33 / 11): 11-qubit windows through the tensor-memory extension
        plan.execute(x)  # in place: 64 GiB, no second copy
        torch.cuda.synchronize()
        plan.close()
        assert abs(lc.norm2(x) - 1.0) < 1e-4
        got = x[torch.as_tensor(Ks, device="cuda")].to(torch.complex128)
        _check_samples(got, want, ("n = 33 tones", k))
        # every output index (the full streaming relative L2 against the closed form),
        # in chunks of 2^24: a store that lands a zero on the wrong zero is invisible, a non-zero anywhere is not
        rel, den, mx, rmax = lc.tones_parity(x, n, k, fr, ph, chunk_bits=24, index_chunks=None)
        assert rel <= TOL_LARGE and rel <= REG_L2 and mx <= MAXABS_FRAC * rmax, (k, rel, mx, rmax)
        assert abs(den - 1.0) < 1e-9
        if k == 33:
            g5 = x[torch.as_tensor(fr, device="cuda")].to(torch.complex128).cpu().numpy()
            assert np.max(np.abs(g5 - np.exp(1j * ph) / math.sqrt(5))) < 1e-4


def test_config5_n33_gaussian_parseval_and_sampled_sums():
    """A dense input through config 5's kernel (three 5+5+1 extended passes): every sampled output depends on all 2^33
    inputs and has modulus about 2^-16.5, not 0 as almost everywhere for the tones.  In place: one 64 GiB buffer."""
    import torch

    import large_checks as lc
    import paper_2606_18981_b200 as qft

    if _free_gib() < 70:
        pytest.skip("needs 70 GiB of free device memory")
    n = 33
    x = torch.empty(1 << n, dtype=torch.complex64, device="cuda")
    fr, _ = qi.tone_params(n, 4, 5)
    Ks = _sample_indices(n, fr, 36)
    for k in (33, 16):
        qi.gaussian_device(n, 6, device="cuda", out=x)
        assert abs(lc.norm2(x) - 1.0) < 1e-5
        want = lc.sampled_outputs(x, Ks, k)  # direct fp64 sums over the actual fp32 input, BEFORE the transform
        plan = qft.Plan(n, k)
        assert {(q["kernel"], tuple(q["steps"])) for q in plan.describe()["passes"]} == {("tma2x", (5, 5, 1))}
        plan.execute(x)
        torch.cuda.synchronize()
        plan.close()
        assert abs(lc.norm2(x) - 1.0) < 1e-4
        got = x[torch.as_tensor(Ks, device="cuda")].to(torch.complex128)
        assert float(want.abs().min().item()) > 1e-8  # dense: no sampled output is (nearly) zero
        _check_samples(got, want, ("n = 33 Gaussian", k))


@pytest.mark.parametrize("k", [31, 9])
def test_dense_n31_extended_plan_against_plain_plan(k):
    """Every output element of a Gaussian input at n = 31, the default plan (5+5+1 extended passes through tensor
    memory, as at n = 33) against the plan without the extension (QFT_FLAG_NO_EXT_TILE: four plain 2^14-tile passes
    of the kind that the smaller sizes compare with the oracle element by element).  Two independent schedules and
    kernel instantiations, no host oracle: 2 x 16 GiB on the device."""
    import torch

    import paper_2606_18981_b200 as qft

    if _free_gib() < 40:
        pytest.skip("needs 40 GiB of free device memory")
    n = 31
    x = qi.gaussian_device(n, 8, device="cuda")
    y = x.clone()
    ext = qft.Plan(n, k)
    plain = qft.Plan(n, k, flags=qft.QFT_FLAG_NO_EXT_TILE)
    shapes = lambda p: [(q["kernel"], tuple(q["steps"])) for q in p.describe()["passes"]]
    assert ("tma2x", (5, 5, 1)) in shapes(ext) and all(kind == "tma2" for kind, _ in shapes(plain))
    ext.execute(x)
    plain.execute(y)
    torch.cuda.synchronize()
    ext.close()
    plain.close()
    cp = ChunkedParity()
    C = 1 << 26
    for c in range((1 << n) // C):
        cp.add(x[c * C:(c + 1) * C], y[c * C:(c + 1) * C].to(torch.complex128))
    rel, mx = cp.check(n, ("n = 31 extended vs plain", k))
    assert abs(cp.den - 1.0) < 1e-4  # and the reference side is a unit vector (Parseval)
    print(f"n=31 k={k} extended vs plain: rel_l2={rel:.3e} max_abs/max_ref={mx:.3e}")


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
    Ks = _sample_indices(n, fr, 35)
    want = lc.sampled_outputs(x, Ks, n)
    plan = qft.Plan(n, n)
    plan.self_check()
    plan.execute(x)
    torch.cuda.synchronize()
    plan.close()
    assert abs(lc.norm2(x) - 1.0) < 1e-4
    got = x[torch.as_tensor(Ks, device="cuda")].to(torch.complex128)
    _check_samples(got, want, "n = 34 tones")
    rng = np.random.default_rng(34)
    near = sorted({int(f) >> 22 for f in fr})
    chunks = sorted(set(near) | {int(c) for c in rng.integers(0, 1 << (n - 22), size=24)})
    rel, _, mx, rmax = lc.tones_parity(x, n, n, fr, ph, chunk_bits=22, index_chunks=chunks)
    assert rel <= TOL_LARGE and rel <= REG_L2 and mx <= MAXABS_FRAC * rmax, (rel, mx, rmax)
    g5 = x[torch.as_tensor(fr, device="cuda")].to(torch.complex128).cpu().numpy()
    assert np.max(np.abs(g5 - np.exp(1j * ph) / math.sqrt(5))) < 1e-4
