"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element.

Tolerances (tests/parity_bounds.py): north_star's relative L2 error <= 2e-5 for n <= 20 and
<= 1e-4 up to n = 33, plus a regression bound near the measured level and a max-abs element bound.
"""
import math

import numpy as np
import pytest

import oracle
import qft_inputs as qi

pytestmark = pytest.mark.gpu

from parity_bounds import TOL_LARGE, TOL_SMALL, assert_parity_numpy


def tol(n):
    return TOL_SMALL if n <= 20 else TOL_LARGE


def parity(got, ref, what=""):
    """All three bounds of tests/parity_bounds.py against an oracle result."""
    n = int(np.asarray(ref).shape[0]).bit_length() - 1
    return assert_parity_numpy(np.asarray(got), np.asarray(ref, dtype=np.complex128), n, what)


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.complex128)
    b = np.asarray(b, dtype=np.complex128)
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def gpu_qft(x, k=None, **kw):
    import torch

    import paper_2606_18981_b200 as qft

    n = int(x.shape[0]).bit_length() - 1
    plan = qft.Plan(n, n if k is None else k, **kw)
    plan.self_check()
    t = torch.from_numpy(np.ascontiguousarray(x, dtype=np.complex64)).cuda()
    plan.execute(t)
    torch.cuda.synchronize()
    out = t.cpu().numpy()
    plan.close()
    return out


@pytest.mark.parametrize("n", list(range(1, 17)))
def test_exact_small_n(n):
    x = qi.gaussian(n, 40 + n)
    parity(gpu_qft(x), oracle.qft(x))


def test_config1_n10():
    """BASELINE config 1: n = 10, Gaussian seed 0, forward, unitary."""
    x = qi.gaussian(10, 0)
    got = gpu_qft(x)
    parity(got, oracle.qft(x))
    parity(got, oracle.naive_dft(x))


@pytest.mark.parametrize("k", [0, 1, 2, 3, 4, 5, 8, 11, 12])
@pytest.mark.parametrize("n", [7, 12, 15])
def test_aqft_cutoffs(n, k):
    x = qi.gaussian(n, 7 * n + k)
    parity(gpu_qft(x, k), oracle.qft(x, k))


@pytest.mark.parametrize("sign", [-1, 1])
@pytest.mark.parametrize("norm", [0, 1, 2])
def test_sign_and_normalisation(sign, norm):
    for n, k in ((9, 9), (14, 14), (14, 3)):
        x = qi.gaussian(n, 3)
        parity(gpu_qft(x, k, sign=sign, normalisation=norm), oracle.qft(x, k, sign, norm))


@pytest.mark.parametrize("w", [1, 2, 3, 4, 6, 9, 10, 13])
@pytest.mark.parametrize("n", [11, 16, 18])
def test_result_independent_of_max_fused_qubits(n, w):
    x = qi.gaussian(n, 5)
    ref = oracle.qft(x, 6)
    parity(gpu_qft(x, 6, max_fused_qubits=w), ref)


@pytest.mark.parametrize("tile_bits,hub_bits", [(4, 1), (5, 2), (6, 2), (7, 3), (9, 3), (12, 4), (14, 3), (14, 4)])
def test_tuned_layouts(tile_bits, hub_bits):
    """Small tiles force many passes, pair (cluster) passes and ragged windows at small n."""
    for n in (5, 8, 11, 13, 15, 17):
        for flags in (0, 2):
            for k in (n, 3):
                x = qi.gaussian(n, n)
                got = gpu_qft(x, k, tile_bits=tile_bits, hub_bits=hub_bits, flags=flags)
                parity(got, oracle.qft(x, k), (n, flags, k))


def test_config2_n20_three_inputs():
    n, N = 20, 1 << 20
    xg = qi.gaussian(n, 0)
    parity(gpu_qft(xg), oracle.qft(xg))
    xt = qi.tone(n, 12345)
    got = gpu_qft(xt)
    parity(got, oracle.qft(xt))
    assert abs(abs(got[12345]) - 1.0) < 1e-4 and np.linalg.norm(np.delete(got, 12345)) < 1e-3
    xd = qi.delta(n, 777)
    got = gpu_qft(xd)
    parity(got, oracle.qft(xd))
    K = np.arange(N)
    want = np.exp(-2j * np.pi * ((777 * K) % N) / N) / 1024.0
    parity(got, want)


def test_paper_workload_n22_tone2():
    """The paper's own correctness input: single tone at bin k0 = 2, n = 22."""
    n = 22
    x = qi.tone(n, 2)
    got = gpu_qft(x)
    parity(got, oracle.qft(x))
    for k in (4, 8):
        gk = gpu_qft(x, k)
        parity(gk, oracle.qft(x, k))
        leak = 1 - abs(gk[2]) ** 2 / float(np.vdot(gk, gk).real)
        pred = (4 * np.pi ** 2 / 3) * 4.0 ** (-(k + 2))
        assert 0.5 * pred < leak < 2.0 * pred


def test_linearity_and_round_trip_on_device():
    n = 17
    a, b = qi.gaussian(n, 1), qi.gaussian(n, 2)
    al, be = np.complex64(0.3 - 1.1j), np.complex64(-2.0 + 0.25j)
    lhs = gpu_qft((al * a + be * b).astype(np.complex64), 5)
    rhs = al * gpu_qft(a, 5) + be * gpu_qft(b, 5)
    assert rel_l2(lhs, rhs) <= 1e-5
    back = gpu_qft(gpu_qft(a), sign=1)
    assert rel_l2(back, a) <= 1e-5


def test_execute_host_matches_device_path():
    import paper_2606_18981_b200 as qft

    n = 16
    x = qi.gaussian(n, 8)
    h = x.copy()
    plan = qft.Plan(n, 7)
    plan.execute_host(h)
    plan.close()
    parity(h, oracle.qft(x, 7))


def test_plan_reuse_and_streams():
    import torch

    import paper_2606_18981_b200 as qft

    n = 15
    plan = qft.Plan(n, n)
    s = torch.cuda.Stream()
    xs = [qi.gaussian(n, i) for i in range(3)]
    outs = []
    for x in xs:
        t = torch.from_numpy(x).cuda()
        with torch.cuda.stream(s):
            plan.execute(t)
        s.synchronize()
        outs.append(t.cpu().numpy())
    for x, o in zip(xs, outs):
        parity(o, oracle.qft(x))
    plan.close()


def test_error_codes_on_device():
    import torch

    import paper_2606_18981_b200 as qft

    plan = qft.Plan(8, 8)
    t = torch.zeros(256 + 1, dtype=torch.complex64, device="cuda")
    with pytest.raises(qft.QftError):
        qft.qft_execute(plan.handle, t.data_ptr() + 8, 0)  # misaligned
    with pytest.raises(qft.QftError):
        qft.qft_execute(plan.handle, 0, 0)  # null
    plan.close()


def test_aqft_accuracy_vs_cutoff_paper_workload():
    """The paper's AQFT accuracy experiment (Fig. 6): n = 22, single tone at bin 2, unit
    norm; infidelity 1 - F against the exact output and top-bin leakage, both falling as k grows.  The
    GPU path must reproduce the oracle's values, and both follow (4 pi^2 / 3) 4^-(k+2), the closed form
    the product formula of the AQFT gives for a low-frequency tone."""
    n, f = 22, 2
    x = qi.tone(n, f)
    exact = gpu_qft(x).astype(np.complex128)
    assert abs(abs(exact[f]) - 1.0) <= 1e-5
    prev = None
    for k in (4, 6, 8, 10):
        got = gpu_qft(x, k).astype(np.complex128)
        ref = oracle.qft(x, k)
        parity(got, ref)

        def metrics(out):
            leak = 1.0 - abs(out[f]) ** 2 / float(np.vdot(out, out).real)
            fid = abs(np.vdot(exact, out)) ** 2 / float(np.vdot(exact, exact).real * np.vdot(out, out).real)
            return leak, 1.0 - fid

        (lg, ig), (lo, io) = metrics(got), metrics(ref)
        pred = (4.0 * math.pi ** 2 / 3.0) * 4.0 ** (-(k + 2))
        assert abs(lo - pred) <= 0.05 * pred            # the oracle follows the closed form
        assert abs(lg - lo) <= 0.02 * lo + 2e-6          # the GPU path follows the oracle (fp32 floor ~1e-6)
        assert abs(ig - io) <= 0.02 * io + 2e-6
        if prev is not None:
            assert lg < prev                             # monotone in k
        prev = lg


@pytest.mark.parametrize("n,k", [(12, 2), (18, 3), (22, 5), (24, 0)])
def test_aqft_round_trip(n, k):
    """sign = +1 with the same cutoff inverts the forward AQFT (reading c12)."""
    x = qi.gaussian(n, 9)
    y = gpu_qft(x, k)
    z = gpu_qft(y, k, sign=1)
    assert rel_l2(z, x) <= tol(n)


@pytest.mark.parametrize("n_lo,n_hi,count", [(13, 20, 160), (20, 24, 48)])
def test_random_plan_configurations(n_lo, n_hi, count):
    """A seeded sweep over the planner's knobs (tile / hub bits, window cap, cutoff, sign, normalisation, unfolded /
    deferred schedules) at n = 13 ... 23: whatever plan comes out must match the oracle.  Unschedulable combinations
    must be refused with QFT_ERR_UNSUPPORTED, never fail the self-check."""
    import torch

    import paper_2606_18981_b200 as qft

    rng = np.random.default_rng(20261105 + n_lo)
    ran = 0
    for _ in range(count):
        n = int(rng.integers(n_lo, n_hi))
        tile_bits = int(rng.choice([0, 0, 9, 10, 11, 12, 13, 14]))
        hub_bits = int(rng.choice([0, 0, 2, 3, 4, 5]))
        w = int(rng.choice([2, 3, 4, 5, 6, 7, 9, 13]))
        k = int(rng.choice([n, n, 0, 1, 2, 3, 5, 9]))
        sign = int(rng.choice([-1, 1]))
        norm = int(rng.integers(0, 3))
        flags = int(rng.choice([0, 0, 0, qft.QFT_FLAG_UNFOLDED, qft.QFT_FLAG_DEFER_SWAPS, qft.QFT_FLAG_NO_TMA]))
        try:
            plan = qft.Plan(n, k, w, sign, norm, tile_bits, hub_bits, flags)
        except qft.QftError as e:
            assert e.status == qft.QFT_ERR_UNSUPPORTED, (n, tile_bits, hub_bits, w, k, flags, str(e))
            continue
        plan.self_check()
        x = qi.gaussian(n, 1000 + ran)
        t = torch.from_numpy(x).cuda()
        plan.execute(t)
        torch.cuda.synchronize()
        got = t.cpu().numpy().astype(np.complex128)
        what = (n, tile_bits, hub_bits, w, k, sign, norm, flags, [p["kernel"] for p in plan.describe()["passes"]])
        if flags == qft.QFT_FLAG_DEFER_SWAPS:
            # the plan reports where every qubit ended: undo that layout on the host, compare with the natural-order oracle
            order = plan.output_order()
            K = np.arange(1 << n, dtype=np.int64)
            J = np.zeros_like(K)
            for a, q in enumerate(order):
                J |= ((K >> (n - 1 - q)) & 1) << a
            got = got[J]
        parity(got, oracle.qft(x, k, sign, norm), what)
        plan.close()
        ran += 1
    assert ran >= count * 5 // 8
