"""Encode / decode and accuracy metrics (include/qft.h) against numpy in float64:
scale_in = ||x||_2, rescale, fidelity and top-bin leakage."""
import numpy as np
import pytest

import oracle
import qft_inputs as qi

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n", [1, 2, 9, 16, 21])
def test_encode_rescale_fidelity_leakage(n):
    import torch

    import paper_2606_18981_b200 as qft

    rng = np.random.default_rng(n)
    N = 1 << n
    a = (rng.normal(size=N) + 1j * rng.normal(size=N)).astype(np.complex64) * np.float32(3.7)
    b = (a + 0.05 * (rng.normal(size=N) + 1j * rng.normal(size=N))).astype(np.complex64)
    a64, b64 = a.astype(np.complex128), b.astype(np.complex128)
    ta, tb = torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda()
    s = torch.cuda.current_stream().cuda_stream
    n2 = qft.qft_norm_sq(ta.data_ptr(), n, s)
    assert abs(n2 - oracle.norm_sq(a64)) <= 1e-12 * n2
    fid = qft.qft_fidelity(ta.data_ptr(), tb.data_ptr(), n, s)
    ref = oracle.fidelity(a64, b64)
    assert abs(fid - ref) <= 1e-12
    k0 = N // 3
    leak = qft.qft_leakage(tb.data_ptr(), n, k0, s)
    assert abs(leak - oracle.leakage(b64, k0)) <= 1e-12
    scale_in = qft.qft_encode(ta.data_ptr(), n, s)
    enc_ref, scale_ref = oracle.encode(a64)
    assert abs(scale_in - scale_ref) <= 1e-12 * scale_in
    enc = ta.cpu().numpy().astype(np.complex128)
    assert np.linalg.norm(enc - enc_ref) <= 2e-7 * 1.0
    assert abs(qft.qft_norm_sq(ta.data_ptr(), n, s) - 1.0) <= 1e-6
    qft.qft_rescale(ta.data_ptr(), n, scale_in, s)
    torch.cuda.synchronize()
    dec = ta.cpu().numpy().astype(np.complex128)
    assert np.linalg.norm(dec - a64) <= 3e-7 * np.linalg.norm(a64)


def test_fft_style_round_trip_through_the_wrappers():
    """array in -> encode -> QFT -> decode -> array out equals the unnormalised DFT."""
    import torch

    import paper_2606_18981_b200 as qft

    n = 18
    rng = np.random.default_rng(5)
    x = (rng.normal(size=1 << n) + 1j * rng.normal(size=1 << n)).astype(np.complex64) * np.float32(11.0)
    t = torch.from_numpy(x).cuda()
    s = torch.cuda.current_stream().cuda_stream
    scale_in = qft.qft_encode(t.data_ptr(), n, s)
    plan = qft.Plan(n, n)
    plan.execute(t)
    qft.qft_rescale(t.data_ptr(), n, scale_in * np.sqrt(float(1 << n)), s)
    torch.cuda.synchronize()
    plan.close()
    ref = np.fft.fft(x.astype(np.complex128))
    got = t.cpu().numpy().astype(np.complex128)
    assert np.linalg.norm(got - ref) / np.linalg.norm(ref) <= 2e-5


def test_metrics_argument_errors():
    import torch

    import paper_2606_18981_b200 as qft

    z = torch.zeros(1 << 8, dtype=torch.complex64, device="cuda")
    with pytest.raises(qft.QftError):
        qft.qft_encode(z.data_ptr(), 8)          # zero vector
    with pytest.raises(qft.QftError):
        qft.qft_leakage(z.data_ptr(), 8, 1 << 8)  # bin out of range
    with pytest.raises(qft.QftError):
        qft.qft_norm_sq(0, 8)


@pytest.mark.parametrize("n", [1, 4, 10, 17])
def test_encode_padded_against_oracle(n):
    """The whole input-encoding step of PAPER.md:124 (n = ceil(log2 N) qubits, a 2^n-element state, zero padding,
    division by scale_in) against oracle.encode on a zero-padded copy: lengths 1, 3, 1000, 2^n - 1, 2^n (those that
    fit), the source in a buffer of its own and the source being the front of the state itself."""
    import torch

    import paper_2606_18981_b200 as qft

    N = 1 << n
    s = torch.cuda.current_stream().cuda_stream
    for length in sorted({L for L in (1, 3, 1000, N - 1, N) if 1 <= L <= N}):
        assert qft.qft_num_qubits_for(length) <= n
        rng = np.random.default_rng(1000 * n + length)
        x = ((rng.normal(size=length) + 1j * rng.normal(size=length)) * 2.3).astype(np.complex64)
        padded = np.zeros(N, dtype=np.complex128)
        padded[:length] = x
        enc_ref, scale_ref = oracle.encode(padded)
        for in_place in (False, True):
            # the state starts as garbage: the padding must be written, not assumed
            state = torch.full((N,), complex(7.0, -3.0), dtype=torch.complex64, device="cuda")
            if in_place:
                state[:length] = torch.from_numpy(x).cuda()
                src = state
            else:
                src = torch.from_numpy(x).cuda()
            scale_in = qft.qft_encode_padded(state.data_ptr(), n, src.data_ptr(), length, s)
            torch.cuda.synchronize()
            assert abs(scale_in - scale_ref) <= 1e-12 * scale_ref, (n, length, in_place)
            got = state.cpu().numpy().astype(np.complex128)
            assert np.all(got[length:] == 0.0), (n, length, in_place)
            assert np.linalg.norm(got - enc_ref) <= 2e-7, (n, length, in_place)  # the bound of the encode test above
            if not in_place:
                assert np.array_equal(src.cpu().numpy(), x)  # the source is left alone


def test_encode_padded_refuses_partial_overlap_and_bad_lengths():
    import torch

    import paper_2606_18981_b200 as qft

    n = 8
    buf = torch.ones(3 << n, dtype=torch.complex64, device="cuda")
    base = buf.data_ptr()
    state = base + 8 * (1 << n)  # the middle third
    for src, length in ((state + 16, 10), (state - 16, 10), (state + 8 * ((1 << n) - 1), 4), (base, (1 << n) + 1)):
        with pytest.raises(qft.QftError) as ei:
            qft.qft_encode_padded(state, n, src, length)
        assert ei.value.status == qft.QFT_ERR_INVALID_ARG, (src - state, length)
    with pytest.raises(qft.QftError):
        qft.qft_encode_padded(state, n, base, 0)             # empty input
    with pytest.raises(qft.QftError):
        qft.qft_encode_padded(state, n, base, (1 << n) + 1)  # longer than the state
    torch.cuda.synchronize()
    assert bool((buf == 1).all())  # nothing was written by a refused call
    # the neighbours on both sides are legal sources: they touch the state's range without overlapping it
    qft.qft_encode_padded(state, n, base, 1 << n)
    qft.qft_encode_padded(state, n, state + 8 * (1 << n), 5)
    torch.cuda.synchronize()
