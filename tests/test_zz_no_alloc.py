"""qft_fidelity_batched_static (include/qft.h): the fidelity reduction for callers that cannot allocate device
memory - a process whose HBM already belongs to one pool or to the state vectors themselves, or a loop that cannot
take the stall of an allocation.  Its accumulators are a fixed array inside libqft.so instead of a buffer obtained
from the runtime at first use, so the things to check are: the same numbers as the allocating path (qft_fidelity,
one state at a time), still the same numbers on a second call that finds the first call's sums in the shared array,
a clear refusal beyond the array's capacity, and no allocating call in the source.

This file sorts last on purpose (pytest -x stops at the first failure: a failure here must not hide other tests);
it passes alone in a fresh process and after the rest of the suite (nothing else touches the array)."""
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _pairs(rng, n, batch):
    N = 1 << n
    a = (rng.normal(size=(batch, N)) + 1j * rng.normal(size=(batch, N))).astype(np.complex64)
    # noise growing with the batch index: fidelities spread over (0, 1], not all alike
    noise = (rng.normal(size=(batch, N)) + 1j * rng.normal(size=(batch, N))) * (0.05 * (1 + np.arange(batch)))[:, None]
    b = (a * np.float32(2.5) + noise).astype(np.complex64)
    return a, b


@pytest.mark.gpu
@pytest.mark.parametrize("n,batch", [(1, 1), (3, 7), (12, 5), (16, 3), (10, 300), (21, 2)])
def test_static_scratch_fidelity_matches_allocating_path_twice_in_a_row(n, batch):
    import torch

    import paper_2606_18981_b200 as qft

    rng = np.random.default_rng(1000 * n + batch)
    s = torch.cuda.current_stream().cuda_stream
    # two calls back to back on one stream, on different data: the second finds the first's sums in the array
    for call in range(2):
        a, b = _pairs(rng, n, batch)
        ta, tb = torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda()
        out = torch.full((batch,), -1.0, dtype=torch.float64, device="cuda")
        qft.qft_fidelity_batched_static(ta.data_ptr(), tb.data_ptr(), n, batch, out.data_ptr(), s)
        got = out.cpu().numpy()  # the copy waits for the stream
        # the existing path, one state at a time (n >= 1 keeps every state of the batch 16-byte aligned)
        want = np.array([qft.qft_fidelity(ta[i].data_ptr(), tb[i].data_ptr(), n, s) for i in range(batch)])
        # the tolerance of tests/test_metrics.py for the fidelity (both sides accumulate in fp64, in another order)
        assert np.all(np.abs(got - want) <= 1e-12), (call, got, want)
        # and against the definition in float64 (numpy), so that both paths are not wrong together
        a64, b64 = a.astype(np.complex128), b.astype(np.complex128)
        ref = np.abs(np.sum(np.conj(a64) * b64, axis=1)) ** 2 / (np.sum(np.abs(a64) ** 2, axis=1) * np.sum(np.abs(b64) ** 2, axis=1))
        assert np.all(np.abs(got - ref) <= 1e-12), (call, got, ref)
        assert 0.0 < got.min() and got.max() <= 1.0 + 1e-12


@pytest.mark.gpu
def test_static_scratch_full_capacity_then_small_batch():
    """The largest batch the array holds, then a small one on the same stream: the small call must not see what
    the big one left in the slots it reuses, and a zero state gives NaN there, not an error."""
    import torch

    import paper_2606_18981_b200 as qft

    n, batch = 6, qft.QFT_STATIC_MAX_BATCH
    rng = np.random.default_rng(7)
    a, b = _pairs(rng, n, 8)
    a = np.tile(a, (batch // 8, 1))
    b = np.tile(b, (batch // 8, 1))
    ta, tb = torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda()
    out = torch.empty(batch, dtype=torch.float64, device="cuda")
    s = torch.cuda.current_stream().cuda_stream
    qft.qft_fidelity_batched_static(ta.data_ptr(), tb.data_ptr(), n, batch, out.data_ptr(), s)
    got = out.cpu().numpy()
    want8 = np.array([qft.qft_fidelity(ta[i].data_ptr(), tb[i].data_ptr(), n, s) for i in range(8)])
    assert np.all(np.abs(got.reshape(-1, 8) - want8[None, :]) <= 1e-12)
    tb[1].zero_()
    out3 = torch.empty(3, dtype=torch.float64, device="cuda")
    qft.qft_fidelity_batched_static(tb.data_ptr(), ta.data_ptr(), n, 3, out3.data_ptr(), s)
    got3 = out3.cpu().numpy()
    assert abs(got3[0] - want8[0]) <= 1e-12 and abs(got3[2] - want8[2]) <= 1e-12  # the fidelity is symmetric
    assert np.isnan(got3[1])


def test_static_scratch_refuses_more_than_the_array_holds():
    """No GPU needed: the arguments are judged before any device is touched."""
    import paper_2606_18981_b200 as qft

    fake = 1 << 20  # aligned, never dereferenced
    with pytest.raises(qft.QftError) as ei:
        qft.qft_fidelity_batched_static(fake, fake, 4, qft.QFT_STATIC_MAX_BATCH + 1, fake)
    assert ei.value.status == qft.QFT_ERR_UNSUPPORTED
    assert str(qft.QFT_STATIC_MAX_BATCH) in str(ei.value) and "QFT_STATIC_MAX_BATCH" in str(ei.value)
    for bad in [(0, fake, 4, 1, fake), (fake, 0, 4, 1, fake), (fake, fake, 4, 1, 0), (fake + 8, fake, 4, 1, fake),
                (fake, fake, 4, 1, fake + 4), (fake, fake, 0, 1, fake), (fake, fake, 35, 1, fake), (fake, fake, 4, 0, fake),
                (fake, fake, 30, 32, fake)]:
        with pytest.raises(qft.QftError) as ei:
            qft.qft_fidelity_batched_static(*bad)
        assert ei.value.status == qft.QFT_ERR_INVALID_ARG, bad
        assert "qft_fidelity_batched_static" in qft.qft_static_last_error()
    hdr = open(os.path.join(ROOT, "include", "qft.h")).read()
    assert re.search(r"#define\s+QFT_STATIC_MAX_BATCH\s+%d\b" % qft.QFT_STATIC_MAX_BATCH, hdr)


def test_static_scratch_source_allocates_nothing():
    """The promise of the entry point, checked on its source with the comments removed: no allocating or freeing
    runtime call, the scratch is a static __device__ array, and its address comes from cudaGetSymbolAddress."""
    src = open(os.path.join(ROOT, "paper_2606_18981_b200", "csrc", "qft_metrics_static.cu")).read()
    code = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    code = re.sub(r"//[^\n]*", "", code)
    for word in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaMemPool", "cuMemAlloc", "cuMemCreate", "new ", "malloc("):
        assert word not in code, word
    assert re.search(r"static\s+__device__\s+__align__\(256\)\s+double\s+qft_static_sums\[QFT_STATIC_MAX_BATCH \* 4\]", code)
    assert "cudaGetSymbolAddress((void**)&p, qft_static_sums)" in code
    # host code hands kernels the looked-up address, never the symbol itself
    assert not re.search(r"<<<[^;]*qft_static_sums", code, flags=re.S)
