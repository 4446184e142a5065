"""GPU parity of the TMA-staged pass kernel (tma2) against the CPU oracle, element by element.

The sizes (n = 20 ... 24) are the smallest at which the planner emits tma2 passes, chosen so that the
tile / hub knobs of qft_plan_create_tuned put it in every position (first pass with the hub swap, mid
pass with the 2-CTA-cluster pair store, last pass with the scale), with every register-group shape
(4+3, 4+4, 5+4, 5+5 only at n >= 28: tests/test_gpu_large.py) and every in-group AQFT truncation
(k = 0 ... 3 and k >= 4 are separate kernel instantiations).  Tolerance: north_star's 2e-5 (n <= 20),
1e-4 above.
"""
import numpy as np
import pytest

import oracle
import qft_inputs as qi
from parity_bounds import assert_parity_numpy

pytestmark = pytest.mark.gpu

CFGS = [(20, 12, 3), (20, 13, 3), (21, 12, 4), (22, 13, 3), (22, 13, 4), (22, 12, 4), (23, 14, 4), (24, 13, 3),
        (24, 14, 4), (24, 12, 3), (24, 12, 4)]
VARIANTS = [(None, -1, 0), (3, -1, 0), (1, 1, 1), (None, 1, 2), (0, -1, 0), (2, -1, 0), (9, -1, 0)]


@pytest.mark.parametrize("n,tile_bits,hub_bits", CFGS)
def test_tma2_against_oracle(n, tile_bits, hub_bits):
    import torch

    import paper_2606_18981_b200 as qft

    x = qi.gaussian(n, n)
    saw_tma2 = False
    for k, sign, norm in VARIANTS:
        kk = n if k is None else k
        plan = qft.Plan(n, kk, 13, sign, norm, tile_bits, hub_bits, 0)
        plan.self_check()
        kinds = [p["kernel"] for p in plan.describe()["passes"]]
        saw_tma2 |= "tma2" in kinds
        t = torch.from_numpy(x).cuda()
        plan.execute(t)
        torch.cuda.synchronize()
        got = t.cpu().numpy().astype(np.complex128)
        plan.close()
        ref = oracle.qft(x, kk, sign, norm)
        assert_parity_numpy(got, ref, n, (n, tile_bits, hub_bits, kk, sign, norm, kinds))
    assert saw_tma2, "this configuration was chosen to exercise the tma2 kernel"


# tensor-memory extended tiles (kernel "tma2x"): the smallest sizes at which the planner emits them are n = 25 with
# 512-byte granules (hub 6: windows 9 = 4+4+1) and n = 28 with 256-byte granules (hub 5: 5+4+1, the bench's kernels;
# tests/test_gpu_large.py); the 5+5+1 shape needs n >= 31 and is checked there against the closed forms.
@pytest.mark.parametrize("n,hub_bits", [(25, 6), (26, 6), (27, 6)])
def test_tma2x_against_oracle(n, hub_bits):
    import torch

    import paper_2606_18981_b200 as qft

    x = qi.gaussian(n, n)
    for k, sign, norm in [(None, -1, 0), (3, 1, 0), (12, -1, 1), (0, -1, 0), (1, -1, 2)]:
        kk = n if k is None else k
        plan = qft.Plan(n, kk, 13, sign, norm, 14, hub_bits, 0)
        plan.self_check()
        kinds = [p["kernel"] for p in plan.describe()["passes"]]
        assert "tma2x" in kinds
        t = torch.from_numpy(x).cuda()
        plan.execute(t)
        torch.cuda.synchronize()
        got = t.cpu().numpy().astype(np.complex128)
        plan.close()
        assert_parity_numpy(got, oracle.qft(x, kk, sign, norm), n, (n, hub_bits, kk, sign, norm, kinds))
        # the same transform without the extension (one pass more or smaller windows) must agree
        if k is None:
            plain = qft.Plan(n, kk, 13, sign, norm, 14, hub_bits, qft.QFT_FLAG_NO_EXT_TILE)
            assert "tma2x" not in [p["kernel"] for p in plain.describe()["passes"]]
            t2 = torch.from_numpy(x).cuda()
            plain.execute(t2)
            torch.cuda.synchronize()
            plain.close()
            assert float(np.linalg.norm(t2.cpu().numpy() - got) / np.linalg.norm(got)) <= 2e-6


def test_tma2_matches_generic_kernel_bitwise_layout():
    """Same plan with and without the fused kernels (flags = QFT_FLAG_GENERIC_ONLY): the generic
    shared-memory kernel is the slow reference implementation of the same pass list, so the two
    results must agree to rounding; a tone input must land in one bin."""
    import torch

    import paper_2606_18981_b200 as qft

    n = 25
    x = qi.tone(n, 12345)
    outs = []
    for flags in (0, qft.QFT_FLAG_GENERIC_ONLY):
        plan = qft.Plan(n, n, 13, -1, 0, 13, 4, flags)
        t = torch.from_numpy(x).cuda()
        plan.execute(t)
        torch.cuda.synchronize()
        outs.append(t)
        plan.close()
    d = float(torch.linalg.vector_norm(outs[0] - outs[1]).item())
    assert d <= 1e-5
    peak = int(torch.argmax(outs[0].abs()).item())
    assert peak == 12345
    assert abs(abs(outs[0][peak].item()) - 1.0) <= 1e-4


def test_plan_reuse_across_streams_and_states():
    """A plan is immutable and reusable (include/qft.h): the same plan on two streams, two states in
    flight at once, several executes back to back (programmatic dependent launch between the passes),
    then exact-k round trip sign=-1 / sign=+1 back to the input."""
    import torch

    import paper_2606_18981_b200 as qft

    n = 21
    xa, xb = qi.gaussian(n, 1), qi.gaussian(n, 2)
    fwd = qft.Plan(n, n)
    inv = qft.Plan(n, n, sign=1)
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    ta, tb = torch.from_numpy(xa).cuda(), torch.from_numpy(xb).cuda()
    torch.cuda.synchronize()
    for _ in range(3):
        fwd.execute(ta, sa.cuda_stream)
        fwd.execute(tb, sb.cuda_stream)
        inv.execute(ta, sa.cuda_stream)
        inv.execute(tb, sb.cuda_stream)
    fwd.execute(ta, sa.cuda_stream)
    torch.cuda.synchronize()
    ref = oracle.qft(xa)
    got = ta.cpu().numpy().astype(np.complex128)
    # seven transforms in a row on ta, six on tb: rounding adds in quadrature (about sqrt(7) x 3e-7), inside the bounds
    assert_parity_numpy(got, ref, n, "reuse across streams: forward after three round trips")
    back = tb.cpu().numpy().astype(np.complex128)
    assert_parity_numpy(back, xb.astype(np.complex128), n, "reuse across streams: three round trips")
    fwd.close()
    inv.close()


def test_execute_is_cuda_graph_capturable():
    """qft_execute only enqueues kernels (tensor maps are kernel parameters encoded on the host), so a whole
    transform can be captured into a CUDA graph and replayed - the launch-bound regime of the paper's sizes."""
    import torch

    import paper_2606_18981_b200 as qft

    n = 18
    x = qi.gaussian(n, 4)
    plan = qft.Plan(n, n)
    t = torch.from_numpy(x).cuda()
    s = torch.cuda.Stream()
    plan.execute(t, s.cuda_stream)  # warm-up outside the capture
    torch.cuda.synchronize()
    t.copy_(torch.from_numpy(x).cuda())
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s):
        plan.execute(t, s.cuda_stream)
    g.replay()
    torch.cuda.synchronize()
    ref = oracle.qft(x)
    got = t.cpu().numpy().astype(np.complex128)
    assert_parity_numpy(got, ref, n, "graph replay")
    # replay on fresh data gives the transform of the fresh data
    y = qi.gaussian(n, 5)
    t.copy_(torch.from_numpy(y).cuda())
    g.replay()
    torch.cuda.synchronize()
    ref = oracle.qft(y)
    got = t.cpu().numpy().astype(np.complex128)
    assert_parity_numpy(got, ref, n, "graph replay on fresh data")
    plan.close()


# Small max_fused_qubits (BASELINE config 3 sweeps it down to 2): the planner cuts the folded schedule's windows into
# sub-passes that run on large tiles, so a small window high up in the tile sees up to 12 in-tile qubits below it
# (the split end table of the TMA kernel: more than 7).  Every sub-window shape (1+1, 2+1, 2+2, 3+2, 3+3), three tile
# sizes, exact and truncated rotations, both signs.
@pytest.mark.parametrize("n,tile_bits", [(18, 12), (20, 13), (21, 13), (22, 14), (23, 12), (24, 14)])
@pytest.mark.parametrize("w", [2, 3, 4, 5, 6])
def test_small_windows_against_oracle(n, tile_bits, w):
    import torch

    import paper_2606_18981_b200 as qft

    x = qi.gaussian(n, 100 + n)
    deepest = 0
    for k, sign, norm in [(None, -1, 0), (3, 1, 1), (1, -1, 0), (7, -1, 2)]:
        kk = n if k is None else k
        plan = qft.Plan(n, kk, w, sign, norm, tile_bits, 0, 0)
        plan.self_check()
        passes = plan.describe()["passes"]
        kinds = [p["kernel"] for p in passes]
        assert all(len(p["window"]) <= w for p in passes)
        for p in passes:
            if p["kernel"] == "tma2":
                deepest = max(deepest, sum(1 for q in p["canon_qubits"] if q < min(p["window"])))
        t = torch.from_numpy(x).cuda()
        plan.execute(t)
        torch.cuda.synchronize()
        got = t.cpu().numpy().astype(np.complex128)
        plan.close()
        assert_parity_numpy(got, oracle.qft(x, kk, sign, norm), n, (n, tile_bits, w, kk, sign, norm, kinds))
    if w <= 4:
        assert deepest > 7, "this configuration was chosen to exercise the split end table"

