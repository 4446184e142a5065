"""the variants around the path, against the CPU oracle on the GPU.

  QFT_FLAG_DEFER_SWAPS   the paper's own mode: no swap network, the plan reports the layout it
                         left the qubits in; reference = the oracle's gate list WITHOUT its swap gates
                         (oracle.run_gates), re-indexed by the reported layout.
  qft_execute_oop        out of place: same result as in place, input untouched.
"""
import numpy as np
import pytest

import oracle
import qft_inputs as qi
from parity_bounds import assert_parity_numpy

pytestmark = pytest.mark.gpu


def _reindex(noswap, order):
    """stored[J] = noswap[j'],  bit order[a] of j' = bit a of J  (qft.h, QFT_FLAG_DEFER_SWAPS)."""
    n = len(order)
    J = np.arange(1 << n, dtype=np.int64)
    jp = np.zeros(1 << n, dtype=np.int64)
    for a, q in enumerate(order):
        jp |= ((J >> a) & 1) << q
    return noswap[jp]


@pytest.mark.parametrize("n", [9, 12, 16, 20, 23, 26])
def test_deferred_swaps_against_the_oracle_without_swap_gates(n):
    import torch

    import paper_2606_18981_b200 as qft

    x = qi.gaussian(n, 60 + n)
    for k, sign in ((n, -1), (4, -1), (7, 1)):
        gates = oracle.gate_list(n, k)
        gates = gates[gates[:, 0] != oracle.GATE_SWAP]
        noswap = oracle.run_gates(x, gates, sign)  # qubit q on bit q: the circuit's state before the swap network
        plan = qft.Plan(n, k, 13, sign, 0, 0, 0, qft.QFT_FLAG_DEFER_SWAPS)
        plan.self_check()
        d = plan.describe()
        assert d["swaps"] == "deferred" and all(not p["pair_swaps"] for p in d["passes"])
        order = plan.output_order()
        assert sorted(order) == list(range(n)) and order == d["out_qubit_of_bit"]
        t = torch.from_numpy(x).cuda()
        plan.execute(t)
        torch.cuda.synchronize()
        got = t.cpu().numpy().astype(np.complex128)
        assert_parity_numpy(got, _reindex(noswap, order), n, (n, k, sign, order))
        # and the caller's permutation gives the natural-order transform
        if k == n:
            K = np.arange(1 << n, dtype=np.int64)
            Jn = np.zeros(1 << n, dtype=np.int64)
            for a, q in enumerate(order):
                Jn |= ((K >> (n - 1 - q)) & 1) << a
            assert_parity_numpy(got[Jn], oracle.qft(x, k, sign), n, "caller-side permutation")
        # never more passes than the plan that applies the swaps
        ref_plan = qft.Plan(n, k, 13, sign)
        assert plan.num_passes <= ref_plan.num_passes
        ref_plan.close()
        plan.close()


@pytest.mark.parametrize("n", [8, 12, 15, 20, 26])
def test_out_of_place_execute(n):
    import torch

    import paper_2606_18981_b200 as qft

    x = qi.gaussian(n, 70 + n)
    for k, sign, flags in ((n, -1, 0), (5, 1, 0), (n, -1, qft.QFT_FLAG_DEFER_SWAPS)):
        plan = qft.Plan(n, k, 13, sign, 0, 0, 0, flags)
        src = torch.from_numpy(x).cuda()
        dst = torch.full((1 << n,), float("nan"), dtype=torch.complex64, device="cuda")
        plan.execute_oop(src, dst)
        inplace = torch.from_numpy(x).cuda()
        plan.execute(inplace)
        torch.cuda.synchronize()
        assert torch.equal(src.cpu(), torch.from_numpy(x)), "the input must be left untouched"
        assert torch.equal(dst, inplace), "same passes, same arithmetic: bit-identical to the in-place result"
        if flags == 0:
            assert_parity_numpy(dst.cpu().numpy(), oracle.qft(x, k, sign), n, (n, k, sign))
        plan.close()


def test_out_of_place_argument_checks():
    import torch

    import paper_2606_18981_b200 as qft

    plan = qft.Plan(12, 12)
    buf = torch.zeros(3 << 12, dtype=torch.complex64, device="cuda")
    with pytest.raises(qft.QftError):  # partial overlap
        qft.qft_execute_oop(plan.handle, buf.data_ptr(), buf.data_ptr() + 8 * 1024, 0)
    with pytest.raises(qft.QftError):  # misaligned
        qft.qft_execute_oop(plan.handle, buf.data_ptr() + 8, buf.data_ptr() + (8 << 13), 0)
    with pytest.raises(qft.QftError):
        qft.qft_execute_oop(plan.handle, 0, buf.data_ptr(), 0)
    plan.close()
