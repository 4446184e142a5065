"""Batched plans (qft_plan_create_batched): 2^b independent n-qubit transforms
stored back to back, one set of launches.  CPU: the planner's self-check over a grid.  GPU: every state
against the CPU oracle, element by element (the three bounds of tests/parity_bounds.py, per state)."""
import numpy as np
import pytest

import oracle
import qft_inputs as qi
from parity_bounds import assert_parity_numpy


def test_batched_plans_self_check_grid():
    import paper_2606_18981_b200 as qft

    for n in range(1, 23):
        for b in range(0, min(12, 34 - n) + 1):
            for k in (n, 2):
                p = qft.Plan(n, k, log2_batch=b)
                p.self_check()
                d = p.describe()
                assert d["n"] == n and d["batch_bits"] == b
                assert p.gate_counts()[0] == n  # counters are per transform
                p.close()
    with pytest.raises(qft.QftError):
        qft.Plan(30, 30, log2_batch=5)  # 35 address bits
    with pytest.raises(qft.QftError):
        qft.Plan(10, 10, log2_batch=-1)


@pytest.mark.gpu
@pytest.mark.parametrize("n,b", [(1, 3), (3, 5), (6, 10), (8, 12), (9, 9), (10, 10), (10, 1), (12, 6), (13, 5),
                                 (14, 4), (16, 4), (18, 3), (20, 2), (21, 1)])
def test_batched_against_oracle(n, b):
    import torch

    import paper_2606_18981_b200 as qft

    B = 1 << b
    xs = np.stack([qi.gaussian(n, 100 * n + i) for i in range(min(B, 8))])
    # cycle the distinct inputs through the batch so that every slot is checked against a known state
    idx = np.arange(B) % xs.shape[0]
    state = np.ascontiguousarray(xs[idx].reshape(-1))
    for k, sign, norm in ((n, -1, 0), (2, 1, 1)):
        refs = np.stack([oracle.qft(x, k, sign, norm) for x in xs])
        plan = qft.Plan(n, k, 13, sign, norm, log2_batch=b)
        plan.self_check()
        t = torch.from_numpy(state).cuda()
        plan.execute(t)
        torch.cuda.synchronize()
        got = t.cpu().numpy().astype(np.complex128).reshape(B, 1 << n)
        plan.close()
        ref = refs[idx]
        for slot in range(B):  # every state of the batch against the three bounds of parity_bounds
            assert_parity_numpy(got[slot], ref[slot], n, (n, b, k, sign, norm, slot))
