"""CPU-only checks of libqft.so: it loads, exports every symbol of include/qft.h, validates
arguments, and its planner's schedules pass the host-side proof (no kernel is launched here)."""
import ctypes
import os
import re

import pytest

import paper_2606_18981_b200 as qft

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "qft.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(qft_[a-z_]+)\s*\(", hdr))
    assert {"qft_plan_create", "qft_execute", "qft_plan_destroy"} <= declared
    lib = ctypes.CDLL(qft.LIB_PATH)
    for name in sorted(declared):
        assert hasattr(lib, name), name
    assert declared == set(qft.EXPORTS)


def test_status_strings():
    assert qft.qft_status_string(0) == "ok"
    for s in range(1, 6):
        assert qft.qft_status_string(s) not in ("ok", "unknown status")


@pytest.mark.parametrize("args", [
    (0, 1, 13, -1, 0), (35, 1, 13, -1, 0), (10, -1, 13, -1, 0), (10, 3, 0, -1, 0), (10, 3, 13, 0, 0),
    (10, 3, 13, 2, 0), (10, 3, 13, -1, 3), (10, 3, 13, -1, -1),
])
def test_invalid_arguments(args):
    with pytest.raises(qft.QftError) as e:
        qft.qft_plan_create(*args)
    assert e.value.status == qft.QFT_ERR_INVALID_ARG


def test_null_out_pointer_and_null_plan():
    L = qft.load()
    assert L.qft_plan_create(None, 10, 10, 13, -1, 0) == qft.QFT_ERR_INVALID_ARG
    assert L.qft_execute(None, None, None) == qft.QFT_ERR_INVALID_ARG
    assert L.qft_plan_num_passes(None) == -1
    assert L.qft_plan_destroy(None) == qft.QFT_OK
    h = qft.qft_plan_create(10, 10)
    assert L.qft_execute(h, None, None) == qft.QFT_ERR_INVALID_ARG
    assert L.qft_execute(h, ctypes.c_void_p(8), None) == qft.QFT_ERR_INVALID_ARG  # misaligned
    small = ctypes.create_string_buffer(8)
    assert L.qft_plan_describe(h, small, 8) == qft.QFT_ERR_INVALID_ARG
    qft.qft_plan_destroy(h)


def test_unsupported_tuning():
    with pytest.raises(qft.QftError) as e:
        qft.qft_plan_create_tuned(10, 10, 13, -1, 0, tile_bits=15)
    assert e.value.status == qft.QFT_ERR_UNSUPPORTED
    with pytest.raises(qft.QftError):
        qft.qft_plan_create_tuned(34, 10, 13, -1, 0, tile_bits=2, hub_bits=1)


def test_gate_counters_table2():
    """The plan carries the 1- and 2-qubit gate counters before fusion;
    Table 2 fixes the controlled-R_m count at n = 22."""
    with open(os.path.join(GOLD, "table2_cr_counts_n22.txt")) as fh:
        rows = [tuple(l.split()) for l in fh if l.strip() and not l.startswith("#")]
    for k, cnt, _ in rows:
        p = qft.Plan(22, int(k))
        assert p.gate_counts() == (22, int(cnt), 11)
        p.close()
    p = qft.Plan(30, 30)
    assert p.gate_counts() == (30, 435, 15)
    p.close()
    p = qft.Plan(33, 16)
    assert p.gate_counts() == (33, 392, 16)
    p.close()


@pytest.mark.parametrize("n", list(range(1, 35)))
def test_every_schedule_passes_the_host_proof(n):
    for w in (1, 2, 3, 4, 6, 10, 13, 40):
        for flags in (0, qft.QFT_FLAG_UNFOLDED):
            p = qft.Plan(n, n, w, flags=flags)
            p.self_check()
            d = p.describe()
            assert d["n"] == n and len(d["passes"]) == p.num_passes
            done = []
            for ps in d["passes"]:
                assert len(ps["window"]) <= max(1, min(w, 13))
                done += ps["window"]
            assert done == list(range(n - 1, -1, -1))  # circuit order, every qubit once
            p.close()


@pytest.mark.parametrize("tile_bits,hub_bits", [(4, 1), (5, 2), (6, 2), (7, 3), (9, 3), (12, 4), (14, 3), (14, 4)])
def test_tuned_schedules_pass_the_host_proof(tile_bits, hub_bits):
    for n in range(1, 31):
        for w in (1, 3, 13):
            for flags in (0, qft.QFT_FLAG_UNFOLDED):
                p = qft.Plan(n, 5, w, tile_bits=tile_bits, hub_bits=hub_bits, flags=flags)
                p.self_check()
                p.close()


def test_pass_counts_at_the_bench_configs():
    """Folded schedule: ceil(n / window) passes with no stand-alone bit-reversal pass."""
    # (n = 13 would fit one 2^13 tile, but one 8192-amplitude CTA is slower than three multi-CTA passes on
    # 2^12 tiles: 30 us vs 17 us on a B200, so the planner's default takes the latter)
    want = {10: 1, 12: 1, 13: 3, 20: 3, 26: 3, 30: 3, 33: 3, 34: 4}
    for n, passes in want.items():
        p = qft.Plan(n, n)
        assert p.num_passes == passes, n
        assert p.num_launches == passes
        p.close()
    # config 3: sweep of max_fused_qubits at n = 26
    # (ceil(26 / w) passes, every one of them in the TMA-staged kernel: small windows are sub-passes of the folded
    # schedule's windows, not the natural-order schedule with its stand-alone reversal)
    got = []
    for w in (2, 4, 6, 10, 13):
        p = qft.Plan(26, 26, w)
        got.append(p.num_passes)
        assert {ps["kernel"] for ps in p.describe()["passes"]} == {"tma2"}, w
        p.close()
    assert got == [13, 7, 5, 3, 3]


def test_k_is_clamped_and_reported():
    p = qft.Plan(12, 1000)
    assert p.describe()["k"] == 12
    assert p.gate_counts()[1] == 66
    p.close()


def test_deferred_swaps_plans():
    """QFT_FLAG_DEFER_SWAPS: the host proof holds for every n, the reported layout is a permutation of the qubits, no
    pass exchanges tiles between CTAs, and there are never more passes than with the swaps applied."""
    for n in range(1, 35):
        for w in (13, 4):
            p = qft.Plan(n, 6, w, flags=qft.QFT_FLAG_DEFER_SWAPS)
            p.self_check()
            d = p.describe()
            assert d["swaps"] == "deferred"
            assert sorted(p.output_order()) == list(range(n))
            assert all(not ps["pair_swaps"] for ps in d["passes"])
            q = qft.Plan(n, 6, w)
            assert q.output_order() == [n - 1 - a for a in range(n)] and q.describe()["swaps"] == "applied"
            if w == 13:
                assert p.num_passes <= q.num_passes
            p.close()
            q.close()
    b = qft.qft_plan_create_batched(12, 4, 12, 13, -1, 0)  # sanity: batched plans exist ...
    assert qft.qft_plan_output_order(b) == [11 - a for a in range(12)]  # ... and report the per-state order
    with pytest.raises(ValueError):
        qft.qft_plan_output_order(b, 3)  # a caller's wrong idea of n is refused, not written past
    qft.qft_plan_destroy(b)
    with pytest.raises(qft.QftError) as ei:
        qft.qft_plan_create_tuned(12, 12, 13, -1, 0, 0, 0, qft.QFT_FLAG_DEFER_SWAPS | qft.QFT_FLAG_UNFOLDED)
    assert ei.value.status == qft.QFT_ERR_UNSUPPORTED


def test_passes_name_their_gates():
    """PAPER.md:145 / :147: every fused block records the contiguous sub-range of the time-ordered gate list it folds.
    The ranges must tile the list [0, n_h + n_cr) in order, and their H / CR counts must add up to the plan's counters,
    i.e. to Table 2's seven rows at n = 22."""
    table2 = {21: 231, 16: 216, 12: 186, 10: 165, 8: 140, 6: 111, 4: 78}
    for k, n_cr in table2.items():
        for w, flags in ((13, 0), (3, 0), (13, qft.QFT_FLAG_UNFOLDED), (5, qft.QFT_FLAG_DEFER_SWAPS)):
            p = qft.Plan(22, k, w, flags=flags)
            d = p.describe()
            nxt, th, tc = 0, 0, 0
            for ps in d["passes"]:
                if ps["n_h"] == 0:
                    assert ps["gate_first"] == -1 and not ps["window"]  # permutation only: part of the swap network
                    continue
                assert ps["gate_first"] == nxt and ps["gate_last"] == nxt + ps["n_h"] + ps["n_cr"] - 1
                assert ps["n_h"] == len(ps["window"])
                assert ps["n_cr"] == sum(min(k, t) for t in ps["window"])
                nxt = ps["gate_last"] + 1
                th += ps["n_h"]
                tc += ps["n_cr"]
            assert (th, tc) == (22, n_cr) and nxt == 22 + n_cr
            assert p.gate_counts() == (22, n_cr, 11)
            p.close()
    # the n = 30 bench plan: three fused blocks of 10 Hadamards each
    p = qft.Plan(30, 30)
    assert [(ps["n_h"], ps["n_cr"]) for ps in p.describe()["passes"]] == [(10, 245), (10, 145), (10, 45)]
    p.close()


def test_unschedulable_tuning_is_unsupported_not_internal():
    """tile_bits < 2 * hub_bits cannot hold the hub beside a window (or twice, in the stand-alone
    reversal tile); qft.h promises QFT_ERR_UNSUPPORTED for that, never QFT_ERR_INTERNAL."""
    for tile_bits, hub_bits in ((3, 2), (4, 3), (5, 3), (5, 4), (6, 4), (7, 4), (8, 5), (9, 5)):
        for flags in (0, qft.QFT_FLAG_UNFOLDED):
            with pytest.raises(qft.QftError) as ei:
                qft.qft_plan_create_tuned(20, 20, 13, -1, 0, tile_bits, hub_bits, flags)
            assert ei.value.status == qft.QFT_ERR_UNSUPPORTED
    # fuzz: whatever the knobs, the planner answers ok / unsupported / invalid, never "internal"
    import random

    rng = random.Random(5)
    for _ in range(1500):
        n, t, h = rng.randint(1, 34), rng.randint(0, 15), rng.randint(0, 7)
        w, fl = rng.randint(1, 14), rng.choice([0, 1, 2, 4, 16, 32, 6, 17, 33])
        try:
            qft.qft_plan_destroy(qft.qft_plan_create_tuned(n, rng.randint(0, 40), w, -1, 0, t, h, fl))
        except qft.QftError as e:
            assert e.status in (qft.QFT_ERR_UNSUPPORTED, qft.QFT_ERR_INVALID_ARG), (n, t, h, w, fl, str(e))


def test_describe_length_and_small_buffers():
    import ctypes

    L = qft.load()
    p = qft.Plan(34, 34, 1)  # 35 passes: the longest description
    need = qft.qft_plan_describe_length(p.handle)
    assert need > 8192
    small = ctypes.create_string_buffer(need - 1)
    assert L.qft_plan_describe(p.handle, small, need - 1) == qft.QFT_ERR_INVALID_ARG
    exact = ctypes.create_string_buffer(need)
    assert L.qft_plan_describe(p.handle, exact, need) == qft.QFT_OK and len(exact.value) == need - 1
    assert qft.qft_plan_describe_length(None) == 0
    p.close()


def test_num_qubits_for_length():
    assert [qft.qft_num_qubits_for(v) for v in (1, 2, 3, 4, 5, 1000, 1024, 1025)] == [1, 1, 2, 2, 3, 10, 10, 11]
    assert qft.qft_num_qubits_for(0) == -1 and qft.qft_num_qubits_for((1 << 34) + 1) == -1
