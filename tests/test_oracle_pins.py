"""Pins of the CPU oracle (oracle/) against what the paper and mathematics fix.

Nothing here touches the CUDA path.  Each test names the passage it pins.
"""
import os

import numpy as np
import pytest

import oracle
import qft_inputs as qi

GOLD = os.path.join(os.path.dirname(__file__), "golden")
RNG = np.random.default_rng(1234)


def rand_state(n, rng=RNG):
    x = rng.standard_normal(1 << n) + 1j * rng.standard_normal(1 << n)
    return x / np.linalg.norm(x)


def rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


# --------------------------------------------------------------------------
# Kronecker-product matrices written from PAPER.md:96-106, independent of the
# oracle's loops (numpy only).
# --------------------------------------------------------------------------
I2 = np.eye(2)
E1 = np.diag([1.0, 0.0])
E2 = np.diag([0.0, 1.0])
HM = np.array([[1, 1], [1, -1]]) / np.sqrt(2)  # Eq. 1 x 1/sqrt 2 (:138)


def one_wire(U, t, n):
    """I_{2^{n-1-t}} (x) U (x) I_{2^t}."""
    return np.kron(np.kron(np.eye(1 << (n - 1 - t)), U), np.eye(1 << t))


def two_wire_diag(c, t, m, n, sign):
    """controlled-R_m = E1 (x) I + E2 (x) R_m on wires c (control), t (target)
    (PAPER.md:105-106), embedded in n wires."""
    Rm = np.diag([1.0, np.exp(sign * 2j * np.pi / 2 ** m)])
    ops0 = [I2] * n
    ops1 = [I2] * n
    ops0[c] = E1
    ops1[c] = E2
    ops1[t] = Rm

    def chain(ops):  # wire n-1 is the leftmost Kronecker factor (MSB)
        M = np.eye(1)
        for q in range(n - 1, -1, -1):
            M = np.kron(M, ops[q])
        return M

    return chain(ops0) + chain(ops1)


def swap_matrix(a, b, n):
    N = 1 << n
    P = np.zeros((N, N))
    for j in range(N):
        ba, bb = (j >> a) & 1, (j >> b) & 1
        j2 = (j & ~((1 << a) | (1 << b))) | (bb << a) | (ba << b)
        P[j2, j] = 1
    return P


def circuit_matrix(n, k, sign=-1):
    """The range-k circuit of Fig. 1 as a dense matrix, gate by gate, from the
    paper's description -- NOT from oracle.gate_list."""
    M = np.eye(1 << n, dtype=complex)
    for t in range(n - 1, -1, -1):
        M = one_wire(HM, t, n) @ M
        for d in range(1, min(k, t) + 1):
            M = two_wire_diag(t - d, t, d + 1, n, sign) @ M
    for i in range(n // 2):
        M = swap_matrix(i, n - 1 - i, n) @ M
    return M


# --------------------------------------------------------------------------
# naive DFT = the definition; pinned to the library FFT
# --------------------------------------------------------------------------
@pytest.mark.parametrize("n", [0, 1, 2, 3, 5, 8, 10])
def test_naive_dft_matches_library_fft(n):
    x = rand_state(n) if n else np.array([0.3 - 0.7j])
    N = 1 << n
    assert rel(oracle.naive_dft(x, -1, oracle.NORM_NONE), np.fft.fft(x)) < 1e-13
    assert rel(oracle.naive_dft(x, -1, oracle.NORM_UNITARY), np.fft.fft(x) / np.sqrt(N)) < 1e-13
    assert rel(oracle.naive_dft(x, +1, oracle.NORM_INV_N), np.fft.ifft(x)) < 1e-13
    assert rel(oracle.naive_dft(x, +1, oracle.NORM_NONE), np.fft.ifft(x) * N) < 1e-13


def test_naive_dft_matrix_definition():
    """DFT_N = [omega^{k l}], omega = exp(-2 pi i / N)."""
    n, N = 4, 16
    W = np.exp(-2j * np.pi * np.outer(np.arange(N), np.arange(N)) / N)
    x = rand_state(n)
    assert rel(oracle.naive_dft(x, -1, oracle.NORM_NONE), W @ x) < 1e-13


# --------------------------------------------------------------------------
# single gates vs Kronecker matrices
# --------------------------------------------------------------------------
def test_hadamard_matches_kron():
    n = 5
    x = rand_state(n)
    for t in range(n):
        assert rel(oracle.apply_h(x, t), one_wire(HM, t, n) @ x) < 1e-14


def test_controlled_phase_matches_kron_and_is_symmetric():
    n = 5
    x = rand_state(n)
    for c in range(n):
        for t in range(n):
            if c == t:
                continue
            for m in (2, 3, 5):
                for sign in (-1, 1):
                    ref = two_wire_diag(c, t, m, n, sign) @ x
                    assert rel(oracle.apply_cr(x, c, t, m, sign), ref) < 1e-14
                    # controlled phase is symmetric in its two wires (reading c7)
                    assert rel(oracle.apply_cr(x, t, c, m, sign), ref) < 1e-14


def test_controlled_phase_value():
    """R_k = diag(1, e^{-2 pi i / 2^k}) on the |11> amplitude only."""
    x = np.array([1, 1, 1, 1], dtype=complex)
    y = oracle.apply_cr(x, 0, 1, 3, -1)
    assert np.allclose(y[:3], 1)
    assert abs(y[3] - np.exp(-2j * np.pi / 8)) < 1e-15


def test_swap_matches_permutation():
    n = 5
    x = rand_state(n)
    for a in range(n):
        for b in range(n):
            assert rel(oracle.apply_swap(x, a, b), swap_matrix(a, b, n) @ x) < 1e-15


# --------------------------------------------------------------------------
# gate list: Table 2, Fig. 1 worked circuit, n(n-1)/2
# --------------------------------------------------------------------------
def test_gate_counts_table2():
    rows = []
    with open(os.path.join(GOLD, "table2_cr_counts_n22.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            k, cnt, pct = line.split()
            rows.append((int(k), int(cnt), float(pct)))
    assert len(rows) == 7
    for k, cnt, pct in rows:
        g = oracle.gate_list(22, k)
        ncr = int(np.sum(g[:, 0] == oracle.GATE_CR))
        assert ncr == cnt
        assert abs(100.0 * ncr / 231 - pct) < 0.051
        assert int(np.sum(g[:, 0] == oracle.GATE_H)) == 22
        assert int(np.sum(g[:, 0] == oracle.GATE_SWAP)) == 11


def _parse_fig1():
    circuits, cur = {}, None
    with open(os.path.join(GOLD, "fig1_circuit_n3.txt")) as fh:
        for line in fh:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            if line.startswith("["):
                cur = int(line.strip("[]").split("=")[1])
                circuits[cur] = []
                continue
            p = line.split()
            if p[0] == "H":
                circuits[cur].append(("H", int(p[1])))
            elif p[0] == "CR":
                circuits[cur].append(("CR", int(p[1]), int(p[2]), int(p[3])))
            else:
                circuits[cur].append(("SWAP", int(p[1]), int(p[2])))
    return circuits


def _stages(gates):
    """Split a gate sequence at H gates; CRs inside a stage compared as a set."""
    out = []
    for g in gates:
        if g[0] == "H":
            out.append([g, set()])
        elif g[0] == "CR":
            out[-1][1].add(g)
        else:
            out.append([g, set()])
    return out


@pytest.mark.parametrize("k", [1, 2])
def test_gate_list_fig1(k):
    want = _parse_fig1()[k]
    got = []
    for ty, q0, q1, m in oracle.gate_list(3, k):
        if ty == oracle.GATE_H:
            got.append(("H", int(q0)))
        elif ty == oracle.GATE_CR:
            got.append(("CR", int(m), int(q0), int(q1)))
        else:
            got.append(("SWAP", int(q0), int(q1)))
    assert _stages(got) == _stages(want)


@pytest.mark.parametrize("n", [1, 2, 3, 7, 22, 33])
def test_exact_gate_count(n):
    """"With no cutoff (k = n-1), the n-wire circuit has n(n-1)/2 controlled phases"."""
    for k in (n - 1, n, n + 5):
        g = oracle.gate_list(n, k)
        assert int(np.sum(g[:, 0] == oracle.GATE_CR)) == n * (n - 1) // 2
    for k in range(0, n + 2):
        g = oracle.gate_list(n, k)
        want = sum(n - d for d in range(1, min(k, n - 1) + 1))
        assert int(np.sum(g[:, 0] == oracle.GATE_CR)) == want
        # every kept rotation has distance <= k and order m = d+1 <= k+1
        cr = g[g[:, 0] == oracle.GATE_CR]
        if len(cr):
            d = cr[:, 2] - cr[:, 1]
            assert d.min() >= 1 and d.max() <= k
            assert np.all(cr[:, 3] == d + 1)


def test_gate_order_constraints():
    """H(q_t) precedes every CR targeting q_t, which precedes H(q_c) (reading c7)."""
    g = oracle.gate_list(9, 4)
    hpos = {int(r[1]): i for i, r in enumerate(g) if r[0] == oracle.GATE_H}
    for i, r in enumerate(g):
        if r[0] == oracle.GATE_CR:
            assert hpos[int(r[2])] < i < hpos[int(r[1])]


# --------------------------------------------------------------------------
# whole circuit vs dense matrices and vs the naive DFT
# --------------------------------------------------------------------------
@pytest.mark.parametrize("n", [1, 2, 3, 4, 5])
def test_circuit_matches_dense_matrix_all_k(n):
    for sign in (-1, 1):
        for k in range(0, n + 1):
            M = circuit_matrix(n, k, sign)
            x = rand_state(n)
            assert rel(oracle.qft(x, k, sign), M @ x) < 1e-13
            assert np.allclose(M.conj().T @ M, np.eye(1 << n), atol=1e-13)  # unitary


def test_dft8_worked_example():
    """DFT_8 = three butterfly banks + diagonals T~_2^4, T~_2^8: the
    exact 3-wire circuit is DFT_8 / sqrt 8."""
    W = np.exp(-2j * np.pi * np.outer(np.arange(8), np.arange(8)) / 8) / np.sqrt(8)
    assert np.allclose(circuit_matrix(3, 2), W, atol=1e-14)
    for j in range(8):
        e = np.zeros(8, dtype=complex)
        e[j] = 1
        assert np.allclose(oracle.qft(e, 2), W[:, j], atol=1e-14)
    # k = 1 drops R3: NOT the DFT any more
    assert not np.allclose(circuit_matrix(3, 1), W, atol=1e-3)


@pytest.mark.parametrize("n", list(range(1, 11)))
def test_exact_qft_equals_naive_dft(n):
    x = qi.gaussian(n, 100 + n)
    for sign in (-1, 1):
        for norm in (0, 1, 2):
            a = oracle.qft(x, n, sign, norm)
            b = oracle.naive_dft(x, sign, norm)
            assert rel(a, b) < 1e-12


def test_exact_qft_equals_naive_dft_n12():
    x = qi.gaussian(12, 7)
    assert rel(oracle.qft(x, 12), oracle.naive_dft(x)) < 1e-12


def test_config1_equals_library_fft():
    """BASELINE config 1: n = 10, Gaussian seed 0 (secondary, library cross-check)."""
    x = qi.gaussian(10, 0)
    assert rel(oracle.qft(x), np.fft.fft(x.astype(np.complex128)) / 32.0) < 1e-13


# --------------------------------------------------------------------------
# fixed properties (north_star): delta, tone, Parseval, linearity, k >= n-1,
# AQFT error shrinks with k, k = 0
# --------------------------------------------------------------------------
def test_delta_gives_constant_magnitude_phase_ramp():
    n, idx = 12, 777
    N = 1 << n
    y = oracle.qft(qi.delta(n, idx))
    K = np.arange(N)
    want = np.exp(-2j * np.pi * ((idx * K) % N) / N) / np.sqrt(N)
    assert np.max(np.abs(y - want)) < 1e-14
    assert np.allclose(np.abs(y), 2.0 ** (-n / 2), atol=1e-15)


def test_tone_maps_to_single_index():
    """Single tone at bin k0 -> all energy in bin k0 (k0 = 2 is the paper's)."""
    n = 12
    for f in (2, 1234):
        y = oracle.qft(qi.tone(n, f).astype(np.complex128))
        e = np.zeros(1 << n)
        e[f] = 1
        assert np.max(np.abs(y - e)) < 1e-6  # complex64 input rounding
        N = 1 << n
        xd = np.exp(2j * np.pi * ((np.arange(N) * f) % N) / N) / np.sqrt(N)
        assert np.max(np.abs(oracle.qft(xd) - e)) < 1e-13


@pytest.mark.parametrize("k", [0, 1, 3, 6, 11])
def test_parseval_every_k(k):
    n = 11
    x = qi.gaussian(n, 5)
    nx = np.linalg.norm(x.astype(np.complex128))
    assert abs(np.linalg.norm(oracle.qft(x, k)) - nx) < 1e-13
    assert abs(np.linalg.norm(oracle.qft(x, k, -1, 1)) - nx * np.sqrt(1 << n)) < 1e-10
    assert abs(np.linalg.norm(oracle.qft(x, k, -1, 2)) - nx / np.sqrt(1 << n)) < 1e-15


def test_linearity():
    n = 10
    a, b = rand_state(n), rand_state(n)
    al, be = 0.3 - 1.1j, -2.0 + 0.25j
    for k in (2, n):
        lhs = oracle.qft(al * a + be * b, k)
        rhs = al * oracle.qft(a, k) + be * oracle.qft(b, k)
        assert rel(lhs, rhs) < 1e-14


def test_k_ge_n_minus_1_is_exact_bitwise():
    n = 9
    x = qi.gaussian(n, 3)
    ref = oracle.qft(x, n - 1)
    for k in (n, n + 3, 40):
        assert np.array_equal(oracle.qft(x, k), ref)
    assert not np.array_equal(oracle.qft(x, n - 2), ref)


def test_aqft_error_shrinks_with_k():
    n = 12
    x = qi.gaussian(n, 11)
    exact = oracle.qft(x, n)
    errs = [rel(oracle.qft(x, k), exact) for k in range(0, n)]
    # k = 0, 1 are saturated (error ~ sqrt 2, the distance of two unrelated unit vectors);
    # from there on the error falls strictly with k
    assert all(e1 > e2 for e1, e2 in zip(errs[2:], errs[3:]))
    assert errs[-1] == 0.0
    # tail ~ 2^-k: roughly halves per extra k
    for k in range(3, n - 3):
        assert 1.5 < errs[k] / errs[k + 1] < 3.2


def test_aqft_fidelity_and_leakage_single_tone():
    """1-F and top-bin leakage fall with k and coincide for a single tone;
    magnitude ~ (4 pi^2 / 3) 4^-(k+2) (derived in SURVEY.md 8(c), consistency only)."""
    n, f = 14, 2
    N = 1 << n
    x = np.exp(2j * np.pi * ((np.arange(N) * f) % N) / N) / np.sqrt(N)
    exact = oracle.qft(x, n)
    prev = None
    for k in (2, 4, 6, 8):
        y = oracle.qft(x, k)
        F = abs(np.vdot(exact, y)) ** 2 / (np.vdot(y, y).real * np.vdot(exact, exact).real)
        leak = 1 - abs(y[f]) ** 2 / np.vdot(y, y).real
        assert abs((1 - F) - leak) < 1e-12
        pred = (4 * np.pi ** 2 / 3) * 4.0 ** (-(k + 2))
        assert 0.5 * pred < leak < 2.0 * pred
        if prev is not None:
            assert leak < prev
        prev = leak


def test_k0_is_walsh_hadamard_then_bit_reversal():
    from scipy.linalg import hadamard

    n = 8
    N = 1 << n
    x = rand_state(n)
    wht = hadamard(N) @ x / np.sqrt(N)  # natural (Hadamard) order, textbook routine
    rev = np.array([int(format(j, "0%db" % n)[::-1], 2) for j in range(N)])
    want = np.empty(N, dtype=complex)
    want[rev] = wht
    assert rel(oracle.qft(x, 0), want) < 1e-13


def test_exact_round_trip():
    n = 10
    x = qi.gaussian(n, 9).astype(np.complex128)
    y = oracle.qft(oracle.qft(x, n, -1), n, +1)
    assert rel(y, x) < 1e-13


# --------------------------------------------------------------------------
# closed forms for AQFT (any k), obtained by factorising the sum over input bits
# --------------------------------------------------------------------------
def aqft_tone_closed_form(n, k, f, K):
    """out[K] for x_j = N^-1/2 exp(2 pi i f j / N), forward sign: the sum over j
    factorises over the bits of j:  prod_c (1 + exp(2 pi i alpha_c)) / 2,
    alpha_c = f 2^c / N - sum_{t=c}^{min(n-1,c+k)} y_t 2^{c-t-1}, y_t = bit n-1-t of K."""
    N = 1 << n
    out = 1.0 + 0j
    for c in range(n):
        al = ((f << c) % N) / N
        for t in range(c, min(n - 1, c + k) + 1):
            if (K >> (n - 1 - t)) & 1:
                al -= 2.0 ** (c - t - 1)
        out *= (1 + np.exp(2j * np.pi * al)) / 2
    return out


def aqft_delta_closed_form(n, k, j0, K, sign=-1):
    """<K| AQFT_k |j0> = N^-1/2 exp(sign 2 pi i sum_t y_t tr_{k,t}(j0) / 2^{t+1}),
    tr_{k,t}(j) = (j mod 2^{t+1}) with the bits below t-k cleared."""
    ph = 0.0
    for t in range(n):
        if (K >> (n - 1 - t)) & 1:
            tr = j0 & ((1 << (t + 1)) - 1)
            if t - k > 0:
                tr &= ~((1 << (t - k)) - 1)
            ph += tr / 2.0 ** (t + 1)
    return np.exp(sign * 2j * np.pi * ph) / np.sqrt(1 << n)


@pytest.mark.parametrize("k", [0, 1, 2, 4, 7, 8])
def test_aqft_closed_forms(k):
    n = 8
    N = 1 << n
    for f in (2, 77, 200):
        x = np.exp(2j * np.pi * ((np.arange(N) * f) % N) / N) / np.sqrt(N)
        y = oracle.qft(x, k)
        want = np.array([aqft_tone_closed_form(n, k, f, K) for K in range(N)])
        assert np.max(np.abs(y - want)) < 1e-13
    for j0 in (0, 1, 77, 255):
        for sign in (-1, 1):
            y = oracle.qft(qi.delta(n, j0), k, sign)
            want = np.array([aqft_delta_closed_form(n, k, j0, K, sign) for K in range(N)])
            assert np.max(np.abs(y - want)) < 1e-14


def test_multi_tone_exact_closed_form():
    n = 11
    N = 1 << n
    fr, ph = qi.tone_params(n, 3, 5)
    assert len(set(fr.tolist())) == 5
    x = qi.multi_tone(n, fr, ph)
    y = oracle.qft(x)
    want = np.zeros(N, dtype=complex)
    want[fr] = np.exp(1j * ph) / np.sqrt(5)
    assert np.max(np.abs(y - want)) < 1e-6  # complex64 input rounding


# --------------------------------------------------------------------------
# sampled-output routine (matrix elements) vs the gate-by-gate circuit
# --------------------------------------------------------------------------
@pytest.mark.parametrize("k", [0, 2, 5, 9])
def test_outputs_at_matches_circuit(k):
    n = 9
    x = qi.gaussian(n, 21)
    Ks = np.array([0, 1, 77, 300, 511])
    for sign in (-1, 1):
        for norm in (0, 1, 2):
            full = oracle.qft(x, k, sign, norm)
            got = oracle.outputs_at(x, Ks, k, sign, norm)
            assert np.max(np.abs(got - full[Ks])) < 1e-13 * max(1.0, np.max(np.abs(full)))


# --------------------------------------------------------------------------
# seeded input recipes
# --------------------------------------------------------------------------
def test_input_recipes():
    x = qi.gaussian(10, 0)
    assert x.dtype == np.complex64 and x.shape == (1024,)
    assert abs(np.linalg.norm(x.astype(np.complex128)) - 1) < 1e-6
    assert np.array_equal(x, qi.gaussian(10, 0))
    t = qi.tone(10, 5)
    assert abs(np.linalg.norm(t.astype(np.complex128)) - 1) < 1e-6
    d = qi.delta(10, 777)
    assert d[777] == 1 and np.count_nonzero(d) == 1


def test_metric_definitions_closed_forms():
    """Pins of oracle.norm_sq / encode / fidelity / leakage to cases with a known value."""
    rng = np.random.default_rng(11)
    a = rng.normal(size=64) + 1j * rng.normal(size=64)
    assert abs(oracle.norm_sq([3 + 4j, 0, 12j]) - 169.0) < 1e-12          # 3-4-5 and 5-12-13
    e, s = oracle.encode([3 + 4j, 0, 12j])
    assert abs(s - 13.0) < 1e-12 and abs(oracle.norm_sq(e) - 1.0) < 1e-12
    assert abs(oracle.fidelity(a, a) - 1.0) < 1e-12
    assert abs(oracle.fidelity(a, (2 - 3j) * a) - 1.0) < 1e-12            # insensitive to scale and global phase
    u = np.zeros(8, complex); v = np.zeros(8, complex); u[1] = 1; v[5] = 1j
    assert oracle.fidelity(u, v) == 0.0                                     # orthogonal states
    assert abs(oracle.fidelity(u, (u + v) / np.sqrt(2)) - 0.5) < 1e-12
    assert oracle.leakage(u, 1) == 0.0 and oracle.leakage(u, 2) == 1.0
    assert abs(oracle.leakage([1, 1, 1, 1], 3) - 0.75) < 1e-12
    # for a single-tone input the AQFT's infidelity against the exact output equals its top-bin leakage
    n, f = 8, 2
    x = qi.tone(n, f)
    exact = oracle.qft(x)
    for k in (2, 4):
        out = oracle.qft(x, k)
        assert abs((1.0 - oracle.fidelity(exact, out)) - oracle.leakage(out, f)) < 1e-7  # complex64 input rounding


def test_aqft_matrix_is_symmetric_so_conjugate_is_inverse():
    """DESIGN.md reading c12: the (A)QFT matrix including the swaps is symmetric for every cutoff k
    (H and CR are symmetric, the kept rotations are invariant under q -> n-1-q, the reversed gate list is
    the same circuit on the reversed qubit order), hence its inverse is its complex conjugate: sign = +1
    undoes sign = -1 with the same k.  Checked on the oracle's full matrix and by round trips."""
    for n in (1, 2, 3, 4, 6):
        N = 1 << n
        eye = np.eye(N, dtype=np.complex128)
        for k in range(0, n + 1):
            A = np.stack([oracle.qft(eye[j], k) for j in range(N)], axis=1)      # columns = images of basis states
            assert np.abs(A - A.T).max() < 1e-14
            assert np.abs(A.conj().T @ A - eye).max() < 1e-13                     # unitary
            B = np.stack([oracle.qft(eye[j], k, sign=1) for j in range(N)], axis=1)
            assert np.abs(B - A.conj()).max() < 1e-14
            assert np.abs(B @ A - eye).max() < 1e-13
    x = qi.gaussian(10, 3).astype(np.complex128)
    for k in (0, 1, 3, 5):
        assert np.linalg.norm(oracle.qft(oracle.qft(x, k), k, sign=1) - x) < 1e-13
