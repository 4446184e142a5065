/*
 * qft_oracle.c -- TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, obviously-correct double-precision state-vector simulator of
 * the QFT / AQFT circuit of arxiv/paper_2606_18981 ("Not Your Usual FFT"),
 * written from the paper, gate by gate, in the paper's order and notation.
 * It shares no code with the CUDA path (paper_2606_18981_b200/csrc) and may be
 * imported / linked / executed only by tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs.  It is never tuned.
 *
 * Parity status: every function below is pinned by tests/test_oracle_*.py
 * (naive DFT vs the library FFT; gates vs Kronecker-product matrices built from
 * PAPER.md:96; gate list vs PAPER.md Table 2 and the Fig. 1 worked circuit;
 * exact QFT vs the O(N^2) DFT; delta / tone / Parseval / linearity / k>=n-1 /
 * monotone AQFT error / k=0 Walsh-Hadamard).  No function is "parity unpinned".
 *
 * Conventions (readings c3, c4, c6 of SURVEY.md section 8(c), listed in DESIGN.md):
 *   - array index j = sum_q b_q 2^q, qubit q_0 is the least-significant bit
 *     (Fig. 1 caption, PAPER.md:96 operator formula);
 *   - forward sign is MINUS: omega_N = exp(-2 pi i / N),
 *     R_m = diag(1, exp(-2 pi i / 2^m)); sign=+1 conjugates;
 *   - H is Eq. 1 times 1/sqrt(2), so that the whole circuit is
 *     the unitary U = DFT_N / sqrt(N).
 *
 * State layout: interleaved (re, im) doubles, 2^n amplitudes.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_GATE_H 0
#define ORC_GATE_CR 1
#define ORC_GATE_SWAP 2

static const double ORC_TWO_PI = 6.283185307179586476925286766559;

int orc_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Hadamard on qubit t.  PAPER.md:37 (Eq. 1) scaled by 1/sqrt(2);
 * a 1-wire gate on q_t is I (x) U (x) I_{2^t} and updates the
 * 2^{n-1} pairs (j, j | 2^t) with the same 2x2 matvec. */
void orc_apply_h(double* s, int n, int t) {
    const int64_t N = (int64_t)1 << n;
    const int64_t bit = (int64_t)1 << t;
    const double r = 1.0 / sqrt(2.0);
    int64_t j;
#pragma omp parallel for schedule(static)
    for (j = 0; j < N; ++j) {
        if (j & bit) continue;
        const int64_t j1 = j | bit;
        const double ar = s[2 * j], ai = s[2 * j + 1];
        const double br = s[2 * j1], bi = s[2 * j1 + 1];
        s[2 * j] = (ar + br) * r;
        s[2 * j + 1] = (ai + bi) * r;
        s[2 * j1] = (ar - br) * r;
        s[2 * j1 + 1] = (ai - bi) * r;
    }
}

/* Controlled-R_m between qubits `control` and `target`:
 * R_m = diag(1, exp(sign * 2 pi i / 2^m)), sign=-1 is the paper's;
 * controlled-R_m = E1 (x) I + E2 (x) R_m: an elementwise phase on
 * the amplitudes whose control and target bits are both 1. */
void orc_apply_cr(double* s, int n, int control, int target, int m, int sign) {
    const int64_t N = (int64_t)1 << n;
    const int64_t both = ((int64_t)1 << control) | ((int64_t)1 << target);
    const double ang = (double)sign * ORC_TWO_PI / ldexp(1.0, m);
    const double c = cos(ang), d = sin(ang);
    int64_t j;
#pragma omp parallel for schedule(static)
    for (j = 0; j < N; ++j) {
        if ((j & both) != both) continue;
        const double ar = s[2 * j], ai = s[2 * j + 1];
        s[2 * j] = ar * c - ai * d;
        s[2 * j + 1] = ar * d + ai * c;
    }
}

/* SWAP of qubits a and b: "the final SWAPs are just index swaps". */
void orc_apply_swap(double* s, int n, int a, int b) {
    const int64_t N = (int64_t)1 << n;
    const int64_t ba = (int64_t)1 << a, bb = (int64_t)1 << b;
    int64_t j;
    if (a == b) return;
#pragma omp parallel for schedule(static)
    for (j = 0; j < N; ++j) {
        /* visit each exchanged pair once: bit a = 1, bit b = 0 */
        if ((j & ba) && !(j & bb)) {
            const int64_t j1 = (j & ~ba) | bb;
            const double tr = s[2 * j], ti = s[2 * j + 1];
            s[2 * j] = s[2 * j1];
            s[2 * j + 1] = s[2 * j1 + 1];
            s[2 * j1] = tr;
            s[2 * j1 + 1] = ti;
        }
    }
}

/* Number of gates of the n-qubit range-k (A)QFT circuit, swaps included. */
int64_t orc_gate_count(int n, int k) {
    int64_t c = 0;
    int t, d;
    for (t = n - 1; t >= 0; --t) {
        c += 1;
        for (d = 1; d <= t && d <= k; ++d) c += 1;
    }
    return c + n / 2;
}

/* The circuit, as a time-ordered gate list (PAPER.md:82 Fig. 1, :116, :137).
 *   for t = n-1 .. 0:  H(q_t);  for d = 1 .. min(k, t): CR_{d+1}(q_{t-d} -> q_t)
 *   then SWAP(q_i, q_{n-1-i}) for i < floor(n/2)   (output bit reversal P).
 * Range-k AQFT keeps only controlled rotations with control-target distance
 * d <= k, i.e. R_m with m <= k+1 (reading c1).
 * Each gate is 4 ints: {type, q0, q1, m}; H: q0 = wire; CR: q0 = control,
 * q1 = target, m = order; SWAP: q0, q1.  Returns the gate count (the list is
 * filled only while it fits in `cap` gates). */
int64_t orc_gate_list(int n, int k, int32_t* out, int64_t cap) {
    int64_t g = 0;
    int t, d, i;
    for (t = n - 1; t >= 0; --t) {
        if (g < cap) { out[4 * g] = ORC_GATE_H; out[4 * g + 1] = t; out[4 * g + 2] = -1; out[4 * g + 3] = 0; }
        ++g;
        for (d = 1; d <= t && d <= k; ++d) {
            if (g < cap) { out[4 * g] = ORC_GATE_CR; out[4 * g + 1] = t - d; out[4 * g + 2] = t; out[4 * g + 3] = d + 1; }
            ++g;
        }
    }
    for (i = 0; i < n / 2; ++i) {
        if (g < cap) { out[4 * g] = ORC_GATE_SWAP; out[4 * g + 1] = i; out[4 * g + 2] = n - 1 - i; out[4 * g + 3] = 0; }
        ++g;
    }
    return g;
}

/* State evolution: "the simulator applies the circuit gates in sequence"
 * (PAPER.md:138), one full sweep per gate. */
void orc_run_gates(double* s, int n, const int32_t* gates, int64_t ngates, int sign) {
    int64_t g;
    for (g = 0; g < ngates; ++g) {
        const int32_t* q = gates + 4 * g;
        if (q[0] == ORC_GATE_H) orc_apply_h(s, n, q[1]);
        else if (q[0] == ORC_GATE_CR) orc_apply_cr(s, n, q[1], q[2], q[3], sign);
        else orc_apply_swap(s, n, q[1], q[2]);
    }
}

void orc_scale(double* s, int n, double f) {
    const int64_t N2 = (int64_t)2 << n;
    int64_t j;
#pragma omp parallel for schedule(static)
    for (j = 0; j < N2; ++j) s[j] *= f;
}

/* Whole path, in place: circuit + swaps + normalisation.
 * norm: 0 unitary 1/sqrt(N) -> nothing more;
 *       1 none (plain DFT_N)  -> multiply by sqrt(N);
 *       2 1/N                 -> multiply by 1/sqrt(N) ("other conventions").
 * Returns 0, or -1 on allocation failure / bad arguments. */
int orc_qft(double* s, int n, int k, int sign, int norm) {
    int64_t ng;
    int32_t* gates;
    if (n < 1 || n > 34 || k < 0 || (sign != 1 && sign != -1) || norm < 0 || norm > 2) return -1;
    ng = orc_gate_count(n, k);
    gates = (int32_t*)malloc((size_t)ng * 4 * sizeof(int32_t));
    if (!gates) return -1;
    orc_gate_list(n, k, gates, ng);
    orc_run_gates(s, n, gates, ng, sign);
    free(gates);
    if (norm == 1) orc_scale(s, n, sqrt(ldexp(1.0, n)));
    else if (norm == 2) orc_scale(s, n, 1.0 / sqrt(ldexp(1.0, n)));
    return 0;
}

/* Naive O(N^2) DFT, the definition: y[K] = c * sum_j x[j] w^{jK},
 * w = exp(sign 2 pi i / N); c = 1/sqrt(N), 1, 1/N for norm 0, 1, 2.  The phase
 * index (j*K mod N) is reduced in integers so the angle is exact to rounding. */
int orc_naive_dft(const double* x, double* y, int n, int sign, int norm) {
    const int64_t N = (int64_t)1 << n;
    double c;
    int64_t K;
    if (n < 0 || n > 16) return -1;
    c = norm == 0 ? 1.0 / sqrt((double)N) : (norm == 1 ? 1.0 : 1.0 / (double)N);
#pragma omp parallel for schedule(static)
    for (K = 0; K < N; ++K) {
        long double ar = 0.0L, ai = 0.0L;
        int64_t j;
        for (j = 0; j < N; ++j) {
            const int64_t p = (j * K) & (N - 1);
            const double ang = (double)sign * ORC_TWO_PI * (double)p / (double)N;
            const double cr = cos(ang), ci = sin(ang);
            ar += (long double)(x[2 * j] * cr - x[2 * j + 1] * ci);
            ai += (long double)(x[2 * j] * ci + x[2 * j + 1] * cr);
        }
        y[2 * K] = (double)ar * c;
        y[2 * K + 1] = (double)ai * c;
    }
    return 0;
}

/* One matrix element <K| circuit |j> of the range-k circuit (unitary scaling),
 * obtained by following the single computational-basis input |j> through the
 * gates symbolically: H(q_t) turns bit t of the index into the output bit
 * y_t (amplitude 2^{-1/2} (-1)^{y_t b_t}), every kept CR_{d+1}(q_{t-d} -> q_t)
 * multiplies by exp(sign 2 pi i y_t b_{t-d} / 2^{d+1}) (b_{t-d} is still the
 * input bit because H(q_{t-d}) comes later), and the swaps put y_t at bit
 * n-1-t of K.  Used to evaluate single outputs as sum_j x[j] <K|.|j> where the
 * full state does not fit the oracle; pinned against orc_qft in the tests.
 * Returns the phase in turns (the element is 2^{-n/2} exp(2 pi i * turns)). */
double orc_element_turns(int n, int k, int sign, int64_t K, int64_t j) {
    double turns = 0.0;
    int t, d;
    for (t = n - 1; t >= 0; --t) {
        const int yt = (int)((K >> (n - 1 - t)) & 1);
        const int bt = (int)((j >> t) & 1);
        if (!yt) continue;
        if (bt) turns += 0.5; /* (-1)^{y_t b_t}: half a turn, either sign */
        for (d = 1; d <= t && d <= k; ++d)
            if ((j >> (t - d)) & 1) turns += (double)sign * ldexp(1.0, -(d + 1));
    }
    return turns - floor(turns);
}

/* out[K] = norm_factor * 2^{-n/2} * sum_j x[j] exp(2 pi i turns(K, j)) for the
 * sampled output indices Ks[0..ns).  x is interleaved complex64 or complex128
 * (is_f32 selects) of length 2^n.  O(ns * 2^n * n). */
int orc_outputs_at(const void* x, int is_f32, int n, int k, int sign, int norm,
                   const int64_t* Ks, int ns, double* out) {
    const int64_t N = (int64_t)1 << n;
    const float* xf = (const float*)x;
    const double* xd = (const double*)x;
    const double c0 = 1.0 / sqrt(ldexp(1.0, n));
    const double c = norm == 0 ? c0 : (norm == 1 ? 1.0 : c0 * c0);
    int s;
    for (s = 0; s < ns; ++s) {
        const int64_t K = Ks[s];
        double ar = 0.0, ai = 0.0;
        int64_t j;
#pragma omp parallel for schedule(static) reduction(+ : ar, ai)
        for (j = 0; j < N; ++j) {
            const double xr = is_f32 ? (double)xf[2 * j] : xd[2 * j];
            const double xi = is_f32 ? (double)xf[2 * j + 1] : xd[2 * j + 1];
            const double ang = ORC_TWO_PI * orc_element_turns(n, k, sign, K, j);
            const double cr = cos(ang), ci = sin(ang);
            ar += xr * cr - xi * ci;
            ai += xr * ci + xi * cr;
        }
        out[2 * s] = ar * c;
        out[2 * s + 1] = ai * c;
    }
    return 0;
}
