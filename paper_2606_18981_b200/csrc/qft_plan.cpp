// qft_plan.cpp -- host planner: gate list -> fused passes + layout adapters.
//
// The circuit (PAPER.md:82 Fig. 1, :116, :137) is
//     for t = n-1 .. 0:  H(q_t);  CR_{d+1}(q_{t-d} -> q_t), d = 1 .. min(k, t);   then bit reversal.
// Every CR that targets q_t is diagonal and commutes with the others, sits after
// H(q_t) and before H of its control, so their product is one phase per amplitude computed from index
// bits: after H(q_t), amp[j] *= exp(sign 2 pi i b_t(j) m_t(j) / 2^{t+1}) with
// m_t(j) = (j mod 2^t) with the bits below t-k cleared.  A pass that holds q_t inside its tile can
// therefore apply H(q_t) and ALL rotations onto q_t whatever their control, because the control bits
// are known from the address.  The planner's job is the data movement: which address bits form the
// tile of each pass, which qubits each pass processes, and how the store permutes address bits so that
// the final layout is the bit reversal, in place.
#include "qft_plan.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <set>
#include <sstream>

namespace {

struct PassSpec {
    std::vector<int> window;                 // logical qubits, descending; empty = permutation only
    std::vector<int> F;                      // tile address bits
    std::vector<int> Fbase;                  // F before the passive extras were added
    int extras_above = -1;                   // >= 0: take passive extras from address bits above this one first
    std::vector<std::pair<int, int>> moves;  // in-tile: data on address first goes to address second
    std::vector<std::pair<int, int>> swaps;  // non-tile address pairs (lo, hi) that trade places
};

int ilog2_ceil_div(int a, int b) { return (a + b - 1) / b; }

void add_extras(PassSpec& ps, int n, int ftarget) {
    if (ps.Fbase.empty()) ps.Fbase = ps.F;
    else ps.F = ps.Fbase;
    std::set<int> used(ps.F.begin(), ps.F.end());
    std::set<int> sw;
    for (auto& s : ps.swaps) { sw.insert(s.first); sw.insert(s.second); }
    // natural-order passes: the bits right above the window hold qubits that are already processed, which
    // contribute no phases (fewer table rows) and extend the window's run (fewer tensor-map dims)
    if (ps.extras_above >= 0)
        for (int a = ps.extras_above + 1; a < n && (int)ps.F.size() < ftarget; ++a) {
            if (used.count(a) || sw.count(a)) continue;
            ps.F.push_back(a);
            used.insert(a);
        }
    for (int a = 0; a < n && (int)ps.F.size() < ftarget; ++a) {
        if (used.count(a) || sw.count(a)) continue;
        ps.F.push_back(a);
        used.insert(a);
    }
    std::sort(ps.F.begin(), ps.F.end());
}

std::vector<int> split_balanced(int total, int parts) {
    std::vector<int> v(parts, total / parts);
    for (int i = 0; i < total % parts; ++i) v[i] += 1;
    return v;
}

// Natural-order compute passes, then one stand-alone tiled bit-reversal pass ("unfolded").
void build_unfolded(int n, int wcap, int fmax, int l, std::vector<PassSpec>* out) {
    const int f = std::min(fmax, n);
    const int wmax = (n <= fmax) ? std::min(wcap, n) : std::min(wcap, fmax - l);
    const int npass = ilog2_ceil_div(n, wmax);
    std::vector<int> sizes = split_balanced(n, npass);
    int t = n - 1;
    for (int p = 0; p < npass; ++p) {
        PassSpec ps;
        for (int i = 0; i < sizes[p]; ++i) ps.window.push_back(t - i);
        std::set<int> F;
        for (int a = 0; a < std::min(l, n); ++a) F.insert(a);
        for (int q : ps.window) F.insert(q);
        ps.F.assign(F.begin(), F.end());
        if (n > fmax) ps.extras_above = t;
        add_extras(ps, n, f);
        t -= sizes[p];
        out->push_back(ps);
    }
    if (n <= fmax) {
        // whole state in one tile: fold the reversal into the last pass's store
        PassSpec& last = out->back();
        for (int a = 0; a < n; ++a) last.moves.push_back({a, n - 1 - a});
        return;
    }
    PassSpec rv;
    const int h = std::min(fmax / 2, n / 2);
    for (int a = 0; a < h; ++a) { rv.F.push_back(a); rv.F.push_back(n - 1 - a); }
    std::sort(rv.F.begin(), rv.F.end());
    for (int a = 0; a < h; ++a) { rv.moves.push_back({a, n - 1 - a}); rv.moves.push_back({n - 1 - a, a}); }
    for (int a = h; a < n - 1 - a; ++a) rv.swaps.push_back({a, n - 1 - a});
    add_extras(rv, n, f);  // only the centre bit of an odd n is eligible
    out->push_back(rv);
}

// Folded schedule: K = 2 + #mid passes, no stand-alone reversal.
//   regions: H=[0,l)  A=[l,we)  Mid=[we,n-we)  B=[n-we,n-l)  T=[n-l,n)
//   we_force > 0: that width for the first and the last window instead of the balanced one.
bool build_folded(int n, int wcap, int fmax, int l, std::vector<PassSpec>* out, int we_force = 0) {
    if (n <= fmax) return false;
    int w = std::min(wcap, fmax - l);
    if (n <= 2 * w) w = (n - 1) / 2;
    if (w < l || w < 1) return false;
    int nmid_passes, we;
    if (we_force > 0) {
        we = we_force;
        if (we > w || n - 2 * we < 1) return false;
        nmid_passes = ilog2_ceil_div(n - 2 * we, w);
    } else {
        nmid_passes = ilog2_ceil_div(n - 2 * w, w);
        const int K = 2 + nmid_passes;
        we = std::min(w, ilog2_ceil_div(n, K));
        while (n - 2 * we > nmid_passes * w) ++we;
    }
    if (we < l || n - 2 * we < 1) return false;
    const int nmid = n - 2 * we;
    std::vector<int> chunks = split_balanced(nmid, nmid_passes);
    const int f = fmax;

    // first pass: top we qubits
    {
        PassSpec ps;
        for (int i = 0; i < we; ++i) ps.window.push_back(n - 1 - i);
        for (int a = 0; a < l; ++a) ps.F.push_back(a);
        for (int a = n - we; a < n; ++a) ps.F.push_back(a);
        for (int a = 0; a < l; ++a) { ps.moves.push_back({a, n - 1 - a}); ps.moves.push_back({n - 1 - a, a}); }
        if (nmid_passes > 1)
            for (int a = we; a < n - 1 - a; ++a) ps.swaps.push_back({a, n - 1 - a});
        add_extras(ps, n, f);
        out->push_back(ps);
    }
    // mid passes
    int t = n - we - 1;
    for (int c = 0; c < nmid_passes; ++c) {
        PassSpec ps;
        for (int i = 0; i < chunks[c]; ++i) ps.window.push_back(t - i);
        for (int a = 0; a < l; ++a) ps.F.push_back(a);
        if (nmid_passes == 1) {
            for (int a = we; a < n - we; ++a) { ps.F.push_back(a); ps.moves.push_back({a, n - 1 - a}); }
        } else {
            for (int q : ps.window) ps.F.push_back(n - 1 - q);  // Mid was reversed by the first pass
        }
        if (c == 0)
            for (int a = l; a < we; ++a) ps.swaps.push_back({a, n - 1 - a});
        std::sort(ps.F.begin(), ps.F.end());
        add_extras(ps, n, f);
        t -= chunks[c];
        out->push_back(ps);
    }
    // last pass: qubits we-1 .. 0, already on their final addresses inside Top
    {
        PassSpec ps;
        for (int i = 0; i < we; ++i) ps.window.push_back(we - 1 - i);
        for (int a = 0; a < l; ++a) ps.F.push_back(a);
        for (int a = n - we; a < n; ++a) ps.F.push_back(a);
        add_extras(ps, n, f);
        out->push_back(ps);
    }
    return true;
}

// max_fused_qubits smaller than the hub (PAPER.md:145's cap on the fused size; BASELINE config 3 sweeps it down to 2):
// no window can hold the hub's partner bits, so the folded schedule is laid out for the widest window the tile allows
// and every one of its windows is cut into sub-passes of <= wcap qubits.  Only the last sub-pass of a window carries
// the window's layout adapter (in-tile moves, pair involution); the others run in place on a tile of their own:
// hub + sub-window + the lowest free address bits, i.e. long contiguous rows.
bool build_folded_split(int n, int wcap, int fmax, int l, int we, std::vector<PassSpec>* out) {
    std::vector<PassSpec> sup;
    if (!build_folded(n, fmax - l, fmax, l, &sup, we)) return false;
    std::vector<int> qubit_at(n);
    for (int a = 0; a < n; ++a) qubit_at[a] = a;
    for (const PassSpec& sp : sup) {
        const int W = (int)sp.window.size();
        // smaller sub-windows first: a one-qubit window (only the generic kernel takes it) then runs in place on a small tile
        std::vector<int> sizes = split_balanced(W, ilog2_ceil_div(W, wcap));
        std::reverse(sizes.begin(), sizes.end());
        int off = 0;
        for (size_t c = 0; c < sizes.size(); ++c) {
            std::vector<int> win(sp.window.begin() + off, sp.window.begin() + off + sizes[c]);
            off += sizes[c];
            PassSpec s;
            if (c + 1 == sizes.size()) {
                s = sp;
            } else {
                std::set<int> F;
                for (int a = 0; a < l; ++a) F.insert(a);
                for (int q : win) {
                    int at = -1;
                    for (int a = 0; a < n; ++a)
                        if (qubit_at[a] == q) at = a;
                    if (at < l) return false;  // a window qubit never sits on a hub bit when its turn comes
                    F.insert(at);
                }
                s.F.assign(F.begin(), F.end());
                add_extras(s, n, fmax);
            }
            s.window = win;
            out->push_back(s);
        }
        std::vector<int> nq(qubit_at);
        for (auto& m : sp.moves) nq[m.second] = qubit_at[m.first];
        for (auto& sw : sp.swaps) { nq[sw.first] = qubit_at[sw.second]; nq[sw.second] = qubit_at[sw.first]; }
        qubit_at.swap(nq);
    }
    return true;
}

// Deferred swaps (QFT_FLAG_DEFER_SWAPS; "SWAP can be deferred to I/O or absorbed into layout",
// :137 "the final swaps are not implemented as gates but accounted for in the caller as an output index
// permutation"): the planner no longer steers towards the bit-reversed layout, it takes the cheapest one and the
// plan reports where every qubit ended (QftHostPlan::out_qubit_at).  K = ceil(n / w) passes, no pair passes at
// all: the hub's qubits trade places with the top l qubits in the first pass (a qubit cannot be processed while
// it sits on a hub bit) and are processed up there by the last pass; every other window is processed where it
// sits.  Final layout: the circuit's own (qubit q on bit q) except that bits a and n-1-a are exchanged for a < l.
bool build_deferred(int n, int wcap, int fmax, int l, std::vector<PassSpec>* out) {
    if (n <= fmax) return false;
    const int w = std::min(wcap, fmax - l);
    if (w < 1 || n < 2 * l) return false;
    const int f = fmax;
    // address of qubit q once the hub has traded places with the top l bits
    auto addr_after = [&](int q) { return (q < l || q >= n - l) ? n - 1 - q : q; };
    auto window_pass = [&](int t, int size, bool swapped, bool natural_run) {
        PassSpec ps;
        std::set<int> F;
        for (int a = 0; a < l; ++a) F.insert(a);
        for (int i = 0; i < size; ++i) {
            ps.window.push_back(t - i);
            F.insert(swapped ? addr_after(t - i) : t - i);
        }
        ps.F.assign(F.begin(), F.end());
        if (natural_run) ps.extras_above = t;
        return ps;
    };
    std::vector<int> sizes = split_balanced(n, ilog2_ceil_div(n, w));
    if (sizes.size() >= 2 && sizes.front() >= l && sizes.back() >= l) {
        // the first pass holds the top l qubits next to the hub: it trades them
        int t = n - 1;
        for (size_t p = 0; p < sizes.size(); ++p) {
            PassSpec ps = window_pass(t, sizes[p], p > 0, p > 0 && p + 1 < sizes.size());
            if (p == 0)
                for (int a = 0; a < l; ++a) { ps.moves.push_back({a, n - 1 - a}); ps.moves.push_back({n - 1 - a, a}); }
            add_extras(ps, n, f);
            t -= sizes[p];
            out->push_back(ps);
        }
        return true;
    }
    // windows smaller than the hub: process the top l qubits where they sit, trade hub and top in a pass of its own
    // (permutation only), then process the rest
    int t = n - 1;
    for (int sz : split_balanced(l, ilog2_ceil_div(l, w))) {
        PassSpec ps = window_pass(t, sz, false, false);
        add_extras(ps, n, f);
        t -= sz;
        out->push_back(ps);
    }
    {
        PassSpec ps;
        for (int a = 0; a < l; ++a) { ps.F.push_back(a); ps.moves.push_back({a, n - 1 - a}); ps.moves.push_back({n - 1 - a, a}); }
        for (int a = n - l; a < n; ++a) ps.F.push_back(a);
        add_extras(ps, n, f);
        out->push_back(ps);
    }
    for (int sz : split_balanced(n - l, ilog2_ceil_div(n - l, w))) {
        PassSpec ps = window_pass(t, sz, true, false);
        add_extras(ps, n, f);
        t -= sz;
        out->push_back(ps);
    }
    return true;
}

std::vector<int> step_sizes(int w, bool force2 = false) {
    if (w <= 0) return {};
    if (force2 && w >= 2 && w <= 5) return split_balanced(w, 2);  // two register groups for the TMA kernel
    const int g = ilog2_ceil_div(w, QFT_MAX_RADIX_BITS);
    return split_balanced(w, g);  // larger groups first
}


// ---- QFT_KERNEL_TMA2 lowering -----------------------------------------------------------------
// Choose 4-bit XOR masks for the canonical bits >= 4 such that the four lowest lane bits of step 1's
// writers and of step 2's readers each map to linearly independent bank masks (8-byte accesses are
// served per half-warp: 16 lanes x 8 B = the 32 banks).  Canonical bits < 4 keep their own bank bit.
// Backtracking over the (at most eight) bits involved.
bool independent4(const int (&m)[4]) {
    // Gaussian elimination over GF(2) on four 4-bit vectors
    int v[4] = {m[0], m[1], m[2], m[3]};
    int rank = 0;
    for (int bit = 0; bit < 4; ++bit) {
        int piv = -1;
        for (int i = rank; i < 4; ++i)
            if ((v[i] >> bit) & 1) { piv = i; break; }
        if (piv < 0) continue;
        std::swap(v[rank], v[piv]);
        for (int i = 0; i < 4; ++i)
            if (i != rank && ((v[i] >> bit) & 1)) v[i] ^= v[rank];
        ++rank;
    }
    return rank == 4;
}

bool solve_swizzle(const int (&L1)[4], const int (&L2)[4], int f, uint8_t (&lowmask)[16]) {
    // lowmask[c] = the low-4-bit mask canonical bit c contributes (for c < 4: 1 << c, fixed)
    for (int c = 0; c < 16; ++c) lowmask[c] = (c < 4) ? (uint8_t)(1u << c) : 0;
    std::vector<int> freebits;
    for (int i = 0; i < 4; ++i) {
        for (int c : {L1[i], L2[i]})
            if (c >= 4 && std::find(freebits.begin(), freebits.end(), c) == freebits.end()) freebits.push_back(c);
    }
    (void)f;
    auto ok = [&]() {
        int a[4], b[4];
        for (int i = 0; i < 4; ++i) { a[i] = lowmask[L1[i]]; b[i] = lowmask[L2[i]]; }
        return independent4(a) && independent4(b);
    };
    // depth-first over assignments (16 choices per free bit, <= 8 bits, pruned only at the leaves: the
    // search space is at most 16^8 but a solution is found within the first few thousand leaves)
    std::vector<int> choice(freebits.size(), 0);
    size_t nfree = freebits.size();
    if (nfree == 0) return ok();
    long long budget = 20000000;
    std::vector<int> idx(nfree, 1);
    while (budget-- > 0) {
        for (size_t i = 0; i < nfree; ++i) lowmask[freebits[i]] = (uint8_t)idx[i];
        if (ok()) return true;
        size_t i = 0;
        while (i < nfree) {
            if (++idx[i] < 16) break;
            idx[i] = 1;
            ++i;
        }
        if (i == nfree) break;
    }
    return false;
}

// Fills d->tma and sets d->kernel = QFT_KERNEL_TMA2 when the pass fits the kernel's shape.
// Compile with -DQFT_PLAN_DEBUG to print why a pass was not given to the TMA kernel.
#ifdef QFT_PLAN_DEBUG
#define QFT_REJECT(code)                                                                                              \
    do {                                                                                                              \
        fprintf(stderr, "lower_tma2: reject at #%d (f=%d r=%d+%d)\n", code, d->f, d->steps[0].r, d->steps[1].r);      \
        return;                                                                                                       \
    } while (0)
#else
#define QFT_REJECT(code) return
#endif
void lower_tma2(QftPassDesc* d, int n) {
    const int f = d->f;
    const QftStep s1 = d->steps[0], s2 = d->steps[1];
    const int r1 = s1.r, r2 = s2.r;
    if (f < 12 || f > 14) QFT_REJECT(2);
    if (!((r1 == 5 && r2 == 5) || (r1 == 5 && r2 == 4) || (r1 == 4 && r2 == 4) || (r1 == 4 && r2 == 3) ||
          (r1 == 3 && r2 == 3) || (r1 == 3 && r2 == 2) || (r1 == 2 && r2 == 2) || (r1 == 2 && r2 == 1) ||
          (r1 == 1 && r2 == 1)))
        QFT_REJECT(3);
    if (d->xt && (f != 14 || r1 + r2 < 8)) QFT_REJECT(4);  // the extended tile is built for 2^14 halves only
    if (s1.a != s2.a + r2) QFT_REJECT(5);  // the window is one run of canonical bits
    const int eb = s2.a;            // canonical bits below the window
    // more than QFT_TMA2_EB_DIRECT: the split end table, instantiated for windows of <= 6 qubits (qft_tma_es*.cu)
    if (eb > QFT_TMA2_EB_MAX || (eb > QFT_TMA2_EB_DIRECT && (r1 + r2 > 6 || d->xt))) QFT_REJECT(6);
    if (n - f < 1) QFT_REJECT(7);
    QftTma2Desc t;
    std::memset(&t, 0, sizeof t);
    const int lt = f - 5;
    auto in1 = [&](int c) { return c >= s1.a && c < s1.a + r1; };
    auto in2 = [&](int c) { return c >= s2.a && c < s2.a + r2; };
    std::vector<int> inF(n, 0), canon_at_load(n, -1), st_idx_of_canon(f);
    for (int j = 0; j < f; ++j) {
        inF[d->F[j]] = 1;
        canon_at_load[d->F[j]] = d->ld_canon[j];
        st_idx_of_canon[d->st_canon[j]] = j;
    }
    if (!inF[0] || !inF[1]) QFT_REJECT(8);  // the innermost box dimension must span >= 16 bytes
    // ---- tensor-map dims: runs of address bits inside / outside F.  In-tile runs are cut where the
    // group membership changes and to <= 8 bits (box <= 256); the run that starts at address bit 0 is
    // dimension 0 (TMA's contiguous one).  The box lands in shared memory dimension by dimension, so
    // the order of the other in-tile dims is free: group 1's go last, which keeps its qubits out of
    // the four lowest landing-index bits (conflict-free reads by lanes that run along the low bits).
    struct Dim { int lo, len, box, cls; };
    std::vector<Dim> dims;
    // the four lowest landing-index bits must not hold group-1 qubits; if the address-ascending order
    // would put one there, runs are cut where group-1 membership changes and group 1's dims go last
    bool need_reorder = false;
    for (int j = 0; j < std::min(4, f); ++j)
        if (in1(d->ld_canon[j])) need_reorder = true;
    auto cls_of = [&](int a) { const int c = canon_at_load[a]; return (need_reorder && in1(c)) ? 2 : 0; };
    // box dims: the runs of tile bits.  All tile-INDEX bits share ONE dimension of box 1 that spans from
    // the lowest to the highest of them with the stride of the lowest: its coordinate is the tile's base
    // address shifted down, and since a base address has zeros on every tile bit the sum
    // coordinate x stride still lands on the right element (TMA checks bounds per dimension only).
    int a = 0;
    while (a < n) {
        int b = a + 1;
        if (inF[a]) {
            // dimension 0 may mix classes (it is the hub); the others may not
            while (b < n && inF[b] && b - a < 8 && (cls_of(b) == cls_of(a))) ++b;
            dims.push_back({a, b - a, b - a, cls_of(a)});
        }
        a = b;
    }
    {
        int tlo = -1, thi = -1;
        for (int b = 0; b < n; ++b)
            if (!inF[b]) { if (tlo < 0) tlo = b; thi = b; }
        if (tlo < 0 || thi - tlo + 1 > 31) QFT_REJECT(22);
        dims.push_back({tlo, thi - tlo + 1, 0, -1});
    }
    if (dims.size() > 5 || dims[0].box < 1 || dims[0].cls == 2) QFT_REJECT(9);
    // (only needed when the hub alone does not fill the four lowest landing bits; otherwise keep the
    // natural, address-ascending order)
    if (need_reorder)
        std::stable_sort(dims.begin() + 1, dims.end(), [](const Dim& x, const Dim& y) {
            const int kx = x.cls == 2 ? 1 : 0, ky = y.cls == 2 ? 1 : 0;
            return kx < ky;
        });
    while (dims.size() < 5) dims.push_back({n, 0, 0, -1});  // size-1 padding dims
    int nland = 0;
    std::vector<int> land_idx_of_canon(f, -1);
    for (int i = 0; i < 5; ++i) {
        t.tma_lo[i] = (int8_t)dims[i].lo;
        t.tma_len[i] = (int8_t)dims[i].len;
        t.tma_box[i] = (int8_t)dims[i].box;
        for (int b = 0; b < dims[i].box; ++b) {
            t.land_addr[nland] = (int8_t)(dims[i].lo + b);
            land_idx_of_canon[canon_at_load[dims[i].lo + b]] = nland;
            ++nland;
        }
    }
    if (nland != f) QFT_REJECT(11);
    // ---- threads and registers of the two steps (canonical bits) ----
    // step 1: register bits = group 1 (+ batch bits: the highest landing bits outside the group);
    // thread bits = the remaining landing bits, ascending, so lanes read consecutive shared memory
    std::vector<int> reg1, thr1, reg2, thr2;
    for (int b = 0; b < r1; ++b) reg1.push_back(s1.a + b);
    {
        std::vector<int> rest;
        for (int j = 0; j < f; ++j) {
            const int c = canon_at_load[t.land_addr[j]];
            if (!in1(c)) rest.push_back(c);
        }
        while ((int)reg1.size() < 5) { reg1.push_back(rest.back()); rest.pop_back(); }
        thr1 = rest;
    }
    // step 2: register bits = group 2 (+ batch bits); thread bits = the remaining store-order bits,
    // ascending, so lanes run along the hub and every warp store covers whole granules
    for (int b = 0; b < r2; ++b) reg2.push_back(s2.a + b);
    {
        std::vector<int> rest;
        for (int j = 0; j < f; ++j)
            if (!in2(d->st_canon[j])) rest.push_back(d->st_canon[j]);
        while ((int)reg2.size() < 5) { reg2.push_back(rest.back()); rest.pop_back(); }
        thr2 = rest;
    }
    if ((int)thr1.size() != lt || (int)thr2.size() != lt) QFT_REJECT(15);
    for (int j = 0; j < 4; ++j)
        if (land_idx_of_canon[thr1[j]] != j) QFT_REJECT(19);
    // store lanes: at least the three lowest hub bits (64-byte segments); a fourth hub bit that
    // receives a group-2 qubit becomes a register bit (the two half lines leave the same warp a
    // few instructions apart and merge in L2)
    const int hubrun0 = dims[0].box;
    for (int j = 0; j < std::min(hubrun0, 3); ++j)
        if (st_idx_of_canon[thr2[j]] != j || d->Fst[j] != j) QFT_REJECT(20);
    // exchange layout: canonical index XOR-swizzled
    int L1[4], L2[4];
    for (int j = 0; j < 4; ++j) { L1[j] = thr1[j]; L2[j] = thr2[j]; }
    uint8_t lowmask[16];
    if (!solve_swizzle(L1, L2, f, lowmask)) QFT_REJECT(21);
    auto midcol = [&](int c) -> uint32_t {
        const uint32_t slot = (c < 4) ? (1u << c) : ((1u << c) ^ lowmask[c]);
        return slot << 3;
    };
    auto landcol = [&](int c) -> uint32_t { return 8u << land_idx_of_canon[c]; };
    auto key1 = [&](int c) -> uint32_t {
        if (in2(c)) return 1u << (c - s2.a);
        if (c < eb) return 1u << (8 + c);
        return 0;
    };
    auto key2 = [&](int c) -> uint32_t {
        if (in1(c)) return 1u << (c - s1.a);
        if (c < eb) return 1u << (8 + c);
        return 0;
    };
    for (int j = 0; j < lt; ++j) {
        t.s1_tid_ld[j] = landcol(thr1[j]);
        t.s1_tid_mid[j] = midcol(thr1[j]);
        t.s1_tid_key[j] = key1(thr1[j]);
        t.s2_tid_mid[j] = midcol(thr2[j]);
        t.s2_tid_key[j] = key2(thr2[j]);
        t.s2_tid_addr[j] = d->Fst[st_idx_of_canon[thr2[j]]];
    }
    for (int b = 0; b < 5; ++b) {
        t.s1_reg_ld[b] = landcol(reg1[b]);
        t.s1_reg_mid[b] = midcol(reg1[b]);
        t.s1_reg_key[b] = key1(reg1[b]);
        t.s2_reg_mid[b] = midcol(reg2[b]);
        t.s2_reg_key[b] = key2(reg2[b]);
        t.s2_reg_addr[b] = d->Fst[st_idx_of_canon[reg2[b]]];
    }
    t.eb = (int8_t)eb;
    for (int c = 0; c < eb; ++c) t.e_log[c] = d->log_canon[c];
    t.t1_lo = (int8_t)(s1.t_hi - r1 + 1);
    t.t2_lo = (int8_t)(s2.t_hi - r2 + 1);
    t.r1 = (int8_t)r1;
    t.r2 = (int8_t)r2;
    d->tma = t;
    d->kernel = QFT_KERNEL_TMA2;
    d->log2_threads = lt;
}

#undef QFT_REJECT
// Turn a PassSpec into the kernel descriptor given the current layout; updates qubit_at.
// xt: ps.F is the tile of a tensor-memory extended pass (qft_plan.h): the window's lowest qubit g is taken
// out of the register steps, its address bit becomes the half-tile index bit, and the descriptor describes
// one half; the pass must then lower to the TMA kernel (no other kernel knows about the extension).
bool lower_pass(const PassSpec& ps, int n, int k, int conj, int hub, bool allow_fused, bool allow_tma,
                std::vector<int>& qubit_at, QftPassDesc* d, std::string* err, bool force2 = false, bool xt = false) {
    std::memset(d, 0, sizeof(*d));
    std::vector<int> dest(n);
    for (int a = 0; a < n; ++a) dest[a] = a;
    std::vector<int> inFull(n, 0);
    for (int a : ps.F) inFull[a] = 1;
    for (auto& m : ps.moves) {
        if (!inFull[m.first] || !inFull[m.second]) { *err = "move leaves the tile"; return false; }
        dest[m.first] = m.second;
    }
    std::vector<int> src_of(n, -1);
    for (int a : ps.F) {
        if (src_of[dest[a]] != -1) { *err = "in-tile moves are not a permutation"; return false; }
        src_of[dest[a]] = a;
    }
    for (int a : ps.F)
        if (src_of[a] < 0) { *err = "in-tile moves are not a permutation"; return false; }
    // load-side and store-side tile bits
    std::vector<int> Fld(ps.F), Fst(ps.F);
    int g = -1, a_g = -1, b_g = -1;
    if (xt) {
        if (ps.window.size() < 3) { *err = "extended tile: window too small"; return false; }
        g = ps.window.back();
        for (int a : ps.F)
            if (qubit_at[a] == g) a_g = a;
        if (a_g < 0) { *err = "extended tile: qubit outside the tile"; return false; }
        b_g = dest[a_g];
        if (a_g < hub || b_g < hub) { *err = "extended tile: half-tile bit inside the hub"; return false; }
        Fld.erase(std::find(Fld.begin(), Fld.end(), a_g));
        Fst.erase(std::find(Fst.begin(), Fst.end(), b_g));
    }
    const int f = (int)Fld.size();
    if (f > QFT_MAX_TILE_BITS || n - f > QFT_MAX_TILEIDX_BITS) { *err = "tile too large"; return false; }
    d->n = n; d->f = f; d->ntile = n - f; d->k = k; d->conj = conj; d->scale = 1.0f; d->do_scale = 0;
    d->kernel = QFT_KERNEL_GENERIC;
    d->xt = xt ? 1 : 0;
    d->xt_q = (int8_t)g; d->xt_ld_addr = (int8_t)a_g; d->xt_st_addr = (int8_t)b_g;
    int lt = f - 2;
    if (lt < 5) lt = 5;
    if (lt > 8) lt = 8;
    d->log2_threads = lt;
    // canonical order: the half-tile's qubits ascending by logical id
    std::vector<int> qs;
    for (int a : Fld) qs.push_back(qubit_at[a]);
    std::sort(qs.begin(), qs.end());
    std::vector<int> canon_of_q(n, -1);
    for (int c = 0; c < f; ++c) { canon_of_q[qs[c]] = c; d->log_canon[c] = (int8_t)qs[c]; }
    for (int j = 0; j < f; ++j) {
        d->F[j] = (int8_t)Fld[j];
        d->Fst[j] = (int8_t)Fst[j];
        d->ld_canon[j] = (int8_t)canon_of_q[qubit_at[Fld[j]]];
        d->st_canon[j] = (int8_t)canon_of_q[qubit_at[src_of[Fst[j]]]];
    }
    // tile-index bits: swapped pairs first (lo side, then hi side), then the rest ascending, then the
    // half-tile bit of an extended pass
    const int p = (int)ps.swaps.size();
    d->npair = p;
    std::vector<int> taken(n, 0);
    for (int i = 0; i < p; ++i) {
        const int a = ps.swaps[i].first, b = ps.swaps[i].second;
        if (inFull[a] || inFull[b] || taken[a] || taken[b] || a == b) { *err = "bad swap"; return false; }
        taken[a] = taken[b] = 1;
        d->tile_addr[i] = (int8_t)a;
        d->tile_addr[p + i] = (int8_t)b;
    }
    int ti = 2 * p;
    for (int a = 0; a < n; ++a)
        if (!inFull[a] && !taken[a]) d->tile_addr[ti++] = (int8_t)a;
    if (xt) d->tile_addr[ti++] = (int8_t)a_g;
    if (ti != n - f) { *err = "tile index bits do not add up"; return false; }
    for (int i = 0; i < n - f; ++i) d->log_tile[i] = (int8_t)qubit_at[d->tile_addr[i]];
    // steps
    d->win_lo = -1;
    d->nsteps = 0;
    if (!ps.window.empty()) {
        const int wfull = (int)ps.window.size();
        for (int i = 0; i < wfull; ++i)
            if (ps.window[i] != ps.window[0] - i) { *err = "window not contiguous"; return false; }
        const int w = xt ? wfull - 1 : wfull;
        for (int i = 0; i < w; ++i)
            if (canon_of_q[ps.window[i]] < 0) { *err = "window qubit outside the tile"; return false; }
        d->win_lo = ps.window[w - 1];
        int t = ps.window[0];
        for (int r : step_sizes(w, force2)) {
            QftStep& st = d->steps[d->nsteps++];
            st.r = (int8_t)r;
            st.t_hi = (int8_t)t;
            st.a = (int8_t)canon_of_q[t - r + 1];
            if (canon_of_q[t] != st.a + r - 1) { *err = "window not contiguous in the tile"; return false; }
            t -= r;
        }
    }
    // fused two-step kernel: eligible when the hub's qubits are not in the register group of the
    // step that touches HBM (so that the lanes of a warp can walk whole granules)
    if (d->nsteps == 2 && allow_fused && !xt) {
        const QftStep s1 = d->steps[0], s2 = d->steps[1];
        auto in_group = [](const QftStep& s, int c) { return c >= s.a && c < s.a + s.r; };
        const int l = std::min(hub, f);
        bool ok = true;
        for (int j = 0; j < l; ++j) {
            if (in_group(s1, d->ld_canon[j])) ok = false;
            if (in_group(s2, d->st_canon[j])) ok = false;
        }
        if (f - std::max<int>(s1.r, s2.r) < 5) ok = false;  // at least one warp of butterflies
        if (ok) {
            d->kernel = QFT_KERNEL_FUSED2;
            int lt2 = f - std::max<int>(s1.r, s2.r);
            d->log2_threads = std::min(lt2, 8);
            std::vector<int> addr_of_canon_ld(f), addr_of_canon_st(f);
            for (int j = 0; j < f; ++j) {
                addr_of_canon_ld[d->ld_canon[j]] = d->F[j];
                addr_of_canon_st[d->st_canon[j]] = d->F[j];
            }
            int nt = 0;
            for (int j = 0; j < f; ++j)
                if (!in_group(s1, d->ld_canon[j])) { d->t1_addr[nt] = d->F[j]; d->t1_canon[nt] = d->ld_canon[j]; ++nt; }
            for (int b = 0; b < s1.r; ++b) d->r1_addr[b] = (int8_t)addr_of_canon_ld[s1.a + b];
            nt = 0;
            for (int j = 0; j < f; ++j)
                if (!in_group(s2, d->st_canon[j])) { d->t2_addr[nt] = d->F[j]; d->t2_canon[nt] = d->st_canon[j]; ++nt; }
            for (int b = 0; b < s2.r; ++b) d->r2_addr[b] = (int8_t)addr_of_canon_st[s2.a + b];
            // swizzle: canonical bits 0..3 keep their own bank bit; the four lowest lane bits of each
            // step (a half-warp = one 128-byte shared-memory wavefront of 8-byte accesses) must get
            // linearly independent masks
            for (int c = 0; c < 16; ++c) d->swz_col[c] = 0;
            for (int c = 0; c < std::min(4, f); ++c) d->swz_col[c] = (uint8_t)(1u << c);
            auto fix = [&](const int8_t* lane_canon, int nl) {
                // span of the masks already fixed among these lanes
                std::vector<int> vecs;
                for (int i = 0; i < nl; ++i)
                    if (d->swz_col[lane_canon[i]]) vecs.push_back(d->swz_col[lane_canon[i]]);
                auto span = [&](const std::vector<int>& vs) {
                    std::set<int> sp{0};
                    for (int v : vs) {
                        std::set<int> add;
                        for (int x : sp) add.insert(x ^ v);
                        sp.insert(add.begin(), add.end());
                    }
                    return sp;
                };
                for (int i = 0; i < nl; ++i) {
                    const int c = lane_canon[i];
                    if (d->swz_col[c]) continue;
                    std::set<int> sp = span(vecs);
                    for (int v = 1; v < 16; ++v)
                        if (!sp.count(v)) { d->swz_col[c] = (uint8_t)v; vecs.push_back(v); break; }
                }
            };
            fix(d->t1_canon, std::min(4, f - s1.r));
            fix(d->t2_canon, std::min(4, f - s2.r));
        }
    }
    if (d->nsteps == 2 && allow_tma) lower_tma2(d, n);
    if (xt && d->kernel != QFT_KERNEL_TMA2) { *err = "extended tile: pass does not fit the TMA kernel"; return false; }
    // apply the permutation to the tracking
    std::vector<int> nq(qubit_at);
    for (int a : ps.F) nq[dest[a]] = qubit_at[a];
    for (auto& s : ps.swaps) { nq[s.first] = qubit_at[s.second]; nq[s.second] = qubit_at[s.first]; }
    qubit_at.swap(nq);
    return true;
}

}  // namespace

// Lower every pass spec; false if a pass could not be lowered (err says which and why).
static bool lower_all(const QftPlanParams& prm, std::vector<PassSpec>& specs, int na, int k_eff, int l, int fsmem,
                      QftHostPlan* out, std::string* err) {
    std::vector<int> qubit_at(na);
    for (int a = 0; a < na; ++a) qubit_at[a] = a;
    const int conj = prm.sign == 1 ? 1 : 0;
    const bool allow_fused = !(prm.flags & 1u);
    const bool allow_tma = !(prm.flags & 5u);
    int wmaxseen = 0;
    for (auto& ps : specs) {
        QftPassDesc d;
        // the passive extra tile bits are optional: if the full tile does not fit the TMA kernel
        // (too many tensor-map dims, too many low in-tile qubits), try smaller tiles
        const bool want_tma = allow_tma && ps.window.size() >= 2;
        const int fbase = (int)(ps.Fbase.empty() ? ps.F.size() : ps.Fbase.size());
        bool done = false;
        if (want_tma && !ps.Fbase.empty() && fbase <= fsmem) {
            for (int ft = std::min((int)ps.F.size(), fsmem); ft >= 12 && ft >= fbase && !done; --ft) {
                PassSpec trial = ps;
                add_extras(trial, na, ft);
                if ((int)trial.F.size() != ft) continue;
                std::vector<int> qa = qubit_at;
                QftPassDesc dt;
                std::string e2;
                if (lower_pass(trial, na, k_eff, conj, l, allow_fused, true, qa, &dt, &e2, true) &&
                    dt.kernel == QFT_KERNEL_TMA2) {
                    d = dt;
                    qubit_at = qa;
                    done = true;
                }
            }
        }
        if (!done && fbase > fsmem) {
            // the window and the hub need one bit more than a shared-memory tile holds: tensor-memory extension
            PassSpec trial = ps;
            add_extras(trial, na, fsmem + 1);
            std::vector<int> qa = qubit_at;
            QftPassDesc dt;
            if ((int)trial.F.size() != fsmem + 1 || !want_tma ||
                !lower_pass(trial, na, k_eff, conj, l, false, true, qa, &dt, err, true, true))
                return false;
            d = dt;
            qubit_at = qa;
            done = true;
        }
        if (!done && (int)ps.F.size() > fsmem) add_extras(ps, na, fsmem);  // the other kernels: shared-memory tiles
        if (!done && allow_fused && (ps.window.size() == 4 || ps.window.size() == 5)) {
            // a 4- or 5-qubit window as two register groups, so that the fused kernel can take it
            std::vector<int> qa = qubit_at;
            QftPassDesc dt;
            std::string e2;
            if (lower_pass(ps, na, k_eff, conj, l, true, false, qa, &dt, &e2, true) && dt.kernel == QFT_KERNEL_FUSED2) {
                d = dt;
                qubit_at = qa;
                done = true;
            }
        }
        // a one-qubit window that only the generic kernel takes, in place: a small tile (many CTAs per SM) instead of
        // the plan's large one
        if (!done && ps.window.size() == 1 && ps.moves.empty() && ps.swaps.empty() && !ps.Fbase.empty() && na > fsmem) {
            const int ft = std::max(fbase, std::min((int)ps.F.size(), 11));
            if (ft < (int)ps.F.size()) add_extras(ps, na, ft);
        }
        if (!done && !lower_pass(ps, na, k_eff, conj, l, allow_fused, allow_tma, qubit_at, &d, err)) return false;
        wmaxseen = std::max(wmaxseen, (int)ps.window.size());
        out->passes.push_back(d);
    }
    out->window = wmaxseen;
    out->out_qubit_at = qubit_at;
    return true;
}

int qft_build_plan(const QftPlanParams& prm, QftHostPlan* out, std::string* err) {
    const int n = prm.n;                  // qubits of one transform
    const int na = prm.n + prm.batch_bits;  // address bits of the whole (batched) state
    if (prm.batch_bits < 0 || na > 34) {
        *err = "invalid argument";
        return 1;
    }
    if (n < 1 || n > 34 || prm.k < 0 || prm.max_fused < 1 || (prm.sign != 1 && prm.sign != -1) || prm.norm < 0 ||
        prm.norm > 2) {
        *err = "invalid argument";
        return 1;
    }
    if (prm.flags & ~(1u | 2u | 4u | 16u | 32u)) { *err = "unknown flag"; return 2; }
    if ((prm.flags & 32u) && (prm.flags & 2u)) { *err = "deferred swaps have no unfolded schedule"; return 2; }
    // defaults from the B200 sweeps (profiles/r01_tile_hub_sweep.md, profiles/r02_tile_hub_sweep.md): 128-byte
    // granules (hub 4) as soon as the state is large enough for a hub to exist, 2^14 tiles once three 10-qubit
    // windows pay off (n = 13: three multi-CTA passes on 2^12 tiles take 17 us, one 8192-amplitude CTA takes 30 us)
    // (n = 13 ... 23, state resident in L2: 2^12 tiles put twice as many CTAs in flight, 19 vs 21.5 us at n = 20, 37.8 vs
    // 42.4 us at n = 22; with 128-byte granules from n = 14 on the mid pass fits the TMA kernel too, 13.1 vs 18.5 us
    // at n = 15, 15.4 vs 20.8 us at n = 18: profiles/r02_small_n.md)
    int fmax = prm.tile_bits ? prm.tile_bits : (n >= 26 ? 14 : (prm.batch_bits == 0 && n >= 13 && n <= 23 ? 12 : 13));
    // 256-byte granules (hub 5) where a 10-qubit window still gives the minimum number of passes: with the
    // tensor-memory extension that is n = 26 ... 30 (3 passes) and n = 34 (4 passes); n = 31 ... 33 need 11-qubit
    // windows for 3 passes, i.e. 128-byte granules (profiles/r02_tile_hub_sweep.md)
    int l = prm.hub_bits ? prm.hub_bits : (na >= 20 || (prm.batch_bits == 0 && n >= 14) ? 4 : 3);
    if (!prm.hub_bits && prm.batch_bits == 0 && fmax == 14 && !(prm.flags & (1u | 2u | 4u | 16u)) && ((n >= 26 && n <= 30) || n == 34))
        l = n == 34 ? 6 : 5;  // n = 34 (four passes either way): 512-byte granules, 239 vs 264 ms
    if (fmax < 2 || fmax > QFT_MAX_TILE_BITS || l < 1 || l > 6 || l >= fmax) {
        *err = "unsupported tile_bits / hub_bits";
        return 2;
    }
    if (na - std::min(fmax, na) > 30) { *err = "tile_bits too small for this n"; return 2; }
    // every tile must contain the hub next to its window (and the stand-alone reversal tile holds the hub twice)
    if (na > fmax && fmax < 2 * l) { *err = "tile_bits < 2 * hub_bits cannot be scheduled"; return 2; }
    out->prm = prm;
    out->k_eff = std::min(prm.k, n);
    out->tile_bits = fmax;
    out->hub_bits = l;
    // gate counters before fusion
    out->n_h = n;
    out->n_cr = 0;
    for (int d = 1; d <= std::min(out->k_eff, n - 1); ++d) out->n_cr += n - d;
    out->n_swap = n / 2;

    // tensor-memory extended tiles (one more window qubit per pass than the shared-memory tile holds): only for
    // 2^14 tiles (one 512-thread CTA per SM; the kernel is instantiated for that shape only), single transforms, TMA
    // kernels allowed; tried first, dropped if any pass cannot be lowered
    const bool ext_ok = fmax == 14 && prm.batch_bits == 0 && !(prm.flags & (1u | 2u | 4u | 16u)) && n > fmax + 1;
    if ((prm.flags & 32u) && prm.batch_bits != 0) { *err = "deferred swaps are not available for batched plans"; return 2; }
    for (int attempt = ext_ok ? 0 : 1; attempt < 2; ++attempt) {
        const int fplan = attempt == 0 ? fmax + 1 : fmax;  // tile bits the schedule may use
        std::vector<PassSpec> specs;
        out->passes.clear();
        out->ext_tile = attempt == 0;
        out->folded = false;
        if (prm.flags & 32u) {
            if (n <= fmax) {
                build_unfolded(n, prm.max_fused, fmax, l, &specs);  // one tile: simply leave the reversal out
                specs.back().moves.clear();
            } else if (!build_deferred(n, prm.max_fused, fplan, l, &specs)) {
                if (attempt == 0) continue;
                *err = "deferred swaps: this tile / hub combination cannot be scheduled";
                return 2;
            }
            out->folded = true;  // no stand-alone permutation pass
        } else if (!(prm.flags & 2u)) {
            out->folded = build_folded(n, prm.max_fused, fplan, l, &specs);
        }
        if (!out->folded) {
            if (attempt == 0) continue;  // the extension only exists for folded schedules
            specs.clear();
            // batched transforms that fit one tile: two two-step passes (TMA kernel) beat one three-step pass
            const int wcap = (prm.batch_bits > 0 && n > 10 && n <= fmax) ? std::min(prm.max_fused, (n + 1) / 2) : prm.max_fused;
            build_unfolded(n, wcap, fmax, l, &specs);
        }
        // batched plans: the batch index occupies address bits [n, na); they hold no qubit (ids >= n stand for
        // "never processed"), never move, and serve as tile-index bits or passive in-tile bits
        if (na > n)
            for (auto& ps : specs) add_extras(ps, na, std::min(fmax, na));
        std::string e2;
        if (lower_all(prm, specs, na, out->k_eff, l, fmax, out, &e2)) {
            out->ext_tile = false;
            for (const QftPassDesc& d : out->passes) out->ext_tile = out->ext_tile || d.xt;
            break;
        }
        if (attempt == 1) { *err = e2; return 5; }
    }
    if (!(prm.flags & (1u | 2u | 4u | 16u | 32u)) && prm.max_fused <= 6 && prm.max_fused < fmax - l && n > fmax) {
        // Small windows (PAPER.md:145's cap on the fused size; BASELINE config 3 sweeps it down to 2): besides the
        // schedule above (if it exists), cut the folded schedule's windows into sub-passes.  For every hub size
        // (unless the caller fixed it) and width of the outer windows, lower the candidate and keep the cheapest
        // by a rough per-pass cost of the kernel each pass ended up with.
        auto pass_cost = [](const QftPassDesc& d) -> long {
            return d.kernel == QFT_KERNEL_TMA2 ? (d.npair || d.f < 13 ? 12 : 10) : d.kernel == QFT_KERNEL_FUSED2 ? 25 : (d.f >= 10 && d.f <= 11 && !d.npair ? 40 : 100);
        };
        auto cost_of = [&](std::vector<PassSpec>& cand, int lh, QftHostPlan* tmp) -> long {
            *tmp = *out;
            tmp->passes.clear();
            tmp->hub_bits = lh;
            if (na > n)
                for (auto& ps : cand) add_extras(ps, na, std::min(fmax, na));
            std::string e3;
            if (!lower_all(prm, cand, na, out->k_eff, lh, fmax, tmp, &e3)) return -1;
            long c = 0;
            for (const QftPassDesc& d : tmp->passes) c += pass_cost(d);
            return c;
        };
        QftHostPlan best_plan, tmp;
        long best = 0;  // the cost of the schedule found above
        for (const QftPassDesc& d : out->passes) best += pass_cost(d);
        const long native = best;
        for (int lh = l; lh >= (prm.hub_bits ? l : 3) && lh >= 1; --lh)
            for (int we = lh; we <= fmax - lh; ++we) {
                std::vector<PassSpec> cand;
                if (!build_folded_split(n, prm.max_fused, fmax, lh, we, &cand)) continue;
                if ((long)cand.size() * 10 >= best) continue;  // cannot win
                const long c = cost_of(cand, lh, &tmp);
#ifdef QFT_PLAN_DEBUG
                fprintf(stderr, "split candidate hub %d we %d: %zu passes, cost %ld\n", lh, we, cand.size(), c);
#endif
                if (c >= 0 && c < best) { best = c; best_plan = tmp; }
            }
        if (best < native) {
            *out = best_plan;
            out->folded = true;
            out->ext_tile = false;
        }
    }
    // normalisation: every H contributes 1/sqrt 2; applied once, in the last pass
    double sc = std::pow(2.0, -0.5 * n);
    if (prm.norm == 1) sc = 1.0;
    else if (prm.norm == 2) sc = std::pow(2.0, -1.0 * n);
    // the last pass that has steps carries the scale (a trailing permutation pass has none)
    for (int i = (int)out->passes.size() - 1; i >= 0; --i) {
        if (out->passes[i].nsteps > 0) {
            out->passes[i].scale = (float)sc;
            out->passes[i].do_scale = (sc != 1.0);
            break;
        }
    }
    return qft_check_plan(*out, err);
}

// Independent re-derivation from the descriptors alone.
int qft_check_plan(const QftHostPlan& plan, std::string* err) {
    const int nq = plan.prm.n;                      // qubits of one transform
    const int n = plan.prm.n + plan.prm.batch_bits;  // address bits
    std::vector<int> qubit_at(n);
    for (int a = 0; a < n; ++a) qubit_at[a] = a;
    int next_qubit = nq - 1;
    char buf[256];
    int pi = 0;
    int nscaled = 0;
    for (const QftPassDesc& d : plan.passes) {
        auto fail = [&](const char* what) {
            snprintf(buf, sizeof buf, "self-check: pass %d: %s", pi, what);
            *err = buf;
            return 5;
        };
        if (d.n != n || d.f + d.ntile != n || d.f < 1 || d.f > QFT_MAX_TILE_BITS) return fail("sizes");
        if (d.xt != 0 && d.xt != 1) return fail("xt");
        if (d.xt && d.kernel != QFT_KERNEL_TMA2) return fail("extended tile without the TMA kernel");
        std::vector<int> inF(n, 0), inFst(n, 0);
        for (int j = 0; j < d.f; ++j) {
            if (d.F[j] < 0 || d.F[j] >= n || inF[d.F[j]]) return fail("F not a set of address bits");
            if (j && d.F[j] <= d.F[j - 1]) return fail("F not ascending");
            inF[d.F[j]] = 1;
            if (d.Fst[j] < 0 || d.Fst[j] >= n || inFst[d.Fst[j]]) return fail("Fst not a set of address bits");
            if (j && d.Fst[j] <= d.Fst[j - 1]) return fail("Fst not ascending");
            inFst[d.Fst[j]] = 1;
        }
        // the tile a CTA owns: load side F (+ the half-tile bit), store side Fst (+ the butterfly's bit);
        // in place is safe only if the two are the same set of addresses
        std::vector<int> inTile(inF);
        if (d.xt) {
            const int ag = d.xt_ld_addr, bg = d.xt_st_addr;
            if (ag < 0 || ag >= n || inF[ag] || bg < 0 || bg >= n || inFst[bg]) return fail("extended tile: half-tile bits");
            inTile[ag] = 1;
            inFst[bg] = 1;
            if (d.ntile < 1 || d.tile_addr[d.ntile - 1] != ag) return fail("extended tile: half-tile bit is not the last tile-index bit");
            if (2 * d.npair > d.ntile - 1) return fail("extended tile: half-tile bit inside a pair");
            if (qubit_at[ag] != d.xt_q || d.xt_q != d.win_lo - 1) return fail("extended tile: qubit");
        }
        for (int a = 0; a < n; ++a)
            if (inTile[a] != inFst[a]) return fail("store tile differs from load tile (not in place)");
        const int l = std::min(plan.hub_bits, n);
        for (int j = 0; j < std::min(l, d.f); ++j)
            if (d.F[j] != j || d.Fst[j] != j) return fail("hub not in tile");
        // canonical map consistent with the tracked layout
        std::vector<int> seen(d.f, 0);
        for (int j = 0; j < d.f; ++j) {
            const int c = d.ld_canon[j];
            if (c < 0 || c >= d.f || seen[c]) return fail("ld_canon not a permutation");
            seen[c] = 1;
            if (d.log_canon[c] != qubit_at[d.F[j]]) return fail("log_canon disagrees with the layout");
        }
        for (int c = 1; c < d.f; ++c)
            if (d.log_canon[c] <= d.log_canon[c - 1]) return fail("canonical order not by logical qubit");
        std::fill(seen.begin(), seen.end(), 0);
        for (int j = 0; j < d.f; ++j) {
            const int c = d.st_canon[j];
            if (c < 0 || c >= d.f || seen[c]) return fail("st_canon not a permutation (tile not closed)");
            seen[c] = 1;
        }
        // tile-index bits = exactly the other address bits
        std::vector<int> cover(n, 0);
        for (int i = 0; i < d.ntile; ++i) {
            const int a = d.tile_addr[i];
            if (a < 0 || a >= n || inF[a] || cover[a]) return fail("tile_addr");
            cover[a] = 1;
            if (d.log_tile[i] != qubit_at[a]) return fail("log_tile disagrees with the layout");
        }
        if (2 * d.npair > d.ntile || d.npair < 0) return fail("npair");
        // steps: descending logical order, each target inside the tile on the stated canonical bits
        for (int s = 0; s < d.nsteps; ++s) {
            const QftStep& st = d.steps[s];
            if (st.r < 1 || st.r > QFT_MAX_RADIX_BITS || st.a < 0 || st.a + st.r > d.f) return fail("step shape");
            for (int i = 0; i < st.r; ++i) {
                const int q = st.t_hi - i;
                if (q != next_qubit) return fail("gates out of circuit order");
                if (d.log_canon[st.a + st.r - 1 - i] != q) return fail("step qubit not on its canonical bit");
                --next_qubit;
            }
        }
        if (d.nsteps > 0 && d.win_lo != next_qubit + 1) return fail("win_lo");
        if (d.xt) {
            // the butterfly between the halves comes after every register step of the pass
            if (d.xt_q != next_qubit) return fail("extended tile: gates out of circuit order");
            --next_qubit;
        }
        if (d.kernel == QFT_KERNEL_TMA2) {
            // replay the kernel's index maps: every (thread, register) of both steps
            const QftTma2Desc& t = d.tma;
            const int f = d.f, lt = f - 5, nt = 1 << lt;
            if (d.nsteps != 2 || d.log2_threads != lt) return fail("tma2: shape");
            const QftStep s1 = d.steps[0], s2 = d.steps[1];
            std::vector<int> canon_at_load(n, -1);
            for (int j = 0; j < f; ++j) canon_at_load[d.F[j]] = d.ld_canon[j];
            {
                // landing order = the box bits of the tensor-map dims, dimension by dimension
                int nl = 0;
                for (int i = 0; i < 5; ++i)
                    for (int b = 0; b < t.tma_box[i]; ++b) {
                        if (nl >= f || t.land_addr[nl] != t.tma_lo[i] + b) return fail("tma2: land_addr");
                        if (t.land_addr[nl] < 0 || t.land_addr[nl] >= n || canon_at_load[t.land_addr[nl]] < 0) return fail("tma2: landing bit outside the tile");
                        ++nl;
                    }
                if (nl != f) return fail("tma2: landing bits");
            }
            // canonical index of (tid, B) in step 1, recovered from the load columns
            auto canon1 = [&](int tid, int B) {
                uint32_t off = 0;
                for (int j = 0; j < lt; ++j) if ((tid >> j) & 1) off ^= t.s1_tid_ld[j];
                for (int b = 0; b < 5; ++b) if ((B >> b) & 1) off ^= t.s1_reg_ld[b];
                const uint32_t idx = off >> 3;  // landing index
                uint32_t c = 0;
                for (int j = 0; j < f; ++j) if ((idx >> j) & 1u) c |= 1u << canon_at_load[t.land_addr[j]];
                return std::make_pair(idx, c);
            };
            const uint32_t xslots = 1u << f;
            std::vector<int> mid_canon((size_t)1 << f, -1);
            std::vector<char> seen_ld((size_t)1 << f, 0);
            for (int b = 0; b < s1.r; ++b) if (t.s1_reg_key[b]) return fail("tma2: group bit in key");
            for (int tid = 0; tid < nt; ++tid) {
                uint32_t key = 0, offm_t = 0;
                for (int j = 0; j < lt; ++j) if ((tid >> j) & 1) { key ^= t.s1_tid_key[j]; offm_t ^= t.s1_tid_mid[j]; }
                for (int B = 0; B < 32; ++B) {
                    auto ic = canon1(tid, B);
                    if (ic.first >= (1u << f) || seen_ld[ic.first]) return fail("tma2: step 1 reads are not a bijection");
                    seen_ld[ic.first] = 1;
                    const uint32_t c = ic.second;
                    // register bits [0, r1) must be group 1's canonical bits
                    if (((c >> s1.a) & ((1u << s1.r) - 1u)) != (uint32_t)(B & ((1 << s1.r) - 1))) return fail("tma2: step 1 register bits");
                    uint32_t offm = offm_t;
                    for (int b = 0; b < 5; ++b) if ((B >> b) & 1) offm ^= t.s1_reg_mid[b];
                    // the key comes from thread + batch bits only; group bits contribute 0
                    uint32_t kb = key;
                    for (int b = s1.r; b < 5; ++b) if ((B >> b) & 1) kb ^= t.s1_reg_key[b];
                    if ((kb & 31u) != ((c >> s2.a) & ((1u << s2.r) - 1u))) return fail("tma2: step 1 key (group 2 value)");
                    if (((kb >> 8) & 4095u) != (c & ((1u << t.eb) - 1u))) return fail("tma2: step 1 key (e)");
                    if (offm & 7u) return fail("tma2: mid offset alignment");
                    const uint32_t slot = offm >> 3;
                    if (slot >= xslots || mid_canon[slot] != -1) return fail("tma2: exchange layout is not a bijection");
                    mid_canon[slot] = (int)c;
                }
            }
            // bank check: lanes 0-15 of every warp, same register, distinct 8-byte bank pairs
            for (int w = 0; w < nt / 16; ++w) {
                for (int pass2 = 0; pass2 < 2; ++pass2) {
                    int banks = 0;
                    for (int lane = 0; lane < 16; ++lane) {
                        const int tid = w * 16 + lane;
                        uint32_t off = 0;
                        for (int j = 0; j < lt; ++j)
                            if ((tid >> j) & 1) off ^= pass2 ? t.s2_tid_mid[j] : t.s1_tid_mid[j];
                        banks |= 1 << ((off >> 3) & 15);
                    }
                    if (banks != 0xFFFF) return fail("tma2: exchange layout has bank conflicts");
                }
                int banks = 0;
                for (int lane = 0; lane < 16; ++lane) {
                    const int tid = w * 16 + lane;
                    uint32_t off = 0;
                    for (int j = 0; j < lt; ++j) if ((tid >> j) & 1) off ^= t.s1_tid_ld[j];
                    banks |= 1 << ((off >> 3) & 15);
                }
                if (banks != 0xFFFF) return fail("tma2: landing layout read with bank conflicts");
            }
            auto st_index_of_addr = [&](int addr) {
                for (int jj = 0; jj < f; ++jj) if (d.Fst[jj] == addr) return jj;
                return -1;
            };
            std::vector<char> seen_st((size_t)1 << f, 0);
            for (int tid = 0; tid < nt; ++tid) {
                uint32_t key = 0, offm_t = 0;
                uint32_t st_idx_t = 0;
                for (int j = 0; j < lt; ++j) if ((tid >> j) & 1) {
                    key ^= t.s2_tid_key[j]; offm_t ^= t.s2_tid_mid[j];
                    const int found = st_index_of_addr(t.s2_tid_addr[j]);
                    if (found < 0) return fail("tma2: store address bit outside the tile");
                    st_idx_t |= 1u << found;
                }
                for (int B = 0; B < 32; ++B) {
                    uint32_t offm = offm_t, st_idx = st_idx_t;
                    uint32_t kb = key;
                    for (int b = 0; b < 5; ++b) if ((B >> b) & 1) {
                        offm ^= t.s2_reg_mid[b];
                        const int found = st_index_of_addr(t.s2_reg_addr[b]);
                        if (found < 0) return fail("tma2: store address bit outside the tile");
                        st_idx |= 1u << found;
                        if (b >= s2.r) kb ^= t.s2_reg_key[b];
                    }
                    const uint32_t slot = offm >> 3;
                    if (slot >= xslots || mid_canon[slot] < 0) return fail("tma2: step 2 reads an empty slot");
                    const uint32_t c = (uint32_t)mid_canon[slot];
                    if (((c >> s2.a) & ((1u << s2.r) - 1u)) != (uint32_t)(B & ((1 << s2.r) - 1))) return fail("tma2: step 2 register bits");
                    if ((kb & 31u) != ((c >> s1.a) & ((1u << s1.r) - 1u))) return fail("tma2: step 2 key (group 1 value)");
                    if (((kb >> 8) & 4095u) != (c & ((1u << t.eb) - 1u))) return fail("tma2: step 2 key (e)");
                    // the element with canonical index c must land on store-order index st(c)
                    uint32_t want = 0;
                    for (int j = 0; j < f; ++j) if ((c >> d.st_canon[j]) & 1u) want |= 1u << j;
                    if (want != st_idx) return fail("tma2: store address disagrees with the layout adapter");
                    if (seen_st[st_idx]) return fail("tma2: stores are not a bijection");
                    seen_st[st_idx] = 1;
                }
            }
            for (int j = 0; j < std::min<int>(t.tma_box[0], 3) && j < lt; ++j) if (t.s2_tid_addr[j] != d.Fst[j] || d.Fst[j] != j) return fail("tma2: store lanes do not run along the hub");
            if (t.eb != s2.a || t.eb > QFT_TMA2_EB_MAX || (t.eb > QFT_TMA2_EB_DIRECT && (s1.r + s2.r > 6 || d.xt))) return fail("tma2: eb");
            for (int c = 0; c < t.eb; ++c) if (t.e_log[c] != d.log_canon[c]) return fail("tma2: e_log");
            if (t.t1_lo != s1.t_hi - s1.r + 1 || t.t2_lo != s2.t_hi - s2.r + 1 || t.t1_lo != t.t2_lo + s2.r) return fail("tma2: group qubits");
            if (t.r1 != s1.r || t.r2 != s2.r) return fail("tma2: group sizes");
            // tensor-map dims: the box dims are disjoint runs that together are exactly F, dim 0 starts at
            // bit 0; every tile-index bit lies inside the span of a box-1 dim (its coordinate is the tile's
            // base address, which is zero on all tile bits, shifted down to the dim's lowest bit)
            int boxbits = 0;
            std::vector<int> covered(n + 1, 0), spanned(n + 1, 0);
            if (t.tma_lo[0] != 0) return fail("tma2: dimension 0 is not the contiguous one");
            for (int i = 0; i < 5; ++i) {
                if (t.tma_box[i] != 0 && t.tma_box[i] != t.tma_len[i]) return fail("tma2: box");
                if (t.tma_box[i] > 8 || t.tma_len[i] > 31) return fail("tma2: dim too large");
                for (int b = 0; b < t.tma_len[i]; ++b) {
                    const int bit = t.tma_lo[i] + b;
                    if (bit < 0 || bit >= n) return fail("tma2: tensor-map dim outside the state");
                    if (t.tma_box[i] != 0) {
                        if (covered[bit] || !inF[bit]) return fail("tma2: box bits are not the tile bits");
                        covered[bit] = 1;
                    } else {
                        spanned[bit] = 1;
                    }
                }
                boxbits += t.tma_box[i];
            }
            for (int bit = 0; bit < n; ++bit)
                if (!inF[bit] && !spanned[bit]) return fail("tma2: a tile-index bit is outside the tensor map");
            if (boxbits != f || t.tma_box[0] < 1) return fail("tma2: tensor map does not cover the state");
        } else {
            for (int j = 0; j < d.f; ++j)
                if (d.F[j] != d.Fst[j]) return fail("store tile bits differ from load tile bits");
        }
        if (d.do_scale) ++nscaled;
        // permutation
        std::vector<int> nq2(qubit_at);
        for (int j = 0; j < d.f; ++j) {
            // data on canonical bit st_canon[j] lands on address Fst[j]
            nq2[d.Fst[j]] = d.log_canon[d.st_canon[j]];
        }
        if (d.xt) nq2[d.xt_st_addr] = d.xt_q;
        for (int i = 0; i < d.npair; ++i) {
            const int a = d.tile_addr[i], b = d.tile_addr[d.npair + i];
            nq2[a] = qubit_at[b];
            nq2[b] = qubit_at[a];
        }
        qubit_at.swap(nq2);
        ++pi;
    }
    if (next_qubit != -1) { *err = "self-check: not every qubit was processed"; return 5; }
    const bool deferred = (plan.prm.flags & 32u) != 0;  // swaps left to the caller: any layout, but the reported one
    if ((int)plan.out_qubit_at.size() != n) { *err = "self-check: output layout missing"; return 5; }
    for (int a = 0; a < n; ++a) {
        if (qubit_at[a] != plan.out_qubit_at[a]) { *err = "self-check: final layout differs from the reported one"; return 5; }
        if (!deferred && qubit_at[a] != (a < nq ? nq - 1 - a : a)) { *err = "self-check: final layout is not the bit reversal"; return 5; }
    }
    const bool want_scale = plan.prm.norm != 1;
    if ((want_scale && nscaled != 1) || (!want_scale && nscaled != 0)) { *err = "self-check: scale"; return 5; }
    return 0;
}

// Sharded state (host-side design): the 2^n amplitudes
// live on 2^g ranks, the top g address bits select the rank, and the shards are mapped back to back into one virtual
// range (peer memory over NVLink), so a pass is the same kernel on the same addresses and only the question "which
// rank runs which units" is new.  A rank bit is either a tile-index bit (the units whose value of that bit equals
// the rank's touch only that rank's shard: local) or a tile bit (every unit's rows lie on both values: spanning).
// Rank bits outside the tile are always the top bits of the unit index (they are the highest non-tile addresses), so
// a rank's share is one contiguous unit range: the units whose outside rank bits equal its own, split evenly among
// the 2^g_in ranks that share them.  Unsupported: a rank bit inside a pair involution (the folded schedule never
// does that for g <= hub bits), fewer units than ranks.
// Returns 0, or 2 (unsupported) with *err set.
int qft_shard_range(const QftHostPlan& plan, size_t pass, int rank, int g, long long* unit_lo, long long* unit_n,
                    int* rank_bits_in_tile, std::string* err) {
    const QftPassDesc& d = plan.passes[pass];
    const int n = d.n;
    if (g < 0 || g > 6 || g >= n || rank < 0 || rank >= (1 << g)) { *err = "invalid rank / log2_ranks"; return 1; }
    std::vector<int> inTile(n, 0), inPair(n, 0);
    for (int j = 0; j < d.f; ++j) inTile[d.F[j]] = 1;
    if (d.xt) inTile[d.xt_ld_addr] = 1;
    for (int i = 0; i < 2 * d.npair; ++i) inPair[d.tile_addr[i]] = 1;
    int g_in = 0;
    unsigned o = 0, r_in = 0;
    int m = 0;
    for (int b = 0; b < g; ++b) {
        const int a = n - g + b;
        const unsigned bit = ((unsigned)rank >> b) & 1u;
        if (inPair[a]) { *err = "a rank bit trades places with another address bit in this pass"; return 2; }
        if (inTile[a]) r_in |= bit << g_in++;
        else o |= bit << m++;
    }
    const int ubits = d.ntile - d.xt - (d.npair ? 1 : 0);  // log2 of the number of units
    if (ubits < g) { *err = "fewer units than ranks"; return 2; }
    const long long per_o = 1ll << (ubits - m);  // units that share one value of the outside rank bits
    *unit_n = per_o >> g_in;
    *unit_lo = (long long)o * per_o + (long long)r_in * *unit_n;
    *rank_bits_in_tile = g_in;
    return 0;
}

// Host proof of the sharding rule for every pass and rank: the ranges tile the unit space exactly, and every unit of
// rank r's range has the outside rank bits of r (replayed through the kernel's own unit -> tile -> address maps).
int qft_check_shard(const QftHostPlan& plan, int g, std::string* err) {
    char buf[160];
    for (size_t p = 0; p < plan.passes.size(); ++p) {
        const QftPassDesc& d = plan.passes[p];
        const int n = d.n;
        const int ubits = d.ntile - d.xt - (d.npair ? 1 : 0);
        std::vector<std::pair<long long, long long>> ranges;
        for (int r = 0; r < (1 << g); ++r) {
            long long lo, cnt;
            int g_in;
            const int rc = qft_shard_range(plan, p, r, g, &lo, &cnt, &g_in, err);
            if (rc != 0) return rc;
            ranges.push_back({lo, cnt});
            // first and last unit of the range, and one in the middle: tile-index value -> address bits
            for (long long u : {lo, lo + cnt / 2, lo + cnt - 1}) {
                // unit -> tile index of the unit's first CTA: without pairs the unit itself; with p pairs the
                // cluster id, whose bits above 2p - 1 are the tile-index bits above the pairs
                unsigned long long tile_hi = d.npair ? ((unsigned long long)u >> (2 * d.npair - 1)) << (2 * d.npair) : (unsigned long long)u;
                for (int b = 0; b < g; ++b) {
                    const int a = n - g + b;
                    bool in_tile = d.xt && a == d.xt_ld_addr;
                    for (int j = 0; j < d.f; ++j) in_tile = in_tile || d.F[j] == a;
                    if (in_tile) continue;
                    int idx = -1;
                    for (int i = 0; i < d.ntile - d.xt; ++i)
                        if (d.tile_addr[i] == a) idx = i;
                    if (idx < 0) { *err = "shard check: rank bit is neither a tile nor a tile-index bit"; return 5; }
                    if (((tile_hi >> idx) & 1ull) != (((unsigned)r >> b) & 1u)) {
                        snprintf(buf, sizeof buf, "shard check: pass %zu rank %d: unit %lld lies on another rank", p, r, u);
                        *err = buf;
                        return 5;
                    }
                }
            }
        }
        std::sort(ranges.begin(), ranges.end());
        long long next = 0;
        for (auto& rg : ranges) {
            if (rg.first != next || rg.second < 1) { *err = "shard check: unit ranges do not tile the pass"; return 5; }
            next += rg.second;
        }
        if (next != (1ll << ubits)) { *err = "shard check: unit ranges do not cover the pass"; return 5; }
    }
    return 0;
}

// Per pass, the contiguous sub-range [gate_first, gate_last] of the time-ordered gate list
//   for t = n-1 .. 0:  H(q_t), CR_2(q_{t-1} -> q_t), ..., CR_{min(k,t)+1}(q_{t-min(k,t)} -> q_t);  then the swaps
// that the pass folds ("the contiguous subrange of original gates folded into the block"), with the
// number of Hadamards and controlled rotations in it.  The swaps are not gates of any pass: they are the
// passes' store permutations.
void qft_pass_gates(const QftHostPlan& plan, size_t pass, long long* n_h, long long* n_cr, long long* first,
                    long long* last) {
    const QftPassDesc& d = plan.passes[pass];
    const int k = plan.k_eff;
    *n_h = *n_cr = 0;
    *first = *last = -1;
    if (d.nsteps == 0) return;
    const int t_hi = d.steps[0].t_hi;
    const int t_lo = d.xt ? d.xt_q : d.win_lo;
    long long idx = 0;
    for (int t = plan.prm.n - 1; t > t_hi; --t) idx += 1 + std::min(k, t);
    *first = idx;
    for (int t = t_hi; t >= t_lo; --t) {
        *n_h += 1;
        *n_cr += std::min(k, t);
    }
    *last = idx + *n_h + *n_cr - 1;
}

std::string qft_describe_plan(const QftHostPlan& plan) {
    std::ostringstream o;
    o << "{\"n\":" << plan.prm.n << ",\"batch_bits\":" << plan.prm.batch_bits << ",\"k\":" << plan.k_eff << ",\"sign\":" << plan.prm.sign
      << ",\"norm\":" << plan.prm.norm << ",\"max_fused_qubits\":" << plan.prm.max_fused
      << ",\"tile_bits\":" << plan.tile_bits << ",\"hub_bits\":" << plan.hub_bits
      << ",\"folded\":" << (plan.folded ? "true" : "false") << ",\"swaps\":\"" << ((plan.prm.flags & 32u) ? "deferred" : "applied")
      << "\",\"ext_tile\":" << (plan.ext_tile ? "true" : "false")
      << ",\"n_h\":" << plan.n_h << ",\"n_cr\":" << plan.n_cr
      << ",\"n_swap\":" << plan.n_swap << ",\"out_qubit_of_bit\":[";
    for (size_t a = 0; a < plan.out_qubit_at.size(); ++a) o << (a ? "," : "") << plan.out_qubit_at[a];
    o << "],\"passes\":[";
    for (size_t i = 0; i < plan.passes.size(); ++i) {
        const QftPassDesc& d = plan.passes[i];
        if (i) o << ",";
        o << "{\"kernel\":\"" << (d.kernel == QFT_KERNEL_TMA2 ? (d.xt ? "tma2x" : "tma2") : d.kernel == QFT_KERNEL_FUSED2 ? "fused2" : "generic")
          << "\",\"tile_bits\":" << d.f + d.xt << ",\"F\":[";
        {
            std::vector<int> F(d.F, d.F + d.f);
            if (d.xt) F.push_back(d.xt_ld_addr);
            std::sort(F.begin(), F.end());
            for (size_t j = 0; j < F.size(); ++j) o << (j ? "," : "") << F[j];
        }
        o << "],\"window\":[";
        bool first = true;
        for (int s = 0; s < d.nsteps; ++s)
            for (int q = 0; q < d.steps[s].r; ++q) {
                o << (first ? "" : ",") << (int)d.steps[s].t_hi - q;
                first = false;
            }
        if (d.xt) o << "," << (int)d.xt_q;
        o << "],\"steps\":[";
        for (int s = 0; s < d.nsteps; ++s) o << (s ? "," : "") << (int)d.steps[s].r;
        if (d.xt) o << ",1";
        long long nh, ncr, g0, g1;
        qft_pass_gates(plan, i, &nh, &ncr, &g0, &g1);
        o << "],\"n_h\":" << nh << ",\"n_cr\":" << ncr << ",\"gate_first\":" << g0 << ",\"gate_last\":" << g1;
        o << ",\"store_addr_of_canon\":[";
        {
            std::vector<int> sa(d.f);
            for (int j = 0; j < d.f; ++j) sa[d.st_canon[j]] = d.Fst[j];
            for (int c = 0; c < d.f; ++c) o << (c ? "," : "") << sa[c];
        }
        o << "],\"canon_qubits\":[";
        for (int c = 0; c < d.f; ++c) o << (c ? "," : "") << (int)d.log_canon[c];
        o << "]";
        if (d.xt) o << ",\"ext\":{\"qubit\":" << (int)d.xt_q << ",\"load_addr\":" << (int)d.xt_ld_addr << ",\"store_addr\":" << (int)d.xt_st_addr << "}";
        o << ",\"pair_swaps\":[";
        for (int p = 0; p < d.npair; ++p)
            o << (p ? "," : "") << "[" << (int)d.tile_addr[p] << "," << (int)d.tile_addr[d.npair + p] << "]";
        o << "],\"scale\":" << d.scale << ",\"bytes\":" << (16.0 * std::ldexp(1.0, plan.prm.n + plan.prm.batch_bits)) << "}";
    }
    o << "]}";
    return o.str();
}
