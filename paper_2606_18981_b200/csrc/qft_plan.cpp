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
#include <cstring>
#include <set>
#include <sstream>

namespace {

struct PassSpec {
    std::vector<int> window;                 // logical qubits, descending; empty = permutation only
    std::vector<int> F;                      // tile address bits
    std::vector<std::pair<int, int>> moves;  // in-tile: data on address first goes to address second
    std::vector<std::pair<int, int>> swaps;  // non-tile address pairs (lo, hi) that trade places
};

int ilog2_ceil_div(int a, int b) { return (a + b - 1) / b; }

void add_extras(PassSpec& ps, int n, int ftarget) {
    std::set<int> used(ps.F.begin(), ps.F.end());
    std::set<int> sw;
    for (auto& s : ps.swaps) { sw.insert(s.first); sw.insert(s.second); }
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
bool build_folded(int n, int wcap, int fmax, int l, std::vector<PassSpec>* out) {
    if (n <= fmax) return false;
    int w = std::min(wcap, fmax - l);
    if (n <= 2 * w) w = (n - 1) / 2;
    if (w < l || w < 1) return false;
    int nmid_passes = ilog2_ceil_div(n - 2 * w, w);
    const int K = 2 + nmid_passes;
    int we = std::min(w, ilog2_ceil_div(n, K));
    while (n - 2 * we > nmid_passes * w) ++we;
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

std::vector<int> step_sizes(int w) {
    if (w <= 0) return {};
    const int g = ilog2_ceil_div(w, QFT_MAX_RADIX_BITS);
    return split_balanced(w, g);  // larger groups first
}

// Turn a PassSpec into the kernel descriptor given the current layout; updates qubit_at.
bool lower_pass(const PassSpec& ps, int n, int k, int conj, int hub, bool allow_fused, std::vector<int>& qubit_at,
                QftPassDesc* d, std::string* err) {
    std::memset(d, 0, sizeof(*d));
    const int f = (int)ps.F.size();
    if (f > QFT_MAX_TILE_BITS || n - f > QFT_MAX_TILEIDX_BITS) { *err = "tile too large"; return false; }
    d->n = n; d->f = f; d->ntile = n - f; d->k = k; d->conj = conj; d->scale = 1.0f; d->do_scale = 0;
    d->kernel = QFT_KERNEL_GENERIC;
    int lt = f - 2;
    if (lt < 5) lt = 5;
    if (lt > 8) lt = 8;
    d->log2_threads = lt;
    std::vector<int> inF(n, 0);
    for (int a : ps.F) inF[a] = 1;
    // canonical order: in-tile qubits ascending by logical id
    std::vector<int> qs;
    for (int a : ps.F) qs.push_back(qubit_at[a]);
    std::sort(qs.begin(), qs.end());
    std::vector<int> canon_of_q(n, -1);
    for (int c = 0; c < f; ++c) { canon_of_q[qs[c]] = c; d->log_canon[c] = (int8_t)qs[c]; }
    std::vector<int> dest(n);
    for (int a = 0; a < n; ++a) dest[a] = a;
    for (auto& m : ps.moves) {
        if (!inF[m.first] || !inF[m.second]) { *err = "move leaves the tile"; return false; }
        dest[m.first] = m.second;
    }
    for (int j = 0; j < f; ++j) {
        d->F[j] = (int8_t)ps.F[j];
        d->ld_canon[j] = (int8_t)canon_of_q[qubit_at[ps.F[j]]];
    }
    std::vector<int> src_of(n, -1);
    for (int a : ps.F) {
        if (src_of[dest[a]] != -1) { *err = "in-tile moves are not a permutation"; return false; }
        src_of[dest[a]] = a;
    }
    for (int j = 0; j < f; ++j) {
        if (src_of[ps.F[j]] < 0) { *err = "in-tile moves are not a permutation"; return false; }
        d->st_canon[j] = (int8_t)canon_of_q[qubit_at[src_of[ps.F[j]]]];
    }
    // tile-index bits: swapped pairs first (lo side, then hi side), then the rest ascending
    const int p = (int)ps.swaps.size();
    d->npair = p;
    std::vector<int> taken(n, 0);
    for (int i = 0; i < p; ++i) {
        const int a = ps.swaps[i].first, b = ps.swaps[i].second;
        if (inF[a] || inF[b] || taken[a] || taken[b] || a == b) { *err = "bad swap"; return false; }
        taken[a] = taken[b] = 1;
        d->tile_addr[i] = (int8_t)a;
        d->tile_addr[p + i] = (int8_t)b;
    }
    int ti = 2 * p;
    for (int a = 0; a < n; ++a)
        if (!inF[a] && !taken[a]) d->tile_addr[ti++] = (int8_t)a;
    if (ti != n - f) { *err = "tile index bits do not add up"; return false; }
    for (int i = 0; i < n - f; ++i) d->log_tile[i] = (int8_t)qubit_at[d->tile_addr[i]];
    // steps
    d->win_lo = -1;
    d->nsteps = 0;
    if (!ps.window.empty()) {
        const int w = (int)ps.window.size();
        for (int i = 0; i < w; ++i) {
            if (ps.window[i] != ps.window[0] - i) { *err = "window not contiguous"; return false; }
            if (canon_of_q[ps.window[i]] < 0) { *err = "window qubit outside the tile"; return false; }
        }
        d->win_lo = ps.window[w - 1];
        int t = ps.window[0];
        for (int r : step_sizes(w)) {
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
    if (d->nsteps == 2 && allow_fused) {
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
    // apply the permutation to the tracking
    std::vector<int> nq(qubit_at);
    for (int a : ps.F) nq[dest[a]] = qubit_at[a];
    for (auto& s : ps.swaps) { nq[s.first] = qubit_at[s.second]; nq[s.second] = qubit_at[s.first]; }
    qubit_at.swap(nq);
    return true;
}

}  // namespace

int qft_build_plan(const QftPlanParams& prm, QftHostPlan* out, std::string* err) {
    const int n = prm.n;
    if (n < 1 || n > 34 || prm.k < 0 || prm.max_fused < 1 || (prm.sign != 1 && prm.sign != -1) || prm.norm < 0 ||
        prm.norm > 2) {
        *err = "invalid argument";
        return 1;
    }
    int fmax = prm.tile_bits ? prm.tile_bits : 13;
    int l = prm.hub_bits ? prm.hub_bits : 3;
    if (fmax < 2 || fmax > QFT_MAX_TILE_BITS || l < 1 || l > 5 || l >= fmax) {
        *err = "unsupported tile_bits / hub_bits";
        return 2;
    }
    if (n - std::min(fmax, n) > 30) { *err = "tile_bits too small for this n"; return 2; }
    out->prm = prm;
    out->k_eff = std::min(prm.k, n);
    out->tile_bits = fmax;
    out->hub_bits = l;
    out->passes.clear();
    // gate counters before fusion
    out->n_h = n;
    out->n_cr = 0;
    for (int d = 1; d <= std::min(out->k_eff, n - 1); ++d) out->n_cr += n - d;
    out->n_swap = n / 2;

    std::vector<PassSpec> specs;
    out->folded = false;
    if (!(prm.flags & 2u)) out->folded = build_folded(n, prm.max_fused, fmax, l, &specs);
    if (!out->folded) {
        specs.clear();
        build_unfolded(n, prm.max_fused, fmax, l, &specs);
    }
    std::vector<int> qubit_at(n);
    for (int a = 0; a < n; ++a) qubit_at[a] = a;
    int wmaxseen = 0;
    for (auto& ps : specs) {
        QftPassDesc d;
        if (!lower_pass(ps, n, out->k_eff, prm.sign == 1 ? 1 : 0, l, !(prm.flags & 1u), qubit_at, &d, err)) return 5;
        wmaxseen = std::max(wmaxseen, (int)ps.window.size());
        out->passes.push_back(d);
    }
    out->window = wmaxseen;
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
    const int n = plan.prm.n;
    std::vector<int> qubit_at(n);
    for (int a = 0; a < n; ++a) qubit_at[a] = a;
    int next_qubit = n - 1;
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
        std::vector<int> inF(n, 0);
        for (int j = 0; j < d.f; ++j) {
            if (d.F[j] < 0 || d.F[j] >= n || inF[d.F[j]]) return fail("F not a set of address bits");
            if (j && d.F[j] <= d.F[j - 1]) return fail("F not ascending");
            inF[d.F[j]] = 1;
        }
        const int l = std::min(plan.hub_bits, n);
        for (int j = 0; j < std::min(l, d.f); ++j)
            if (d.F[j] != j) return fail("hub not in tile");
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
        if (d.do_scale) ++nscaled;
        // permutation
        std::vector<int> nq(qubit_at);
        for (int j = 0; j < d.f; ++j) {
            // data on canonical bit st_canon[j] lands on address F[j]
            nq[d.F[j]] = d.log_canon[d.st_canon[j]];
        }
        for (int i = 0; i < d.npair; ++i) {
            const int a = d.tile_addr[i], b = d.tile_addr[d.npair + i];
            nq[a] = qubit_at[b];
            nq[b] = qubit_at[a];
        }
        qubit_at.swap(nq);
        ++pi;
    }
    if (next_qubit != -1) { *err = "self-check: not every qubit was processed"; return 5; }
    for (int a = 0; a < n; ++a)
        if (qubit_at[a] != n - 1 - a) { *err = "self-check: final layout is not the bit reversal"; return 5; }
    const bool want_scale = plan.prm.norm != 1;
    if ((want_scale && nscaled != 1) || (!want_scale && nscaled != 0)) { *err = "self-check: scale"; return 5; }
    return 0;
}

std::string qft_describe_plan(const QftHostPlan& plan) {
    std::ostringstream o;
    o << "{\"n\":" << plan.prm.n << ",\"k\":" << plan.k_eff << ",\"sign\":" << plan.prm.sign
      << ",\"norm\":" << plan.prm.norm << ",\"max_fused_qubits\":" << plan.prm.max_fused
      << ",\"tile_bits\":" << plan.tile_bits << ",\"hub_bits\":" << plan.hub_bits
      << ",\"folded\":" << (plan.folded ? "true" : "false") << ",\"n_h\":" << plan.n_h << ",\"n_cr\":" << plan.n_cr
      << ",\"n_swap\":" << plan.n_swap << ",\"passes\":[";
    for (size_t i = 0; i < plan.passes.size(); ++i) {
        const QftPassDesc& d = plan.passes[i];
        if (i) o << ",";
        o << "{\"kernel\":\"" << (d.kernel == QFT_KERNEL_FUSED2 ? "fused2" : "generic") << "\",\"tile_bits\":" << d.f
          << ",\"F\":[";
        for (int j = 0; j < d.f; ++j) o << (j ? "," : "") << (int)d.F[j];
        o << "],\"window\":[";
        bool first = true;
        for (int s = 0; s < d.nsteps; ++s)
            for (int q = 0; q < d.steps[s].r; ++q) {
                o << (first ? "" : ",") << (int)d.steps[s].t_hi - q;
                first = false;
            }
        o << "],\"steps\":[";
        for (int s = 0; s < d.nsteps; ++s) o << (s ? "," : "") << (int)d.steps[s].r;
        o << "],\"store_addr_of_canon\":[";
        {
            std::vector<int> sa(d.f);
            for (int j = 0; j < d.f; ++j) sa[d.st_canon[j]] = d.F[j];
            for (int c = 0; c < d.f; ++c) o << (c ? "," : "") << sa[c];
        }
        o << "],\"canon_qubits\":[";
        for (int c = 0; c < d.f; ++c) o << (c ? "," : "") << (int)d.log_canon[c];
        o << "],\"pair_swaps\":[";
        for (int p = 0; p < d.npair; ++p)
            o << (p ? "," : "") << "[" << (int)d.tile_addr[p] << "," << (int)d.tile_addr[d.npair + p] << "]";
        o << "],\"scale\":" << d.scale << ",\"bytes\":" << (16.0 * std::ldexp(1.0, plan.prm.n)) << "}";
    }
    o << "]}";
    return o.str();
}
