// qft_tma.cuh -- the persistent TMA-staged two-step pass kernel (QFT_KERNEL_TMA2), sm_100a.
//
// One CTA owns one 2^f-amplitude shared-memory buffer and walks over tiles (stride = grid size).
// Per tile, per amplitude: HBM --TMA--> smem -> registers -> smem -> registers -> HBM.
//   load   : one elected thread issues cp.async.bulk.tensor (UTMALDG) for the whole tile -- a 5-D box of
//            the state seen as a tensor over its address-bit runs -- and everybody waits on an mbarrier;
//            no thread computes a global load address, and the load of tile i+1 is issued as soon as
//            the buffer is free, so it is in flight while tile i is still being transformed and stored;
//   step 1 : each thread takes the 32 amplitudes of its radix-2^R1 butterflies, applies H and the
//            controlled-R_m among the window's R1 highest qubits with packed FP32x2
//            arithmetic and writes to an XOR-swizzled exchange layout;
//   step 2 : first the phases group 2's qubits contribute to group 1 (diagonal, so they
//            may wait until after the exchange), then the same butterflies for the window's R2 lower
//            qubits, then one more phase per amplitude: the product
//            of every controlled-R_m from a qubit *below* the window onto any of the window's qubits.
//            For group 1 that phase was deferred: it is diagonal in bits step 2 does not touch, so it
//            commutes with step 2 and the two multiplications merge into one;
//   store  : straight from registers, lanes along the hub so every warp store covers whole granules,
//            at the addresses the layout adapter dictates; for a pair pass into the
//            partner tile after a cluster barrier (the partner's TMA load has completed by then).
// Tensor-memory extended tiles (XT = 1, QftPassDesc::xt): the tile a CTA owns has 2^(F+1) amplitudes, one
// address bit more than shared memory holds.  The CTA runs its two halves through steps 1 and 2 one after
// the other; the first half's results wait in tensor memory (tcgen05.st, 64 words per thread: Blackwell's
// 256 KB of TMEM per SM are otherwise idle in this kernel), and when the second half is in registers
// each thread reads its own words back (tcgen05.ld) and applies the gates of one more qubit, the window's
// lowest: H as a radix-2 butterfly between the halves, times the controlled-R_m onto it from the qubits
// below the window (one factor per tile row e).  Both halves are then stored: the window grows by one
// qubit, i.e. 11 qubits per pass with 128-byte granules or 10 with 256-byte granules, at 2^14-amplitude
// shared-memory tiles.
// Phase factors are never evaluated per amplitude: per CTA 32 x R1 "mid" bases, per tile 2^eb x (R1+R2)
// "end" bases (sincos on an exact 32-bit fraction of a turn), multiplied up along the subset tree.
#pragma once
#include <cuda.h>

#include "qft_device.cuh"
#include "qft_packed.cuh"

namespace qftk {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

__device__ __forceinline__ void tma_load_5d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2,
                                            int c3, int c4) {
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], "
        "[%2];" ::"r"(smem_u32(dst)),
        "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4)
        : "memory");
}

// ---- tensor memory as a parking lot (XT) ----
// 32x32b shape: thread i of a warp owns TMEM lane 32 (warp % 4) + i; .xN moves N consecutive columns
// (32-bit words) of that lane to / from N registers.
__device__ __forceinline__ void tmem_alloc(uint32_t* smem_dst, uint32_t ncols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(smem_dst)), "r"(ncols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
#define QFT_U(v) "r"(__float_as_uint(v))
// park amplitudes x[BASE .. BASE+15] (32 words) at columns [taddr, taddr + 32)
template <int BASE>
__device__ __forceinline__ void tmem_park16(uint32_t taddr, const float2 (&x)[32]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};" ::"r"(taddr),
        QFT_U(x[BASE + 0].x), QFT_U(x[BASE + 0].y), QFT_U(x[BASE + 1].x), QFT_U(x[BASE + 1].y), QFT_U(x[BASE + 2].x),
        QFT_U(x[BASE + 2].y), QFT_U(x[BASE + 3].x), QFT_U(x[BASE + 3].y), QFT_U(x[BASE + 4].x), QFT_U(x[BASE + 4].y),
        QFT_U(x[BASE + 5].x), QFT_U(x[BASE + 5].y), QFT_U(x[BASE + 6].x), QFT_U(x[BASE + 6].y), QFT_U(x[BASE + 7].x),
        QFT_U(x[BASE + 7].y), QFT_U(x[BASE + 8].x), QFT_U(x[BASE + 8].y), QFT_U(x[BASE + 9].x), QFT_U(x[BASE + 9].y),
        QFT_U(x[BASE + 10].x), QFT_U(x[BASE + 10].y), QFT_U(x[BASE + 11].x), QFT_U(x[BASE + 11].y),
        QFT_U(x[BASE + 12].x), QFT_U(x[BASE + 12].y), QFT_U(x[BASE + 13].x), QFT_U(x[BASE + 13].y),
        QFT_U(x[BASE + 14].x), QFT_U(x[BASE + 14].y), QFT_U(x[BASE + 15].x), QFT_U(x[BASE + 15].y)
        : "memory");
}
#undef QFT_U
// fetch 8 parked amplitudes (16 words) from columns [taddr, taddr + 16)
__device__ __forceinline__ void tmem_fetch8(uint32_t taddr, float2 (&p)[8]) {
    uint32_t r[16];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, "
        "[%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr)
        : "memory");
    // the registers are operands of the wait so that no consumer can be scheduled above it
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]), "+r"(r[4]), "+r"(r[5]), "+r"(r[6]), "+r"(r[7]), "+r"(r[8]),
                   "+r"(r[9]), "+r"(r[10]), "+r"(r[11]), "+r"(r[12]), "+r"(r[13]), "+r"(r[14]), "+r"(r[15])
                 :
                 : "memory");
#pragma unroll
    for (int i = 0; i < 8; ++i) p[i] = make_float2(__uint_as_float(r[2 * i]), __uint_as_float(r[2 * i + 1]));
}

// Plain C++ accesses (not asm): the compiler knows they touch shared memory, keeps them on the right
// side of __syncthreads(), and is otherwise free to schedule them among the arithmetic.
__device__ __forceinline__ float2 lds64(const unsigned char* base, uint32_t off) {
    return *reinterpret_cast<const float2*>(base + off);
}
__device__ __forceinline__ void sts64(unsigned char* base, uint32_t off, float2 v) {
    *reinterpret_cast<float2*>(base + off) = v;
}

// XOR of the columns selected by the set bits of v
template <typename T, int N>
__device__ __forceinline__ T xor_cols(const T (&col)[N], uint32_t v, int nbits) {
    T r = 0;
    for (int j = 0; j < nbits; ++j)
        if ((v >> j) & 1u) r ^= col[j];
    return r;
}

// offset of register B: XOR of the register-bit columns (compile-time B, run-time columns)
template <int B>
__device__ __forceinline__ uint32_t reg_off(const uint32_t (&c)[5]) {
    uint32_t r = 0;
    if constexpr (B & 1) r ^= c[0];
    if constexpr (B & 2) r ^= c[1];
    if constexpr (B & 4) r ^= c[2];
    if constexpr (B & 8) r ^= c[3];
    if constexpr (B & 16) r ^= c[4];
    return r;
}

constexpr int kMidStride = QFT_TMA2_MID_STRIDE;
constexpr int kEndStride = QFT_TMA2_END_STRIDE;

// Multiply the 2^R amplitudes of batch BATCH by the subset products of W (optionally times p0).
template <int R, int BATCH, bool HASP>
__device__ __forceinline__ void apply_tree(float2 (&x)[32], const float2 (&W)[5], float2 p0) {
    qftp::TwTree<5, BATCH << R, R - 1, 0, HASP, 5>::run(x, W, p0);
}

template <int R, int BT, int NB, bool HASP>
struct BatchApply {
    static __device__ __forceinline__ void run(float2 (&x)[32], const float2 (&W)[NB][5], const float2 (&p)[NB]) {
        apply_tree<R, BT, HASP>(x, W[BT], p[BT]);
        if constexpr (BT + 1 < NB) BatchApply<R, BT + 1, NB, HASP>::run(x, W, p);
    }
};

// Profiling builds (-DQFT_PHASE_TIMING): thread 0 of CTA 0 accumulates the clocks between phase boundaries.
#ifdef QFT_PHASE_TIMING
#define QFT_PHASE(i)                                                       \
    if (d.dbg && blockIdx.x == 0 && tid == 0) {                            \
        const long long now_ = clock64();                                  \
        atomicAdd(d.dbg + (i), (unsigned long long)(now_ - tlast_));       \
        tlast_ = now_;                                                     \
    }
#else
#define QFT_PHASE(i)
#endif

// What a pass waits for before it first touches the state: the previous kernel of the stream (programmatic
// dependent launch).  (A functor so that another way of ordering passes can be plugged in: round 2 tried all three
// passes of an L2-resident state in one cooperative launch with grid-wide barriers here; it was slower than
// kernel boundaries with programmatic dependent launch, profiles/r02_small_n.md.)
struct SyncPrevKernel {
    __device__ __forceinline__ void operator()(uint32_t) const { asm volatile("griddepcontrol.wait;" ::: "memory"); }
};
// One pass over the units [d.unit_lo, d.unit_lo + d.unit_n) (the launcher fills the range in: all of them, or one rank's
// share).  The mbarrier behind the tile must have been initialised by the caller; parity carries its phase.
template <int R1, int R2, int KC, int LT, int XT, int ES, typename Sync>
__device__ __forceinline__ void tma2_pass(float2* __restrict__ state, const CUtensorMap* tmap_p, const QftPassDesc& d,
                                          unsigned char* smem_raw, uint32_t& parity, const Sync sync_before_state) {
    constexpr int F = LT + 5;
    constexpr int NT = 1 << LT;
    constexpr int NQ = R1 + R2 + XT;  // columns of the end table: the window's qubits, lowest first ... and the extension's
    float2* midW = reinterpret_cast<float2*>(smem_raw + ((size_t)8 << F));
    uint64_t* mbar = reinterpret_cast<uint64_t*>(midW + 32 * kMidStride);
    int* nextc = reinterpret_cast<int*>(mbar + 1);           // next tile's TMA coordinates (5 ints) + the TMEM base address
    float2* endW = reinterpret_cast<float2*>(nextc + 6);     // two end tables (by parity) of max(32, 2^eb) rows
    const uint32_t tid = threadIdx.x;
    const QftTma2Desc& t = d.tma;
    // split end table (ES = 1, more than QFT_TMA2_EB_DIRECT in-tile qubits below the window): the per-tile tables
    // cover the lowest QFT_TMA2_EB_LO of them, the constant table endHi the rest (the phase is linear over
    // disjoint bit sets, so a factor is the product of the two entries)
    const int eb_lo = ES ? QFT_TMA2_EB_LO : t.eb;
    const uint32_t end_rows = eb_lo > 5 ? (1u << eb_lo) : 32u;
    float2* endHi = endW + 2 * end_rows * kEndStride;
    const uint32_t hi_rows = ES ? (1u << (t.eb - QFT_TMA2_EB_LO)) : 0u;
    // tile-index byte -> address bits (tblA) and logical qubit bits (tblL): 256 entries per byte of the tile index
    const int nslice = (d.ntile + 7) >> 3;
    uint64_t* tblA = reinterpret_cast<uint64_t*>(endHi + hi_rows * kEndStride);
    uint64_t* tblL = tblA + nslice * 256;

    // ---- per-thread constants ----
    uint32_t off1_ld = xor_cols(t.s1_tid_ld, tid, LT);
    uint32_t off1_mid = xor_cols(t.s1_tid_mid, tid, LT);
    uint32_t off2_mid = xor_cols(t.s2_tid_mid, tid, LT);
    const uint32_t key2 = xor_cols(t.s2_tid_key, tid, LT);
    uint64_t st_thread = 0;
    for (int j = 0; j < LT; ++j)
        if ((tid >> j) & 1u) st_thread |= 1ull << t.s2_tid_addr[j];
    uint32_t c1ld[5], c1mid[5], c2mid[5];
    uint64_t c2st[5];
#pragma unroll
    for (int b = 0; b < 5; ++b) {
        c1ld[b] = t.s1_reg_ld[b];
        c1mid[b] = t.s1_reg_mid[b];
        c2mid[b] = t.s2_reg_mid[b];
        c2st[b] = 1ull << t.s2_reg_addr[b];
    }
    const int k = d.k;
    const int win_lo = d.win_lo;
    // this thread's entry of the per-tile end table (see the tile walk): row e, column q, target qubit, the bits
    // below it that may hold controls, and the phase its own row bits e contribute
    const uint32_t end_cnt = (uint32_t)NQ << eb_lo;
    const uint32_t end_e = tid / NQ, end_q = tid % NQ;
    const uint32_t end_slot = end_e * kEndStride + end_q;
    const int end_tq = (XT && end_q == (uint32_t)(R1 + R2)) ? win_lo - 1 : win_lo + (int)end_q;
    const uint64_t end_mask = (1ull << (end_tq < win_lo ? (end_tq > 0 ? end_tq : 0) : (win_lo > 0 ? win_lo : 0))) - 1ull;
    uint32_t end_ph_e;
    {
        uint64_t Le = 0;
        for (int b = 0; b < eb_lo; ++b)
            if ((end_e >> b) & 1u) Le |= 1ull << t.e_log[b];
        end_ph_e = qftp::cr_phase_u32(Le & end_mask, end_tq > 0 ? end_tq : 0, k);
    }

    uint32_t tpark = 0;  // this warp's parking columns in tensor memory
    constexpr uint32_t kTmemCols = (NT / 128) * 64;
    if constexpr (XT) {
        if (tid < 32) tmem_alloc(reinterpret_cast<uint32_t*>(nextc + 5), kTmemCols);
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    }
    // mid bases: midW[u1][b] = the phase that group 2's b-th qubit (when set) contributes to an amplitude
    // whose group-1 frequency bits are u1: the product over the set bits i of u1 of the controlled-R_m
    // from that qubit onto group 1's i-th qubit (phases add exactly as 32-bit fractions of a turn)
    for (uint32_t i = tid; i < 32u * R2; i += NT) {
        const uint32_t u1 = i / R2, b = i % R2;
        uint32_t ph = 0;
#pragma unroll
        for (int q = 0; q < R1; ++q)
            if ((u1 >> q) & 1u) ph += qftp::cr_phase_u32(1ull << (t.t2_lo + (int)b), t.t1_lo + q, k);
        midW[u1 * kMidStride + b] = qftp::cis_fwd_u32(ph);
    }
    if constexpr (ES) {
        // the constant half of the split end table: rows = values of the in-tile qubits e_log[EB_LO ...]
        for (uint32_t i = tid; i < (uint32_t)NQ * hi_rows; i += NT) {
            const uint32_t e = i / NQ, q = i % NQ;
            uint64_t L = 0;
            for (int b = QFT_TMA2_EB_LO; b < t.eb; ++b)
                if ((e >> (b - QFT_TMA2_EB_LO)) & 1u) L |= 1ull << t.e_log[b];
            endHi[e * kEndStride + q] = qftp::cis_fwd_u32(qftp::cr_phase_u32(L, win_lo + (int)q, k));
        }
    }
    for (int i = (int)tid; i < nslice * 256; i += NT) {
        uint64_t a = 0, L = 0;
        for (int b = 0; b < 8; ++b) {
            const int bit = (i >> 8) * 8 + b;
            if (bit < d.ntile && ((i >> b) & 1)) {
                a |= 1ull << d.tile_addr[bit];
                L |= 1ull << d.log_tile[bit];
            }
        }
        tblA[i] = a;
        tblL[i] = L;
    }
    __syncthreads();
    if constexpr (XT) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        const uint32_t warp = tid >> 5;
        tpark = *reinterpret_cast<volatile uint32_t*>(nextc + 5) + (((warp & 3u) * 32u) << 16) + (warp >> 2) * 64u;
    }

    // ---- tile walk ----
    const uint32_t csz = d.npair ? 2u : 1u;
    const uint32_t rho = d.npair ? (blockIdx.x & 1u) : 0u;
    const int nbig = d.ntile - XT;  // index bits of the tiles a CTA owns (an extended tile = two half-tiles)
    const uint32_t nunits = (uint32_t)(d.unit_lo + d.unit_n);  // one past the last unit (the launcher fills the range in)
    const uint32_t ustride = gridDim.x / csz;
    const bool has_end = win_lo > 0;

    // tile index (+ half) -> HBM base address / logical bits, one table lookup per index byte
    auto lut = [&](const uint64_t* T, uint32_t m) {
        uint64_t r = T[m & 255u];
        if (nslice > 1) r |= T[256 + ((m >> 8) & 255u)];
        if (nslice > 2) r |= T[512 + ((m >> 16) & 255u)];
        if (nslice > 3) r |= T[768 + (m >> 24)];
        return r;
    };
    // lanes 0-4 of warp 0 each own one TMA coordinate: the tile's address bits cut into the tensor map's dims
    const int cj = tid < 5u ? (int)tid : 0;
    const int c_lo = t.tma_lo[cj];
    const uint64_t c_mask = (1ull << t.tma_len[cj]) - 1ull;
    auto put_coords = [&](uint32_t un, uint32_t half) {
        uint32_t ml, ms;
        decode_tile(un * csz + rho, d.npair, &ml, &ms);
        nextc[tid] = (int)((lut(tblA, ml | (half << nbig)) >> c_lo) & c_mask);
    };

    // End bases of a half-tile, written into the end table of parity `par`: endW[e][q] = product of the controlled-R_m
    // from every qubit below the window (tile-index bits + in-tile bits e) onto the window's q-th qubit (with an
    // extended tile the last column belongs to the extension's qubit win_lo - 1).  The phase is linear over disjoint
    // bit sets, so a thread's entry is its constant part from e plus the tile's part.  Filled one half-tile ahead (in
    // the shadow of the previous half-tile's step 2), never on the path between two tiles.
    auto fill_end = [&](uint32_t un, uint32_t half, uint32_t par) {
        if (!has_end) return;
        uint32_t ml, ms;
        decode_tile(un * csz + rho, d.npair, &ml, &ms);
        const uint64_t Ltile = lut(tblL, ml | (half << nbig));
        float2* tab = endW + par * (end_rows * kEndStride);
        if (tid < end_cnt) tab[end_slot] = qftp::cis_fwd_u32(end_ph_e + qftp::cr_phase_u32(Ltile & end_mask, end_tq, k));
        for (uint32_t i = tid + NT; i < end_cnt; i += NT) {  // only when 2^eb (R1 + R2 + XT) > threads
            const uint32_t e = i / NQ, q = i % NQ;
            uint64_t L = Ltile;
            for (int b = 0; b < eb_lo; ++b)
                if ((e >> b) & 1u) L |= 1ull << t.e_log[b];
            int tq = win_lo + (int)q;
            if (XT && q == (uint32_t)(R1 + R2)) tq = win_lo - 1;
            L &= (1ull << (tq < win_lo ? tq : win_lo)) - 1ull;
            tab[e * kEndStride + q] = qftp::cis_fwd_u32(qftp::cr_phase_u32(L, tq, k));
        }
    };

    // everything above is independent of the state; the previous pass must have completed (and its
    // writes be visible) before the first load
    sync_before_state(tid);
    uint32_t unit = (uint32_t)d.unit_lo + blockIdx.x / csz;
    if (unit < nunits) fill_end(unit, 0u, parity);
    if (unit < nunits && tid < 32u) {
        if (tid < 5u) put_coords(unit, 0u);
        __syncwarp();
        if (tid == 0) {
            mbar_expect_tx(mbar, 8u << F);
            tma_load_5d(smem_raw, tmap_p, mbar, nextc[0], nextc[1], nextc[2], nextc[3], nextc[4]);
        }
        __syncwarp();
    }
#ifdef QFT_PHASE_TIMING
    long long tlast_ = clock64();
#endif
    for (; unit < nunits; unit += ustride) {
#pragma unroll 1
        for (uint32_t half = 0; half <= (uint32_t)XT; ++half) {
        // ---- bookkeeping while the tile's load is in flight (few registers live here) ----
        const bool last_half = half == (uint32_t)XT;
        const bool has_next = !last_half || unit + ustride < nunits;
        const uint32_t next_unit = last_half ? unit + ustride : unit, next_half = last_half ? 0u : half + 1u;
        uint64_t base_st;
        float2* endWp = endW + parity * (end_rows * kEndStride);  // filled while the previous half-tile was in step 2
        {
            uint32_t ml, ms;
            decode_tile(unit * csz + rho, d.npair, &ml, &ms);
            base_st = lut(tblA, ms);
        }
        float2 x[32];
        // keep the 96 per-register shared-memory offsets out of loop-invariant hoisting (they would
        // spill): one XOR next to each access is cheaper than a local-memory reload
        asm volatile("" : "+r"(off1_ld), "+r"(off1_mid), "+r"(off2_mid));
        QFT_PHASE(0)
        mbar_wait(mbar, parity);
        QFT_PHASE(1)
        // this CTA's whole tile is on chip (or in registers / tensor memory): the partner may overwrite it in HBM
        if (d.npair && last_half) cluster_arrive_relaxed();

        // ------------------------------ step 1 ------------------------------
#define QFT_LD1(B) x[B] = lds64(smem_raw, off1_ld ^ reg_off<B>(c1ld));
#define QFT_ALL32(M)                                                                                          \
    M(0) M(1) M(2) M(3) M(4) M(5) M(6) M(7) M(8) M(9) M(10) M(11) M(12) M(13) M(14) M(15) M(16) M(17) M(18)  \
        M(19) M(20) M(21) M(22) M(23) M(24) M(25) M(26) M(27) M(28) M(29) M(30) M(31)
        QFT_ALL32(QFT_LD1)
#undef QFT_LD1
        __syncthreads();  // every amplitude of the tile is in a register: the buffer becomes the exchange
        if (tid < 5u && has_next) put_coords(next_unit, next_half);  // (read by thread 0 two barriers further down)
        QFT_PHASE(2)
        if (d.conj) {
#pragma unroll
            for (int B = 0; B < 32; ++B) x[B].y = -x[B].y;
        }
        qftp::dif_group<5, R1, KC>(x);
#define QFT_ST1(B) sts64(smem_raw, off1_mid ^ reg_off<B>(c1mid), x[B]);
        QFT_ALL32(QFT_ST1)
#undef QFT_ST1
        __syncthreads();
        QFT_PHASE(3)

        // ------------------------------ step 2 ------------------------------
        // (the next half-tile's end table first: its short arithmetic chain runs under the latency of the reads below)
        if (has_next) fill_end(next_unit, next_half, parity ^ 1u);
#define QFT_LD2(B) x[B] = lds64(smem_raw, off2_mid ^ reg_off<B>(c2mid));
        QFT_ALL32(QFT_LD2)
#undef QFT_LD2
        fence_proxy_async();
        __syncthreads();  // the buffer is free again
        if (tid == 0 && has_next) {
            // prefetch the next tile while this one is transformed and stored
            mbar_expect_tx(mbar, 8u << F);
            tma_load_5d(smem_raw, tmap_p, mbar, nextc[0], nextc[1], nextc[2], nextc[3], nextc[4]);
        }
        QFT_PHASE(4)

        {
            // the phases group 2's qubits put on group 1's frequency bits, applied here, after
            // the exchange, so that the next tile's load is issued before this arithmetic rather than after
            constexpr int NBM = 1 << (5 - R2);
            float2 WM[NBM][5];
            float2 one[NBM];
#pragma unroll
            for (int bt = 0; bt < NBM; ++bt) {
                uint32_t kk = key2;
#pragma unroll
                for (int i = 0; i < 5 - R2; ++i)
                    if (bt & (1 << i)) kk ^= t.s2_reg_key[R2 + i];
                const float2* row = midW + (kk & 31u) * kMidStride;
#pragma unroll
                for (int i = 0; i < R2; ++i) WM[bt][i] = row[i];
                one[bt] = make_float2(1.f, 0.f);
            }
            BatchApply<R2, 0, NBM, false>::run(x, WM, one);
        }
        qftp::dif_group<5, R2, KC>(x);
        constexpr int NB2 = 1 << (5 - R2);
        if (has_end) {
            float2 W2[NB2][5];
            float2 cfac[NB2];
#pragma unroll
            for (int bt = 0; bt < NB2; ++bt) {
                uint32_t kk = key2;
#pragma unroll
                for (int i = 0; i < 5 - R2; ++i)
                    if (bt & (1 << i)) kk ^= t.s2_reg_key[R2 + i];
                const float2* row = endWp + ((kk >> 8) & (ES ? 63u : 127u)) * kEndStride;
                const float2* rowh = endHi + ((kk >> (8 + QFT_TMA2_EB_LO)) & 63u) * kEndStride;  // ES only
#pragma unroll
                for (int i = 0; i < R2; ++i) W2[bt][i] = ES ? qftp::cmul(row[i], rowh[i]) : row[i];
                float2 c = make_float2(d.scale, 0.f);
#pragma unroll
                for (int i = 0; i < R1; ++i) {
                    const float2 w = ES ? qftp::cmul(row[R2 + i], rowh[R2 + i]) : row[R2 + i];
                    const float2 cw = qftp::cmul(c, w);
                    if ((kk >> i) & 1u) c = cw;
                }
                cfac[bt] = c;
            }
            BatchApply<R2, 0, NB2, true>::run(x, W2, cfac);
        } else if (d.do_scale) {
#pragma unroll
            for (int B = 0; B < 32; ++B) x[B] = qftp::cscale(x[B], d.scale);
        }
        QFT_PHASE(5)
        if constexpr (XT) {
            if (!last_half) {
                // first half: park the results in tensor memory until the second half has caught up
                tmem_park16<0>(tpark, x);
                tmem_park16<16>(tpark + 32u, x);
                asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
                parity ^= 1u;
                QFT_PHASE(6)
                continue;
            }
        }
        float2* __restrict__ dst = state + (base_st | st_thread);
        if constexpr (XT) {
            // H on the extension's qubit: butterfly between the parked half (bit = 0) and this one (bit = 1), then
            // the controlled-R_m onto it from the qubits below the window; the frequency
            // bit lands on address bit xt_st_addr
            float2 wg[NB2];
#pragma unroll
            for (int bt = 0; bt < NB2; ++bt) {
                uint32_t kk = key2;
#pragma unroll
                for (int i = 0; i < 5 - R2; ++i)
                    if (bt & (1 << i)) kk ^= t.s2_reg_key[R2 + i];
                wg[bt] = endWp[((kk >> 8) & 127u) * kEndStride + (R1 + R2)];
            }
            if (d.npair) cluster_wait();  // the partner holds its tile on chip: its addresses may be overwritten
            float2* __restrict__ dst1 = dst + (1ull << d.xt_st_addr);
#pragma unroll
            for (int c8 = 0; c8 < 4; ++c8) {
                float2 pk[8];
                tmem_fetch8(tpark + 16u * c8, pk);
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const int B = 8 * c8 + i;
                    float2 lo = qftp::padd(pk[i], x[B]);
                    float2 hi = qftp::cmul(qftp::psub(pk[i], x[B]), wg[B >> R2]);
                    if (d.conj) { lo.y = -lo.y; hi.y = -hi.y; }
                    uint64_t o = 0;
#pragma unroll
                    for (int b = 0; b < 5; ++b)
                        if (B & (1 << b)) o += c2st[b];
                    dst[o] = lo;
                    dst1[o] = hi;
                }
            }
        } else {
            if (d.conj) {
#pragma unroll
                for (int B = 0; B < 32; ++B) x[B].y = -x[B].y;
            }
            if (d.npair) cluster_wait();  // the partner holds its tile on chip: its addresses may be overwritten
#pragma unroll
            for (int B = 0; B < 32; ++B) {
                uint64_t o = 0;
#pragma unroll
                for (int b = 0; b < 5; ++b)
                    if (B & (1 << b)) o += c2st[b];
                dst[o] = x[B];
            }
        }
        parity ^= 1u;
        QFT_PHASE(7)
#ifdef QFT_PHASE_TIMING
        if (d.dbg && blockIdx.x == 0 && tid == 0) atomicAdd(d.dbg + 8, 1ull);
#endif
        }
    }
#undef QFT_ALL32
    if constexpr (XT) {
        // every thread's tensor-memory traffic has completed (wait::ld / wait::st above): give the columns back
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        if (tid < 32) tmem_dealloc(*reinterpret_cast<volatile uint32_t*>(nextc + 5), kTmemCols);
    }
}

template <int LT>
__device__ __forceinline__ uint64_t* tma2_mbar(unsigned char* smem_raw) {
    return reinterpret_cast<uint64_t*>(smem_raw + ((size_t)8 << (LT + 5)) + 32 * kMidStride * sizeof(float2));
}

// One pass per launch (the default for every n whose passes are bound by HBM).
template <int R1, int R2, int KC, int LT, int XT, int ES = 0>
__global__ void __launch_bounds__(1 << LT, (LT == 8) ? 2 : ((LT == 7) ? 4 : 1))
    qft_pass_tma2(float2* __restrict__ state, const __grid_constant__ CUtensorMap tmap,
                  const __grid_constant__ QftPassDesc d) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    // let the next pass's CTAs be scheduled as soon as SM resources free up (they wait inside tma2_pass)
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if (threadIdx.x == 0) {
        mbar_init(tma2_mbar<LT>(smem_raw), 1);
        fence_proxy_async();
    }
    uint32_t parity = 0;
    tma2_pass<R1, R2, KC, LT, XT, ES>(state, &tmap, d, smem_raw, parity, SyncPrevKernel{});
}

}  // namespace qftk
