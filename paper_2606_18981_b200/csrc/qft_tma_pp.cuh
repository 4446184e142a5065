// qft_tma_pp.cuh -- the ping-pong variant of the TMA-staged pass kernel (QFT_KERNEL_TMA2PP), sm_100a.
//
// A 2^14-amplitude tile (16-amplitude = 128-byte hub granules x a 10-qubit window) fills 128 KB of
// shared memory, so only one CTA fits per SM and the plain tma2 kernel runs its phases back to back:
// the FP32 pipe idles while the tile moves through shared memory and HBM idles while it computes.
// Here the CTA's 512 threads are two groups of 256.  The tile splits along its top hub bit into two
// independent halves (the window's gates never touch a hub qubit), one per group, and the groups
// run the same two-step pass skewed against each other:
//   * one TMA load per tile (whole 128-byte granules) into a 128B-swizzled landing buffer; it is
//     re-issued for tile i+1 as soon as BOTH groups hold tile i in registers, i.e. before any
//     arithmetic of tile i, so the load is in flight during the whole transform;
//   * ONE 64 KB exchange buffer that the groups take turns on (named barriers hand it over): while
//     group A moves its half through shared memory between step 1 and step 2, group B is in its
//     butterflies, and vice versa, so the FP32 pipe and the shared-memory pipe overlap;
//   * stores straight from registers; lanes run along hub bits 0-2 (64-byte segments; the other half
//     of each 128-byte line is written by the sibling group, L2 merges them).
// Arithmetic, phase tables and descriptor are those of qft_tma.cuh (thread bit 8 = the group bit).
#pragma once
#include "qft_tma.cuh"

namespace qftk {

__device__ __forceinline__ void named_bar_sync(int id, int count) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory");
}
__device__ __forceinline__ void named_bar_arrive(int id, int count) {
    asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(count) : "memory");
}

constexpr int kPPLanding = 8 << 14;  // bytes
constexpr int kPPExchange = 8 << 13;

template <int R1, int R2, int KC>
__global__ void __launch_bounds__(512, 1)
    qft_pass_tma2pp(float2* __restrict__ state, const __grid_constant__ CUtensorMap tmap,
                    const __grid_constant__ QftPassDesc d) {
    extern __shared__ unsigned char smem_dyn[];
    // the 128B swizzle is a function of absolute shared-memory address bits 4-9: align to 1024
    unsigned char* smem_raw = smem_dyn + ((1024u - (smem_u32(smem_dyn) & 1023u)) & 1023u);
    unsigned char* xbuf = smem_raw + kPPLanding;
    float2* midW = reinterpret_cast<float2*>(xbuf + kPPExchange);
    float2* endW = midW + 32 * kMidStride;  // [group][parity][32 rows]
    uint64_t* mbar = reinterpret_cast<uint64_t*>(endW + 4 * 32 * kEndStride);
    int* nextc = reinterpret_cast<int*>(mbar + 1);  // [group][5] (+ pad)
    unsigned int* counter = reinterpret_cast<unsigned int*>(nextc + 12);
    constexpr int LT = 9;
    constexpr int NT = 512;
    constexpr int F = 14;
    const uint32_t tid = threadIdx.x;
    const uint32_t grp = tid >> 8;
    const uint32_t gtid = tid & 255u;
    const QftTma2Desc& t = d.tma;
    enum { BAR_GRP = 1, BAR_XFREE = 3 };  // ids 1,2: group barriers; 3,4: "exchange buffer free for group 0 / 1"

    // ---- per-thread constants ----
    uint32_t off1_ld = xor_cols(t.s1_tid_ld, tid, LT);
    uint32_t off1_mid = xor_cols(t.s1_tid_mid, tid, LT);
    uint32_t off2_mid = xor_cols(t.s2_tid_mid, tid, LT);
    const uint32_t key1 = xor_cols(t.s1_tid_key, tid, LT);
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
    const uint64_t lbmask = (win_lo > 0) ? ((1ull << win_lo) - 1ull) : 0ull;

    if (tid == 0) {
        mbar_init(mbar, 1);
        *counter = 0;
        fence_proxy_async();
    }
    for (uint32_t i = tid; i < 32u * R1; i += NT) {
        const uint32_t v = i / R1, q = i % R1;
        midW[v * kMidStride + q] = qftp::cis_fwd_u32(qftp::cr_phase_u32((uint64_t)v << t.t2_lo, t.t1_lo + (int)q, k));
    }
    __syncthreads();

    // ---- tile walk ----
    const uint32_t csz = d.npair ? 2u : 1u;
    const uint32_t rho = d.npair ? (blockIdx.x & 1u) : 0u;
    const uint32_t nunits = (1u << d.ntile) / csz;
    const uint32_t ustride = gridDim.x / csz;
    const bool has_end = win_lo > 0;

    auto coords_of = [&](uint32_t un, int (&c)[5]) {
        uint32_t ml, ms;
        decode_tile(un * csz + rho, d.npair, &ml, &ms);
        uint64_t base = 0;
        for (int i = 0; i < d.ntile; ++i)
            if ((ml >> i) & 1u) base |= 1ull << d.tile_addr[i];
#pragma unroll
        for (int j = 0; j < 5; ++j) c[j] = (int)((base >> t.tma_lo[j]) & ((1ull << t.tma_len[j]) - 1ull));
    };

    uint32_t unit = blockIdx.x / csz;
    if (unit < nunits && tid == 0) {
        int c[5];
        coords_of(unit, c);
        mbar_expect_tx(mbar, 8u << F);
        tma_load_5d(smem_raw, &tmap, mbar, c[0], c[1], c[2], c[3], c[4]);
    }
    // the exchange buffer starts out free for group 0: group 1 pre-arrives on group 0's barrier
    if (grp == 1 && unit < nunits) named_bar_arrive(BAR_XFREE + 0, NT);
    uint32_t parity = 0;
    for (; unit < nunits; unit += ustride) {
        const bool has_next = unit + ustride < nunits;
        // ---- bookkeeping while the tile's load is in flight (few registers live here) ----
        uint64_t base_st = 0;
        float2* endWp = endW + (grp * 2 + parity) * (32 * kEndStride);
        {
            uint32_t ml, ms;
            decode_tile(unit * csz + rho, d.npair, &ml, &ms);
            uint64_t Ltile = 0;
            for (int i = 0; i < d.ntile; ++i) {
                if ((ml >> i) & 1u) Ltile |= 1ull << d.log_tile[i];
                if ((ms >> i) & 1u) base_st |= 1ull << d.tile_addr[i];
            }
            if (has_end) {
                const uint32_t nq = R1 + R2;
                const uint32_t cnt = nq << t.eb;
                for (uint32_t i = gtid; i < cnt; i += 256) {
                    const uint32_t e = i / nq, q = i % nq;
                    uint64_t L = Ltile;
                    for (int b = 0; b < t.eb; ++b)
                        if ((e >> b) & 1u) L |= 1ull << t.e_log[b];
                    L &= lbmask;
                    endWp[e * kEndStride + q] = qftp::cis_fwd_u32(qftp::cr_phase_u32(L, win_lo + (int)q, k));
                }
            }
            if (gtid == 0 && has_next) {
                int c[5];
                coords_of(unit + ustride, c);
#pragma unroll
                for (int j = 0; j < 5; ++j) nextc[grp * 6 + j] = c[j];
            }
        }
        float2 x[32];
        asm volatile("" : "+r"(off1_ld), "+r"(off1_mid), "+r"(off2_mid));
        mbar_wait(mbar, parity);
        if (d.npair) cluster_arrive_relaxed();

        // ------------------------------ step 1 ------------------------------
#define QFT_LD1(B) x[B] = lds64(smem_raw, off1_ld ^ reg_off<B>(c1ld));
#define QFT_ALL32(M)                                                                                          \
    M(0) M(1) M(2) M(3) M(4) M(5) M(6) M(7) M(8) M(9) M(10) M(11) M(12) M(13) M(14) M(15) M(16) M(17) M(18)  \
        M(19) M(20) M(21) M(22) M(23) M(24) M(25) M(26) M(27) M(28) M(29) M(30) M(31)
        QFT_ALL32(QFT_LD1)
#undef QFT_LD1
        fence_proxy_async();
        named_bar_sync(BAR_GRP + grp, 256);  // this group's half of the tile is in registers
        if (gtid == 0) {
            // the second group to get here re-arms the landing buffer with the next tile
            __threadfence_block();
            const unsigned int old = atomicAdd(counter, 1u);
            if ((old & 1u) && has_next) {
                mbar_expect_tx(mbar, 8u << F);
                const int* c = nextc + grp * 6;
                tma_load_5d(smem_raw, &tmap, mbar, c[0], c[1], c[2], c[3], c[4]);
            }
        }
        if (d.conj) {
#pragma unroll
            for (int B = 0; B < 32; ++B) x[B].y = -x[B].y;
        }
        qftp::dif_group<5, R1, KC>(x);
        {
            constexpr int NB1 = 1 << (5 - R1);
            float2 W1[NB1][5];
            float2 one[NB1];
#pragma unroll
            for (int bt = 0; bt < NB1; ++bt) {
                uint32_t kk = key1;
#pragma unroll
                for (int i = 0; i < 5 - R1; ++i)
                    if (bt & (1 << i)) kk ^= t.s1_reg_key[R1 + i];
                const float2* row = midW + (kk & 31u) * kMidStride;
#pragma unroll
                for (int i = 0; i < R1; ++i) W1[bt][i] = row[i];
                one[bt] = make_float2(1.f, 0.f);
            }
            BatchApply<R1, 0, NB1, false>::run(x, W1, one);
        }
        // ---- exchange: this group's turn on the shared buffer ----
        named_bar_sync(BAR_XFREE + grp, NT);  // the other group has read its half back
#define QFT_ST1(B) sts64(xbuf, off1_mid ^ reg_off<B>(c1mid), x[B]);
        QFT_ALL32(QFT_ST1)
#undef QFT_ST1
        named_bar_sync(BAR_GRP + grp, 256);
#define QFT_LD2(B) x[B] = lds64(xbuf, off2_mid ^ reg_off<B>(c2mid));
        QFT_ALL32(QFT_LD2)
#undef QFT_LD2
        // hand the buffer to the other group (its next wait must have a matching arrive: group 1's
        // arrive after the last tile would have no taker)
        if (grp == 0 || has_next) named_bar_arrive(BAR_XFREE + (grp ^ 1), NT);

        // ------------------------------ step 2 ------------------------------
        qftp::dif_group<5, R2, KC>(x);
        if (has_end) {
            constexpr int NB2 = 1 << (5 - R2);
            float2 W2[NB2][5];
            float2 cfac[NB2];
#pragma unroll
            for (int bt = 0; bt < NB2; ++bt) {
                uint32_t kk = key2;
#pragma unroll
                for (int i = 0; i < 5 - R2; ++i)
                    if (bt & (1 << i)) kk ^= t.s2_reg_key[R2 + i];
                const float2* row = endWp + ((kk >> 8) & 31u) * kEndStride;
#pragma unroll
                for (int i = 0; i < R2; ++i) W2[bt][i] = row[i];
                float2 c = make_float2(d.scale, 0.f);
#pragma unroll
                for (int i = 0; i < R1; ++i) {
                    const float2 w = row[R2 + i];
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
        if (d.conj) {
#pragma unroll
            for (int B = 0; B < 32; ++B) x[B].y = -x[B].y;
        }
        if (d.npair) cluster_wait();
        float2* __restrict__ dst = state + (base_st | st_thread);
#pragma unroll
        for (int B = 0; B < 32; ++B) {
            uint64_t o = 0;
#pragma unroll
            for (int b = 0; b < 5; ++b)
                if (B & (1 << b)) o += c2st[b];
            dst[o] = x[B];
        }
        parity ^= 1u;
    }
#undef QFT_ALL32
}

}  // namespace qftk
