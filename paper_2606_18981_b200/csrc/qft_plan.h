// qft_plan.h -- pass descriptors shared by the host planner and the kernels.
//
// Vocabulary (DESIGN.md has the full story):
//   address bit a   : bit a of the array index of an amplitude in HBM.
//   logical qubit q : the circuit's wire q_q; pos[q] is the address
//                     bit that currently holds it.  Initially pos[q] = q; after
//                     the last pass pos[q] = n-1-q (the bit reversal).
//   tile            : all addresses that agree outside a set F of f address bits.
//                     F always contains the hub [0, l) so that every global access
//                     moves whole 2^l * 8-byte granules.
//   canonical bit c : position inside the tile's shared-memory image; canonical
//                     bits are ordered by the logical qubit they hold, so a window
//                     of consecutive logical qubits is a run of canonical bits.
//   window          : the logical qubits whose gates (H and every controlled-R_m
//                     that targets them) this pass applies.
//   step            : a group of <= 5 window qubits transformed in registers
//                     (radix-2^r butterfly) between shared-memory exchanges.
#pragma once
#include <stdint.h>

#define QFT_MAX_TILE_BITS 14
#define QFT_MAX_TILEIDX_BITS 34
#define QFT_MAX_STEPS 14
#define QFT_MAX_RADIX_BITS 5
// QFT_KERNEL_TMA2 shared-memory tables after the tile: 32 rows of mid bases, two per-tile end tables (by parity)
// of 2^eb rows (at least 32), one mbarrier, 5 coords + the tensor-memory base address, the tile-index byte tables.
// More than QFT_TMA2_EB_DIRECT in-tile qubits below the window ("split end table", small windows high up in a large
// tile): the per-tile tables cover the lowest QFT_TMA2_EB_LO of them and one table that is constant for the whole
// launch covers the rest; the kernel multiplies the two factors.
#define QFT_TMA2_MID_STRIDE 9   // float2 per row (<= 5 used; odd: rows of different lanes fall into different banks)
#define QFT_TMA2_END_STRIDE 17  // float2 per row (R1 + R2 + 1 <= 11 used; odd for the same reason)
#define QFT_TMA2_EB_DIRECT 7
#define QFT_TMA2_EB_LO 6
#define QFT_TMA2_EB_MAX 12
#define QFT_TMA2_END_ROWS(eb) \
    ((eb) > QFT_TMA2_EB_DIRECT ? 2 * (1 << QFT_TMA2_EB_LO) + (1 << ((eb)-QFT_TMA2_EB_LO)) : 2 * ((eb) > 5 ? (1 << (eb)) : 32))
#define QFT_TMA2_TABLE_BYTES(eb, ntile) \
    ((32 * QFT_TMA2_MID_STRIDE + QFT_TMA2_END_ROWS(eb) * QFT_TMA2_END_STRIDE) * 8 + 8 + 24 + (((ntile) + 7) >> 3) * 256 * 16)

struct QftStep {
    int8_t r;     // qubits in the group
    int8_t a;     // lowest canonical bit of the group: canonical bits [a, a+r)
    int8_t t_hi;  // logical qubit on canonical bit a+r-1 (the first one processed)
    int8_t pad;
};

enum QftKernelKind : int32_t {
    QFT_KERNEL_GENERIC = 0,  // shared-memory staged tile pass, any descriptor
    QFT_KERNEL_FUSED2 = 1,   // two register steps: global -> reg -> smem -> reg -> global
    QFT_KERNEL_TMA2 = 2,     // persistent: TMA tile load -> reg -> smem -> reg -> global, packed FP32x2
};

// QFT_KERNEL_TMA2 only.  Every shared-memory byte offset is a GF(2)-linear function of the thread
// index and the register index, given column by column; "thread bit j" is bit j of threadIdx.x,
// "register bit b" is bit b of the index into the thread's 32 amplitudes.  Register bits [0, r) of a
// step are its group's qubits (ascending), the rest are batch bits.
struct QftTma2Desc {
    uint32_t s1_tid_ld[9], s1_reg_ld[5];    // step 1 read: the TMA landing layout (tile load order)
    uint32_t s1_tid_mid[9], s1_reg_mid[5];  // step 1 write: the swizzled exchange layout
    uint32_t s2_tid_mid[9], s2_reg_mid[5];  // step 2 read: the same layout seen from step 2's threads
    uint32_t s1_tid_key[9], s1_reg_key[5];  // step 1 key: bits 0-4 = value of group 2's qubits, 8-19 = e
    uint32_t s2_tid_key[9], s2_reg_key[5];  // step 2 key: bits 0-4 = value of group 1's qubits, 8-19 = e
    int8_t s2_tid_addr[9], s2_reg_addr[5];  // step 2 store: HBM address bit of each thread / register bit
    int8_t eb;                              // in-tile logical qubits below the window (<= 12); e indexes them
    int8_t e_log[QFT_TMA2_EB_MAX];          // their logical ids, ascending
    int8_t t1_lo, t2_lo;                    // lowest logical qubit of group 1 / group 2
    int8_t r1, r2;
    int8_t tma_lo[5], tma_len[5], tma_box[5];  // tensor-map dims: address bits [lo, lo+len), box 2^box
    int8_t land_addr[16];                      // landing-index bit j of the shared-memory tile <-> address bit
};

// Plain data, passed to the kernels by value (__grid_constant__).
struct QftPassDesc {
    int32_t n;          // qubits
    int32_t f;          // tile bits
    int32_t ntile;      // n - f
    int32_t npair;      // p: tile-index bits [0,p) trade places with bits [p,2p) on store
    int32_t nsteps;
    int32_t k;          // AQFT cutoff (clamped to n)
    int32_t conj;       // sign = +1: conjugate on load and on store
    int32_t kernel;     // QftKernelKind
    int32_t log2_threads;
    float scale;        // applied in the last step (1 unless this is the final pass)
    int32_t do_scale;
    int32_t win_lo;     // lowest logical qubit the register steps process (-1: permutation-only pass)
    // the units (tiles, or pairs of tiles of a pair pass) this launch walks: [unit_lo, unit_lo + unit_n); unit_n = 0:
    // all of them.  Set per launch by qft_execute_pass_shard (one rank's share of a pass), 0 in the plan.
    int32_t unit_lo, unit_n;
    // ---- tensor-memory extended tile (QFT_KERNEL_TMA2 only) ------------------------------------
    // xt = 1: the pass owns tiles of 2^(f+1) amplitudes, F + {xt_ld_addr}.  A CTA runs the two halves
    // (address bit xt_ld_addr = 0, then 1) through the register steps one after the other, parks the
    // first half's results in tensor memory, and then applies the gates of one more qubit, xt_q =
    // win_lo - 1 (H as a radix-2 butterfly between the halves and the controlled-R_m onto it from below),
    // before it stores both halves; the butterfly's frequency bit lands on address bit xt_st_addr.
    // The half-tile index bit is the LAST tile-index bit: tile_addr[ntile-1] = xt_ld_addr.
    int32_t xt;
    int8_t xt_q, xt_ld_addr, xt_st_addr, xt_pad;
    int8_t F[16];         // load-order bit j <-> address bit F[j], ascending, F[j] = j for j < l
    int8_t Fst[16];       // store-order bit j <-> address bit Fst[j], ascending (= F unless xt)
    int8_t ld_canon[16];  // load-order bit j  -> canonical bit
    int8_t st_canon[16];  // store-order bit j -> canonical bit whose data lands on address Fst[j]
    int8_t log_canon[16]; // canonical bit -> logical qubit
    int8_t tile_addr[QFT_MAX_TILEIDX_BITS];  // tile-index bit -> address bit
    int8_t log_tile[QFT_MAX_TILEIDX_BITS];   // tile-index bit -> logical qubit held at load time
    QftStep steps[QFT_MAX_STEPS];
    // ---- QFT_KERNEL_FUSED2 only -------------------------------------------------------------
    // Step 1 reads its 2^r1 amplitudes straight from HBM, step 2 writes its 2^r2 straight back.
    // t?_addr / t?_canon: for every bit of the thread's "other" index (load order for step 1, store
    // order for step 2, the step's own bits left out) the address bit and the canonical bit.
    // r?_addr: address bit of the step's b-th register bit (canonical bit a + b).
    // swz_col[c]: 4-bit XOR mask that canonical bit c contributes to the low 4 bits of the
    // shared-memory index (a GF(2)-linear, conflict-free swizzle chosen by the planner).
    int8_t t1_addr[16], t1_canon[16], r1_addr[QFT_MAX_RADIX_BITS + 3];
    int8_t t2_addr[16], t2_canon[16], r2_addr[QFT_MAX_RADIX_BITS + 3];
    uint8_t swz_col[16];
    QftTma2Desc tma;
#ifdef QFT_PHASE_TIMING
    unsigned long long* dbg;  // profiling builds only: 16 counters, clocks per phase of CTA 0 (qft_tma.cuh)
#endif
};

#include <string>
#include <vector>

struct QftPlanParams {
    int n = 0;
    int batch_bits = 0;  // log2 of the number of independent states stored back to back
    int k = 0;
    int max_fused = 0;
    int sign = -1;
    int norm = 0;
    int tile_bits = 0;  // 0 = default
    int hub_bits = 0;   // 0 = default
    unsigned flags = 0;
};

struct QftHostPlan {
    QftPlanParams prm;
    int k_eff = 0;  // min(k, n)
    int tile_bits = 0, hub_bits = 0, window = 0;
    bool folded = false;
    bool ext_tile = false;  // some passes use the tensor-memory extended tile
    std::vector<QftPassDesc> passes;
    std::vector<int> out_qubit_at;  // after the last pass address bit a holds logical qubit out_qubit_at[a]
    long long n_h = 0, n_cr = 0, n_swap = 0;
};

// Returns 0 (ok), 1 (invalid argument), 2 (unsupported tuning), 5 (internal: self-check failed).
int qft_build_plan(const QftPlanParams& prm, QftHostPlan* out, std::string* err);
int qft_check_plan(const QftHostPlan& plan, std::string* err);
std::string qft_describe_plan(const QftHostPlan& plan);

// sharded state, host side (qft_plan.cpp): rank r's unit range of a pass, and the proof that the ranges tile the pass
int qft_shard_range(const QftHostPlan& plan, size_t pass, int rank, int log2_ranks, long long* unit_lo, long long* unit_n,
                    int* rank_bits_in_tile, std::string* err);
int qft_check_shard(const QftHostPlan& plan, int log2_ranks, std::string* err);
