/*
 * qft.h -- C ABI of the B200-native QFT / AQFT executor (libqft.so).
 *
 * The library executes the n-qubit QFT circuit of arxiv/paper_2606_18981
 * ("Not Your Usual FFT: QFT -> FFT via Classical Quantum-Circuit Simulation")
 * in place on a complex64 state vector of N = 2^n amplitudes that lives in the
 * memory of one B200:
 *
 *     for t = n-1 .. 0:   H(q_t);  CR_{d+1}(q_{t-d} -> q_t), d = 1 .. min(k, t)
 *     then the bit-reversal swaps SWAP(q_i, q_{n-1-i}), i < floor(n/2)
 *
 * (Fig. 1, PAPER.md:116 for the range-k truncation, PAPER.md:137
 * for the swaps), so that for k >= n-1 the result is the DFT of the input,
 *
 *     state[K] <- c * sum_j state[j] * exp(sign * 2 pi i * j K / N),
 *
 * with the paper's forward sign -1 and the paper's unitary
 * scaling c = 1/sqrt(N) by default.  Array index j is the basis
 * state whose qubit q is bit q of j (q_0 = least-significant bit, PAPER.md:82,
 * :96); input and output are both in natural order.  For k < n-1 the result is
 * that of the truncated circuit (the AQFT), which is not the DFT.
 *
 * A plan ("planner", fused blocks, device-agnostic schedule)
 * turns the gate list into a few fused passes over the state.  Each pass loads
 * a tile of amplitudes, applies every gate whose target lies in the tile's
 * window of qubits -- Hadamards as butterflies, all controlled-R_m as
 * per-amplitude phases computed from index bits ("commuting
 * diagonal factors collapse to one diagonal") -- and stores the tile through a
 * layout adapter that folds the bit reversal into the
 * store addressing.  DESIGN.md describes the schedule.
 *
 * All functions return a status code; no exception crosses this boundary and
 * no output argument is written on failure.  No PyTorch type appears here.
 */
#ifndef QFT_B200_H
#define QFT_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct qft_plan_s* qft_plan_t;

typedef enum {
    QFT_OK = 0,
    QFT_ERR_INVALID_ARG = 1, /* null pointer, n out of range, misaligned state, bad sign ... */
    QFT_ERR_UNSUPPORTED = 2, /* a tuning request the planner cannot schedule */
    QFT_ERR_ALLOC = 3,       /* host or device allocation failed */
    QFT_ERR_CUDA = 4,        /* a CUDA runtime call or kernel launch failed (no usable device included) */
    QFT_ERR_INTERNAL = 5     /* planner self-check failed: a bug, never expected */
} qft_status_t;

typedef enum {
    QFT_NORM_UNITARY = 0, /* c = 1/sqrt(N): the paper's U = DFT_N / sqrt(N) */
    QFT_NORM_NONE = 1,    /* c = 1: plain DFT_N, "multiply by scale_in sqrt(N)" of PAPER.md:139 */
    QFT_NORM_INV_N = 2    /* c = 1/N: "other FFT conventions ... one-line rescaling" */
} qft_norm_t;

#define QFT_MAX_QUBITS 34

/*
 * qft_plan_create -- build the fused schedule (host only; no device is touched,
 * so it also works on a machine without a GPU).
 *   out               receives the plan handle.
 *   n_qubits          1 .. QFT_MAX_QUBITS; the state has 2^n complex64 amplitudes.
 *   aqft_cutoff_k     >= 0.  Controlled rotations with control-target distance
 *                     > k are dropped; k >= n-1 is the exact QFT,
 *                     k = 0 leaves the Hadamards only.
 *   max_fused_qubits  >= 1.  Cap on the number of logical qubits whose gates one
 *                     pass applies (the planner's analogue of qsim's
 *                     max_fused_size).  Values above the device
 *                     limit are clamped, not an error: a transform that fits one
 *                     shared-memory tile (n <= 12) is one pass; otherwise a tile holds
 *                     2^12 (n = 13 ... 23), 2^13 (n = 24, 25) or 2^14 amplitudes (n >= 26;
 *                     2^15 with the tensor-memory extension), of which 3 to 6 address bits
 *                     are the contiguous granule, so a pass processes up to 8 ... 11 qubits
 *                     (n = 30: three passes of 10, n = 33: three of 11).  Values of 6 and
 *                     below cut those windows into sub-passes of at most that many qubits
 *                     (n = 26: 13 / 7 / 5 passes for 2 / 4 / 6).  The result does not depend
 *                     on it, only the number of passes does.
 *   sign              -1: the paper's forward transform; +1: every phase
 *                     conjugated.  With unitary normalisation this is the exact
 *                     inverse of the sign = -1 transform with the same k, for every
 *                     k: the (A)QFT matrix including the swaps is symmetric (the
 *                     gate list read backwards is the same circuit on the reversed
 *                     qubit order, reading c12), so its inverse, the
 *                     conjugate transpose, is its conjugate.
 *   normalisation     see qft_norm_t.
 */
qft_status_t qft_plan_create(qft_plan_t* out, int n_qubits, int aqft_cutoff_k, int max_fused_qubits, int sign,
                             qft_norm_t normalisation);

/*
 * qft_plan_create_batched -- plan for 2^log2_batch independent n_qubits-qubit transforms stored back to
 * back: device_state of qft_execute is float2[2^(n_qubits + log2_batch)], state b occupying elements
 * [b 2^n, (b+1) 2^n); every state gets the transform of qft_plan_create, in place, in the same launches.
 * This is SURVEY.md section 8(f1): the paper's measured sizes (n = 12 ... 22) cannot fill a
 * B200 one at a time.  n_qubits + log2_batch <= 34; log2_batch = 0 is qft_plan_create.  Other arguments,
 * errors and ownership as for qft_plan_create.
 */
qft_status_t qft_plan_create_batched(qft_plan_t* out, int n_qubits, int log2_batch, int aqft_cutoff_k,
                                     int max_fused_qubits, int sign, qft_norm_t normalisation);

/*
 * qft_plan_create_tuned -- as qft_plan_create, with the layout knobs exposed for
 * benchmarking: tile_bits (log2 amplitudes per tile, 0 = default), hub_bits
 * (log2 amplitudes per contiguous granule, 0 = default), flags (QFT_FLAG_*).
 * QFT_ERR_UNSUPPORTED if the combination cannot be scheduled (tile_bits outside 2..14, hub_bits outside
 * 1..6 or >= tile_bits, tile_bits < 2 * hub_bits for a state larger than a tile, an unknown flag).
 */
#define QFT_FLAG_GENERIC_ONLY 1u  /* use only the generic shared-memory tile kernel */
#define QFT_FLAG_UNFOLDED 2u      /* natural-order passes + one stand-alone bit-reversal pass */
#define QFT_FLAG_NO_TMA 4u        /* do not use the TMA-staged pass kernels */
#define QFT_FLAG_NO_EXT_TILE 16u  /* do not extend 2^14 tiles by one qubit through tensor memory */
/*
 * QFT_FLAG_DEFER_SWAPS -- the paper's own mode ("the final swaps are not implemented as gates but
 * accounted for in the caller as an output index permutation", "deferred to I/O or absorbed into
 * layout"): the swap network is left out, the planner takes the cheapest layout (no tile exchanges between
 * CTAs at all) and the plan reports it: after qft_execute, address bit a of the state holds the circuit's qubit
 * qubit_of_bit[a] (qft_plan_output_order).  The natural-order result is recovered by the caller as
 *     natural[K] = state[J],   bit a of J = bit (n-1-q) of K  with  q = qubit_of_bit[a].
 * Without the flag qubit_of_bit[a] = n-1-a (J = K).  The layout chosen today is the circuit's own
 * (qubit_of_bit[a] = a, i.e. plain bit-reversed output) except that bits a and n-1-a are exchanged for a below
 * the granule size; callers must read it from the plan, not assume it.  Not available for batched plans.
 */
#define QFT_FLAG_DEFER_SWAPS 32u
qft_status_t qft_plan_create_tuned(qft_plan_t* out, int n_qubits, int aqft_cutoff_k, int max_fused_qubits, int sign,
                                   qft_norm_t normalisation, int tile_bits, int hub_bits, unsigned flags);

/*
 * qft_execute -- enqueue the transform of `device_state` on `stream`, in place.
 *   device_state  DEVICE pointer to 2^n interleaved (re, im) float pairs, 16-byte
 *                 aligned (8-byte when n = 0 is not allowed, so always 16), owned
 *                 by the caller, on the device that is current at the time of the
 *                 call.  No other 2^n-sized buffer is allocated.
 *   stream        a cudaStream_t passed as void* (NULL = the legacy default stream).
 * Only enqueues kernels: no host synchronisation, no device allocation (the tensor
 * maps of the TMA kernels are encoded on the host and passed as kernel parameters),
 * capturable into a CUDA graph.  The schedule is immutable; the plan also keeps, per
 * pass and behind a mutex, the tensor maps it has encoded (keyed by state pointer and
 * device, four entries) and the device its kernel attributes were set on, so a repeated
 * call on the same buffer makes no driver call besides the launches.  A plan may be used
 * again, on other streams and from several threads at once.
 * Errors: QFT_ERR_INVALID_ARG (null / misaligned), QFT_ERR_CUDA (launch failed, or the
 * device has no tensor memory / TMA: the library is built for sm_100a only).
 */
qft_status_t qft_execute(qft_plan_t plan, void* device_state, void* stream);

/*
 * qft_execute_oop -- out of place: device_out receives the transform of device_in, which is left untouched
 * (same layout, alignment and ownership rules as qft_execute for both; the two buffers must be identical --
 * then this is qft_execute -- or disjoint, QFT_ERR_INVALID_ARG otherwise).  The first pass loads its tiles from
 * device_in through its tensor map and stores them into device_out, the remaining passes run in place on
 * device_out, so the bytes moved are those of qft_execute: no extra copy, no scratch.  (A plan whose first pass
 * is not a TMA pass -- states of fewer than about 2^14 amplitudes -- copies first.)  Only enqueues.
 */
qft_status_t qft_execute_oop(qft_plan_t plan, const void* device_in, void* device_out, void* stream);

/*
 * qft_execute_host -- the same transform for a state in HOST memory (pageable or
 * pinned): copies 2^n complex64 to a device buffer owned by the plan (allocated
 * on first use, 8 * 2^n bytes), runs qft_execute, copies the result back into
 * `host_state` and waits for it.  This is the end-to-end entry point timed as
 * "e2e" by bench.py.  Calls on one plan are serialised (it owns one staging buffer, on
 * the device that was current at the first call; QFT_ERR_INVALID_ARG if another device is
 * current later); for a batched plan the state has 2^(n_qubits + log2_batch) elements.
 */
qft_status_t qft_execute_host(qft_plan_t plan, void* host_state, void* stream);

/*
 * qft_execute_pass -- enqueue only pass `pass_index` (0 .. qft_plan_num_passes-1) of the plan.
 * Running every pass in order is exactly qft_execute; a single pass is a profiling aid (per-pass
 * CUDA-event timing for the roofline report) and leaves the state in an intermediate layout.
 */
qft_status_t qft_execute_pass(qft_plan_t plan, int pass_index, void* device_state, void* stream);

/* qft_plan_destroy -- free the plan and everything it owns.  NULL is allowed. */
qft_status_t qft_plan_destroy(qft_plan_t plan);

/*
 * Sharded state, host-side design (PAPER.md:229 outlook "scale with distributed simulators"; not measured on more than
 * one GPU).  The 2^n amplitudes live on 2^log2_ranks ranks; the top log2_ranks address bits select the rank and the
 * shards are mapped back to back into ONE virtual address range on every rank (peer memory over NVLink), so every
 * pass is the same kernel on the same addresses.  Rank r runs its share of the units of pass p,
 * qft_execute_pass_shard(plan, p, base, r, log2_ranks, stream), all ranks synchronise (a barrier, no data-path
 * collective), then pass p + 1.  A pass whose tiles hold no rank bit is local (rank r's units touch only its own
 * shard); a pass whose tiles hold g_in rank bits reads and writes a fraction 1 - 2^-g_in of its bytes on peers:
 * the all-to-all of the classical scheme, fused into the pass's loads and stores.
 *   qft_plan_shard_info: rank r's unit range of the pass, the rank bits inside its tiles and the bytes it moves over
 *     the links in each direction.  QFT_ERR_UNSUPPORTED if a rank bit takes part in a pair involution or the pass has
 *     fewer units than ranks (qft_last_cuda_error says which).
 *   qft_plan_shard_check: host proof for every pass and rank that the ranges tile the pass and that a local pass's
 *     units lie on their own rank (replays the kernel's unit -> tile -> address maps).
 *   qft_execute_pass_shard: enqueue rank r's share.  With every rank's share enqueued one after the other on ONE
 *     device (same buffer) the result is exactly qft_execute_pass; that is how the path is tested on one GPU.
 */
qft_status_t qft_plan_shard_info(qft_plan_t plan, int pass_index, int rank, int log2_ranks, long long* unit_lo,
                                 long long* unit_n, int* rank_bits_in_tile, long long* remote_bytes_each_way);
qft_status_t qft_plan_shard_check(qft_plan_t plan, int log2_ranks);
qft_status_t qft_execute_pass_shard(qft_plan_t plan, int pass_index, void* state_base, int rank, int log2_ranks,
                                    void* stream);

/* Introspection (the paper's plan carries the fused blocks and the counters of
 * 1- and 2-qubit gates before fusion). */
int qft_plan_num_passes(qft_plan_t plan);   /* -1 if plan is NULL */
int qft_plan_num_launches(qft_plan_t plan); /* kernels one qft_execute enqueues; -1 if NULL */
qft_status_t qft_plan_gate_counts(qft_plan_t plan, long long* n_h, long long* n_cr, long long* n_swap);
/* qubit_of_bit[a], a < n_qubits: the circuit's qubit whose (frequency) bit address bit a holds after qft_execute;
 * n-1-a for every plan without QFT_FLAG_DEFER_SWAPS (see there). */
qft_status_t qft_plan_output_order(qft_plan_t plan, int* qubit_of_bit);
/* JSON text describing every pass: kernel, tile address bits, window, register steps, store permutation,
 * pairing, and the fused block's gates ("each descriptor records the participating qubits, the
 * contiguous subrange of original gates folded into the block"): n_h, n_cr and [gate_first, gate_last], indices
 * into the time-ordered list  H(q_{n-1}), CR_2(q_{n-2} -> q_{n-1}), ..., H(q_0)  (the swaps follow it and belong to
 * no pass: they are the passes' store permutations).  Writes at most len-1 characters plus a NUL; returns
 * QFT_ERR_INVALID_ARG if the buffer is smaller than qft_plan_describe_length(plan) (bytes including the NUL;
 * 0 if plan is NULL). */
size_t qft_plan_describe_length(qft_plan_t plan);
qft_status_t qft_plan_describe(qft_plan_t plan, char* buf, size_t len);
/*
 * The steps either side of the circuit.  All take a device pointer to
 * float2[2^n_qubits] (16-byte aligned, n_qubits >= 1), accumulate in double precision, return a number
 * to the host and therefore SYNCHRONISE the stream (qft_rescale only enqueues).
 *   qft_norm_sq     *norm_sq_out = sum_j |x_j|^2.
 *   qft_encode    amplitude encoding of PAPER.md:124: *scale_in_out = ||x||_2 and x /= scale_in, in place;
 *                 QFT_ERR_INVALID_ARG for the zero vector.
 *   qft_rescale   x *= factor, in place: the decode step of PAPER.md:139 (factor = scale_in for the unitary
 *                 convention, scale_in * sqrt(N) for the unnormalised DFT).
 *   qft_fidelity  *fidelity_out = |<a,b>|^2 / (||a||^2 ||b||^2).
 *   qft_leakage   *leakage_out = 1 - |x[bin]|^2 / ||x||^2: the top-bin leakage of PAPER.md:181.
 *   qft_num_qubits_for   n = max(1, ceil(log2 length)) of PAPER.md:124 ("we choose n = ceil(log2 N) qubits and
 *                 allocate a 2^n-element state vector"); -1 if length is 0 or exceeds 2^34.
 *   qft_encode_padded    the whole input-encoding step of PAPER.md:124 for an array of any length <= 2^n_qubits:
 *                 copies device_x (float2[length], device memory; device_state itself or a buffer disjoint from
 *                 it, QFT_ERR_INVALID_ARG for a partial overlap) to the front of
 *                 device_state (float2[2^n_qubits]), zero-fills the rest, then qft_encode.  Note that the
 *                 transform of the padded state is the 2^n-point DFT of the padded array, not a length-point DFT.
 * The reductions keep one 32-byte scratch buffer per device (allocated at the first call on that device) and
 * serialise calls per device; they cannot be captured into a CUDA graph.
 */
int qft_num_qubits_for(unsigned long long length);
qft_status_t qft_encode_padded(void* device_state, int n_qubits, const void* device_x, unsigned long long length,
                               double* scale_in_out, void* stream);
qft_status_t qft_norm_sq(const void* device_state, int n_qubits, double* norm_sq_out, void* stream);
qft_status_t qft_encode(void* device_state, int n_qubits, double* scale_in_out, void* stream);
qft_status_t qft_rescale(void* device_state, int n_qubits, double factor, void* stream);
qft_status_t qft_fidelity(const void* device_a, const void* device_b, int n_qubits, double* fidelity_out, void* stream);
qft_status_t qft_leakage(const void* device_state, int n_qubits, unsigned long long bin, double* leakage_out,
                         void* stream);

/*
 * qft_fidelity_batched_static -- the fidelity of PAPER.md:181 for `batch` pairs of states at once, for callers that
 * cannot allocate device memory: a process whose HBM was all handed to one pool or arena at start-up (or filled by
 * the state vectors themselves: one n = 33 state is 64 GiB), where a cudaMalloc made later by a library fails, and a
 * caller in a latency-critical loop that cannot afford the device-wide stall an allocation or a free may cause.
 * qft_fidelity allocates its accumulators at the first call on a device; this function allocates and frees nothing,
 * on the host side of the runtime or the device, at any call.  Its accumulators (4 doubles per state) are a fixed
 * array inside the library image: QFT_STATIC_MAX_BATCH * 32 bytes = 128 KiB on every GPU that loads libqft.so, held
 * until the process exits.
 *   device_a, device_b   DEVICE pointers, float2[batch * 2^n_qubits] each, 16-byte aligned; pair b is elements
 *                        [b 2^n, (b+1) 2^n) of both (the layout of qft_plan_create_batched, any batch >= 1, not only
 *                        powers of two).  Read only.
 *   n_qubits             1 .. QFT_MAX_QUBITS;  batch * 2^n_qubits <= 2^34.
 *   batch                1 .. QFT_STATIC_MAX_BATCH.  A larger batch is refused with QFT_ERR_UNSUPPORTED and nothing is
 *                        enqueued; qft_static_last_error() then names the limit.  Split the batch, or use qft_fidelity.
 *   device_fidelity_out  DEVICE pointer, double[batch], 8-byte aligned, owned by the caller:
 *                        out[b] = |<a_b, b_b>|^2 / (||a_b||^2 ||b_b||^2), fp64 accumulation as in qft_fidelity;
 *                        NaN where a state of the pair is all zero (qft_fidelity refuses that case on the host; this
 *                        call never waits for the device, so it cannot).
 *   stream               a cudaStream_t as void*.  The call only enqueues (a clear of the accumulators it uses, the
 *                        reduction, a final division); it does not synchronise.
 * Shared scratch: every call on a device uses the same array, which still holds the previous call's sums.  Each
 * call clears its part in stream order, so calls that follow one another on one stream, or that the caller orders
 * with events, are correct; calls whose device work can overlap (two streams, two threads) race on the array and
 * return garbage without any error.
 * First call on a device: looks up the array's address on that device (one CUDA runtime call, under a lock, which
 * may load the module); later calls make no such call.  Make the first call before starting any stream capture.
 * Errors: QFT_ERR_INVALID_ARG (null, misaligned, n_qubits or batch out of range), QFT_ERR_UNSUPPORTED (batch beyond
 * the limit), QFT_ERR_CUDA (no device, address look-up or launch failed).  The text of the last error this function
 * returned on the calling thread is qft_static_last_error() ("" if none); qft_last_cuda_error() is not updated.
 */
#define QFT_STATIC_MAX_BATCH 4096
qft_status_t qft_fidelity_batched_static(const void* device_a, const void* device_b, int n_qubits, int batch,
                                         double* device_fidelity_out, void* stream);
const char* qft_static_last_error(void);

/* Re-runs the planner's host-side proof: follows every qubit through every
 * pass's address permutation and checks that each gate's target was inside the
 * tile when applied, that tiles are closed under the store permutation, and
 * that every qubit ends on its bit-reversed address.  QFT_OK or QFT_ERR_INTERNAL. */
qft_status_t qft_plan_self_check(qft_plan_t plan);

/*
 * qft_tensor_map_fallbacks -- how many pass launches of this process (any plan, any thread) ran the generic
 * shared-memory kernel because the driver refused to encode the pass's tensor map.  qft_execute still returns QFT_OK
 * then and the result is the same, but such a pass runs at roughly a tenth of the TMA kernel's bandwidth; the driver
 * accepts every map the planner produces today, so anything but 0 deserves a look.  bench.py reports it.
 */
unsigned long long qft_tensor_map_fallbacks(void);

const char* qft_status_string(qft_status_t status);
/* Last CUDA error text seen by this library on the calling thread ("" if none). */
const char* qft_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* QFT_B200_H */
