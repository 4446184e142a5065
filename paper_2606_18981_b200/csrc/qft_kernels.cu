// qft_kernels.cu -- the pass kernels (sm_100a) and their launcher.
//
// Generic tile pass (QFT_KERNEL_GENERIC): works for every pass descriptor the planner can emit.
//   1. load the tile (all addresses that agree outside F) into shared memory in canonical order,
//      one 8-byte amplitude per lane, lanes running along the hub so that every warp request covers
//      whole 2^l * 8-byte granules;
//   2. for each step, every thread takes 2^r amplitudes that differ in the step's r canonical bits,
//      applies H and all controlled rotations onto those r qubits (register butterflies with constant
//      twiddles for controls inside the group, index-bit phases for controls outside it:
//      PAPER.md:112, :114), and puts them back;
//   3. store through the pass's layout adapter: canonical bit -> address bit
//      permutation inside the tile and, for pair passes, into the partner tile's addresses after a
//      cluster barrier (both CTAs of the pair have finished loading by then, so in place is safe).
#include <cuda_runtime.h>
#include <stdint.h>

#include "qft_device.cuh"
#include "qft_fused.cuh"
#include "qft_launch.h"

#include <algorithm>
#include <atomic>

namespace qftk {

// bank swizzle of the shared-memory image (any bijection is correct; this one spreads strided steps)
__device__ __forceinline__ uint32_t swz(uint32_t c) { return c ^ ((c >> 4) & 0xFu) ^ ((c >> 8) & 0xFu); }

template <int R, bool FAST>
__device__ __forceinline__ void generic_step(float2* tile, const QftPassDesc& d, const QftStep st, uint64_t Ltile,
                                             bool scale_now) {
    const int a = st.a;
    const int t_hi = st.t_hi;
    const int t_lo = t_hi - R + 1;
    const uint32_t nb = 1u << (d.f - R);
    const uint32_t lowmask = (1u << a) - 1u;
    const uint64_t lmask = (t_lo > 0) ? ((1ull << t_lo) - 1ull) : 0ull;
    // logical bits below the group that this thread's own index bits contribute: the same for all its butterflies
    const int lt = d.log2_threads;
    uint64_t Lthread = Ltile;
    for (int b = 0; b < a && b < lt; ++b)
        if ((threadIdx.x >> b) & 1u) Lthread |= 1ull << d.log_canon[b];
    for (uint32_t o = threadIdx.x; o < nb; o += blockDim.x) {
        const uint32_t c0 = ((o & ~lowmask) << R) | (o & lowmask);
        float2 x[1 << R];
#pragma unroll
        for (int u = 0; u < (1 << R); ++u) x[u] = tile[swz(c0 | ((uint32_t)u << a))];
        dif_group<R, FAST>(x, d.k);
        if (t_lo > 0) {
            // logical bits below the group: from the tile index and from this thread's canonical low bits
            uint64_t L = Lthread;
            for (int b = lt; b < a; ++b)
                if ((c0 >> b) & 1u) L |= 1ull << d.log_canon[b];
            L &= lmask;
#pragma unroll
            for (int i = 0; i < R; ++i) {
                const float2 W = cis_fwd_u32(cr_phase_u32(L, t_hi - i, d.k));
                const int pos = R - 1 - i;
#pragma unroll
                for (int u = 0; u < (1 << R); ++u)
                    if (u & (1 << pos)) x[u] = cmul(x[u], W);
            }
        }
        if (scale_now) {
#pragma unroll
            for (int u = 0; u < (1 << R); ++u) { x[u].x *= d.scale; x[u].y *= d.scale; }
        }
#pragma unroll
        for (int u = 0; u < (1 << R); ++u) tile[swz(c0 | ((uint32_t)u << a))] = x[u];
    }
}

template <int R>
__device__ __forceinline__ void generic_step_dispatch(float2* tile, const QftPassDesc& d, const QftStep st,
                                                      uint64_t Ltile, bool scale_now) {
    if (d.k >= R - 1) generic_step<R, true>(tile, d, st, Ltile, scale_now);
    else generic_step<R, false>(tile, d, st, Ltile, scale_now);
}

// RMAX: the largest register group this instantiation handles.  The one for groups of <= 2 qubits (one-qubit windows
// on small tiles, permutation-only passes) is compiled for 4 CTAs per SM; the general one needs 250 registers for its
// 32-point groups and runs one CTA per SM (profiles/r02_config3_sweep.md).
template <int RMAX>
__global__ void __launch_bounds__(256, RMAX <= 2 ? 4 : 1) qft_tile_pass_generic(float2* __restrict__ state,
                                                                               const __grid_constant__ QftPassDesc d) {
    extern __shared__ float2 tile[];
    const uint32_t tid = threadIdx.x;
    const int lt = d.log2_threads;

    uint32_t mload, mstore;
    decode_tile(blockIdx.x + (uint32_t)d.unit_lo * (d.npair ? 2u : 1u), d.npair, &mload, &mstore);
    uint64_t base_ld = 0, base_st = 0, Ltile = 0;
    for (int i = 0; i < d.ntile; ++i) {
        if ((mload >> i) & 1u) {
            base_ld |= 1ull << d.tile_addr[i];
            Ltile |= 1ull << d.log_tile[i];
        }
        if ((mstore >> i) & 1u) base_st |= 1ull << d.tile_addr[i];
    }

    // ---- load ----
    {
        uint64_t off_t = 0;
        uint32_t can_t = 0;
        for (int j = 0; j < lt && j < d.f; ++j)
            if ((tid >> j) & 1u) { off_t |= 1ull << d.F[j]; can_t |= 1u << d.ld_canon[j]; }
        const uint32_t niter = (d.f > lt) ? (1u << (d.f - lt)) : 1u;
        const bool active = (d.f >= lt) || (tid < (1u << d.f));
        if (active) {
            // eight loads in flight per thread before the first one is consumed
            for (uint32_t it0 = 0; it0 < niter; it0 += 8) {
                float2 v[8];
                uint32_t can[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const uint32_t it = it0 + u;
                    uint64_t off = off_t;
                    can[u] = can_t;
                    for (int j = lt; j < d.f; ++j)
                        if ((it >> (j - lt)) & 1u) { off |= 1ull << d.F[j]; can[u] |= 1u << d.ld_canon[j]; }
                    if (it < niter) v[u] = state[base_ld + off];
                }
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    if (it0 + u >= niter) break;
                    if (d.conj) v[u].y = -v[u].y;
                    tile[swz(can[u])] = v[u];
                }
            }
        }
    }
    __syncthreads();
    if (d.npair) cluster_arrive();  // this CTA has read its whole tile

    // ---- steps ----
    for (int s = 0; s < d.nsteps; ++s) {
        const QftStep st = d.steps[s];
        const bool scale_now = d.do_scale && (s == d.nsteps - 1);
        if constexpr (RMAX <= 2) {
            if (st.r == 1) generic_step_dispatch<1>(tile, d, st, Ltile, scale_now);
            else generic_step_dispatch<2>(tile, d, st, Ltile, scale_now);
        } else {
            switch (st.r) {
                case 1: generic_step_dispatch<1>(tile, d, st, Ltile, scale_now); break;
                case 2: generic_step_dispatch<2>(tile, d, st, Ltile, scale_now); break;
                case 3: generic_step_dispatch<3>(tile, d, st, Ltile, scale_now); break;
                case 4: generic_step_dispatch<4>(tile, d, st, Ltile, scale_now); break;
                default: generic_step_dispatch<5>(tile, d, st, Ltile, scale_now); break;
            }
        }
        __syncthreads();
    }
    if (d.npair) cluster_wait();  // the partner has read its tile: its addresses may be overwritten

    // ---- store ----
    {
        uint64_t off_t = 0;
        uint32_t can_t = 0;
        for (int j = 0; j < lt && j < d.f; ++j)
            if ((tid >> j) & 1u) { off_t |= 1ull << d.F[j]; can_t |= 1u << d.st_canon[j]; }
        const uint32_t niter = (d.f > lt) ? (1u << (d.f - lt)) : 1u;
        const bool active = (d.f >= lt) || (tid < (1u << d.f));
        if (active) {
            for (uint32_t it = 0; it < niter; ++it) {
                uint64_t off = off_t;
                uint32_t can = can_t;
                for (int j = lt; j < d.f; ++j)
                    if ((it >> (j - lt)) & 1u) { off |= 1ull << d.F[j]; can |= 1u << d.st_canon[j]; }
                float2 v = tile[swz(can)];
                if (d.conj) v.y = -v.y;
                state[base_st + off] = v;
            }
        }
    }
}

}  // namespace qftk

// ---------------------------------------------------------------------------------------------
// launcher
// ---------------------------------------------------------------------------------------------
typedef void (*pass_kernel_t)(float2*, const QftPassDesc);

static pass_kernel_t pick_kernel(const QftPassDesc& d) {
    if (d.kernel == QFT_KERNEL_FUSED2) {
        const int r1 = d.steps[0].r, r2 = d.steps[1].r;
        const bool fast = d.k >= 4;  // no in-group truncation for any radix <= 32
#define QFT_PICK(A, B)                                                                   \
    if (r1 == A && r2 == B)                                                              \
        return fast ? (pass_kernel_t)qftk::qft_pass_fused2<A, B, true> : (pass_kernel_t)qftk::qft_pass_fused2<A, B, false>;
        QFT_PICK(5, 5)
        QFT_PICK(5, 4)
        QFT_PICK(4, 4)
        QFT_PICK(4, 3)
        QFT_PICK(3, 3)
        QFT_PICK(3, 2)
        QFT_PICK(2, 2)
#undef QFT_PICK
    }
    int rmax = 0;
    for (int s = 0; s < d.nsteps; ++s) rmax = d.steps[s].r > rmax ? d.steps[s].r : rmax;
    return rmax <= 2 ? (pass_kernel_t)qftk::qft_tile_pass_generic<2> : (pass_kernel_t)qftk::qft_tile_pass_generic<5>;
}

// ---- QFT_KERNEL_TMA2 ---------------------------------------------------------------------------
typedef void (*tma2_kernel_t)(float2*, const CUtensorMap, const QftPassDesc);
tma2_kernel_t qft_pick_tma2_lt7(int r1, int r2, int kc);  // qft_tma_lt7.cu
tma2_kernel_t qft_pick_tma2_lt8(int r1, int r2, int kc);  // qft_tma_lt8.cu
tma2_kernel_t qft_pick_tma2_lt9(int r1, int r2, int kc);  // qft_tma_lt9.cu
tma2_kernel_t qft_pick_tma2_xt(int r1, int r2, int kc);   // qft_tma_xt.cu
tma2_kernel_t qft_pick_tma2_es7(int r1, int r2, int kc);  // qft_tma_es.cu
tma2_kernel_t qft_pick_tma2_es8(int r1, int r2, int kc);
tma2_kernel_t qft_pick_tma2_es9(int r1, int r2, int kc);

static tma2_kernel_t pick_tma2(const QftPassDesc& d) {
    const int kc = d.k < 4 ? d.k : 4;
    if (d.xt) return d.log2_threads == 9 ? qft_pick_tma2_xt(d.tma.r1, d.tma.r2, kc) : nullptr;
    if (d.tma.eb > QFT_TMA2_EB_DIRECT) {
        switch (d.log2_threads) {
            case 7: return qft_pick_tma2_es7(d.tma.r1, d.tma.r2, kc);
            case 8: return qft_pick_tma2_es8(d.tma.r1, d.tma.r2, kc);
            case 9: return qft_pick_tma2_es9(d.tma.r1, d.tma.r2, kc);
        }
        return nullptr;
    }
    switch (d.log2_threads) {
        case 7: return qft_pick_tma2_lt7(d.tma.r1, d.tma.r2, kc);
        case 8: return qft_pick_tma2_lt8(d.tma.r1, d.tma.r2, kc);
        case 9: return qft_pick_tma2_lt9(d.tma.r1, d.tma.r2, kc);
    }
    return nullptr;
}

typedef CUresult (*encode_tiled_t)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                   const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                   CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static encode_tiled_t get_encode_tiled() {
    static encode_tiled_t fn = []() -> encode_tiled_t {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) != cudaSuccess ||
            qres != cudaDriverEntryPointSuccess)
            return nullptr;
        return (encode_tiled_t)p;
    }();
    return fn;
}

static int sm_count(int dev) {
    static int cached[64] = {0};
    if (dev < 0 || dev >= 64) return 148;
    if (cached[dev] > 0) return cached[dev];
    int v = 0;
    if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || v <= 0) return 148;
    cached[dev] = v;  // benign race: every writer stores the same value
    return v;
}

// The opt-in ceiling of dynamic shared memory on this device.  Every kernel gets this value as its attribute
// (it only lifts the 48 KB default; occupancy follows the bytes a launch actually asks for), so passes that
// share one kernel function but need different table sizes cannot lower each other's limit.
static int smem_optin(int dev) {
    static int cached[64] = {0};
    if (dev < 0 || dev >= 64) return 227 * 1024;
    if (cached[dev] > 0) return cached[dev];
    int v = 0;
    if (cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess || v <= 0) return 227 * 1024;
    cached[dev] = v;
    return v;
}

// The units (tiles, or tile pairs of a pair pass) a launch walks: the descriptor's range, or all of them.
static void fill_units(QftPassDesc* d) {
    if (d->unit_n == 0) {
        d->unit_lo = 0;
        d->unit_n = (int32_t)((1ull << (d->ntile - d->xt)) / (d->npair ? 2u : 1u));
    }
}

static cudaError_t launch_plain(const QftPassDesc& d_in, QftPassCache* cache, int dev, void* state, cudaStream_t stream) {
    QftPassDesc d = d_in;
    fill_units(&d);
    pass_kernel_t kern = pick_kernel(d);
    const size_t smem = (size_t)8 << d.f;
    if (smem > 48 * 1024 && cache->attr_dev != dev) {
        cudaError_t e = cudaFuncSetAttribute((const void*)kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin(dev));
        if (e != cudaSuccess) return e;
        cache->attr_dev = dev;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)d.unit_n * (d.npair ? 2u : 1u));
    cfg.blockDim = dim3(1u << d.log2_threads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    cfg.attrs = attr;
    cfg.numAttrs = 0;
    if (d.npair > 0) {
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = 2;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        cfg.numAttrs = 1;
    }
    void* args[2] = {(void*)&state, (void*)&d};
    return cudaLaunchKernelExC(&cfg, (const void*)kern, args);
}

// The tensor map of a pass: the state seen as a 5-D tensor over address-bit runs (qft_plan.cpp, lower_tma2).
// The strides are those of the runs, so a later dimension may have a smaller stride than an earlier one and the
// tile-index dimension overlaps the others; the driver accepts this today.  If it ever refuses, the caller falls
// back to the generic kernel (same descriptor, no tensor map).
static bool encode_map(const QftPassDesc& d, void* state, CUtensorMap* map) {
    encode_tiled_t enc = get_encode_tiled();
    if (!enc) return false;
    cuuint64_t gdim[5], gstr[4];
    cuuint32_t box[5], estr[5];
    for (int i = 0; i < 5; ++i) {
        gdim[i] = 1ull << d.tma.tma_len[i];
        box[i] = 1u << d.tma.tma_box[i];
        estr[i] = 1;
        if (i > 0) gstr[i - 1] = 8ull << d.tma.tma_lo[i];
    }
    return enc(map, CU_TENSOR_MAP_DATA_TYPE_UINT64, 5, state, gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_64B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// The tensor map of pass d for the buffer `src`: from the pass's cache, else encoded now (false: the driver refused).
static bool get_map(const QftPassDesc& d, QftPassCache* cache, int dev, void* src, CUtensorMap* map) {
    for (const auto& e : cache->maps)
        if (e.ptr == src && e.dev == dev) {
            *map = e.map;
            return true;
        }
    if (!encode_map(d, src, map)) return false;
    QftPassCache::Entry& e = cache->maps[cache->next];
    cache->next = (cache->next + 1) % 4;
    e.ptr = src;
    e.dev = dev;
    e.map = *map;
    return true;
}

// Launches that ran the generic kernel because the driver refused the pass's tensor map (about 10x slower, same
// result): counted so that the slow path cannot be taken unnoticed (qft_tensor_map_fallbacks, include/qft.h).
static std::atomic<unsigned long long> g_map_fallbacks{0};
unsigned long long qft_launch_map_fallbacks() { return g_map_fallbacks.load(std::memory_order_relaxed); }

static int tma2_ctas_per_sm(const QftPassDesc& d, size_t smem) {
    int per_sm = d.f == 13 ? 2 : (d.f == 12 ? 4 : 1);
    while (per_sm > 1 && per_sm * (smem + 1024) > 227 * 1024) --per_sm;
    return per_sm;
}

// src: the buffer the tile loads come from (the tensor map's base); state: the buffer the stores go to.  They differ
// only for the first pass of an out-of-place execute.
static cudaError_t launch_tma2(const QftPassDesc& d_in, QftPassCache* cache, int dev, void* src, void* state,
                               cudaStream_t stream) {
    QftPassDesc d = d_in;
    fill_units(&d);
    tma2_kernel_t kern = pick_tma2(d);
    if (!kern) return cudaErrorNotSupported;
    const size_t smem = ((size_t)8 << d.f) + QFT_TMA2_TABLE_BYTES(d.tma.eb, d.ntile);
    CUtensorMap map;
    {
        std::lock_guard<std::mutex> lock(cache->mu);
        if (!get_map(d, cache, dev, src, &map)) {
            if (d.xt || src != state) return cudaErrorNotSupported;
            // no tensor map: the generic kernel runs the same descriptor (F = Fst for every plain pass)
            QftPassDesc g = d;
            g.kernel = QFT_KERNEL_GENERIC;
            g.log2_threads = 8;
            g_map_fallbacks.fetch_add(1, std::memory_order_relaxed);
            // A cold path: a fresh cache per launch, so the shared-memory attribute is set (idempotent) for whichever
            // generic instantiation this pass picks; one shared cache would skip it for the second instantiation.
            QftPassCache plain;
            return launch_plain(g, &plain, dev, state, stream);
        }
        if (cache->attr_dev != dev) {
            cudaError_t e = cudaFuncSetAttribute((const void*)kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin(dev));
            if (e != cudaSuccess) return e;
            cache->attr_dev = dev;
        }
    }
    const unsigned csz = d.npair ? 2u : 1u;
    unsigned long long grid = (unsigned long long)sm_count(dev) * tma2_ctas_per_sm(d, smem);
    if (grid > (unsigned long long)d.unit_n * csz) grid = (unsigned long long)d.unit_n * csz;
    grid -= grid % csz;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(1u << d.log2_threads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[2];
    cfg.attrs = attr;
    cfg.numAttrs = 0;
    if (d.npair > 0) {
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = 2;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        cfg.numAttrs = 1;
    }
    // Programmatic dependent launch: the kernel's prologue (barrier init, phase tables) may overlap the tail
    // of the previous pass; it executes griddepcontrol.wait before it touches the state.
    attr[cfg.numAttrs].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[cfg.numAttrs].val.programmaticStreamSerializationAllowed = 1;
    ++cfg.numAttrs;
    void* args[3] = {(void*)&state, (void*)&map, (void*)&d};
    return cudaLaunchKernelExC(&cfg, (const void*)kern, args);
}

bool qft_pass_reads_through_tensor_map(const QftPassDesc& d) { return d.kernel == QFT_KERNEL_TMA2; }

cudaError_t qft_launch_pass(const QftPassDesc& d, QftPassCache* cache, void* src, void* state, cudaStream_t stream) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (d.kernel == QFT_KERNEL_TMA2) return launch_tma2(d, cache, dev, src, state, stream);
    if (src != state) return cudaErrorNotSupported;
    std::lock_guard<std::mutex> lock(cache->mu);
    return launch_plain(d, cache, dev, state, stream);
}
