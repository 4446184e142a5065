// qft_api.cu -- the C ABI declared in include/qft.h.
#include <cuda_runtime.h>

#include <cstring>
#include <new>
#include <string>

#include <memory>

#include "../../include/qft.h"
#include "qft_launch.h"

struct qft_plan_s {
    QftHostPlan host;
    std::unique_ptr<QftPassCache[]> cache;  // one per pass: encoded tensor maps, kernel attributes (qft_launch.h)
    std::mutex host_mu;                     // serialises qft_execute_host on this plan
    void* dev_buf = nullptr;                // only for qft_execute_host
    int dev_buf_device = -1;
    size_t dev_bytes = 0;
};

static thread_local std::string g_cuda_err;

static qft_status_t cuda_fail(cudaError_t e) {
    g_cuda_err = cudaGetErrorString(e);
    return QFT_ERR_CUDA;
}

extern "C" {

static qft_status_t create_from(qft_plan_t* out, const QftPlanParams& prm) {
    if (!out) return QFT_ERR_INVALID_ARG;
    qft_plan_s* p = new (std::nothrow) qft_plan_s();
    if (!p) return QFT_ERR_ALLOC;
    std::string err;
    int rc;
    try {
        rc = qft_build_plan(prm, &p->host, &err);
        if (rc == 0) p->cache.reset(new QftPassCache[p->host.passes.size()]);
    } catch (const std::bad_alloc&) {
        delete p;
        return QFT_ERR_ALLOC;
    } catch (...) {
        delete p;
        return QFT_ERR_INTERNAL;
    }
    if (rc != 0) {
        delete p;
        g_cuda_err = err;
        return (qft_status_t)rc;
    }
    *out = p;
    return QFT_OK;
}

qft_status_t qft_plan_create_tuned(qft_plan_t* out, int n_qubits, int aqft_cutoff_k, int max_fused_qubits, int sign,
                                   qft_norm_t normalisation, int tile_bits, int hub_bits, unsigned flags) {
    QftPlanParams prm;
    prm.n = n_qubits;
    prm.k = aqft_cutoff_k;
    prm.max_fused = max_fused_qubits;
    prm.sign = sign;
    prm.norm = (int)normalisation;
    prm.tile_bits = tile_bits;
    prm.hub_bits = hub_bits;
    prm.flags = flags;
    return create_from(out, prm);
}

qft_status_t qft_plan_create_batched(qft_plan_t* out, int n_qubits, int log2_batch, int aqft_cutoff_k,
                                     int max_fused_qubits, int sign, qft_norm_t normalisation) {
    QftPlanParams prm;
    prm.n = n_qubits;
    prm.batch_bits = log2_batch;
    prm.k = aqft_cutoff_k;
    prm.max_fused = max_fused_qubits;
    prm.sign = sign;
    prm.norm = (int)normalisation;
    return create_from(out, prm);
}

qft_status_t qft_plan_create(qft_plan_t* out, int n_qubits, int aqft_cutoff_k, int max_fused_qubits, int sign,
                             qft_norm_t normalisation) {
    return qft_plan_create_tuned(out, n_qubits, aqft_cutoff_k, max_fused_qubits, sign, normalisation, 0, 0, 0u);
}

qft_status_t qft_execute(qft_plan_t plan, void* device_state, void* stream) {
    if (!plan || !device_state) return QFT_ERR_INVALID_ARG;
    const uintptr_t align = plan->host.prm.n >= 1 ? 16 : 8;
    if (((uintptr_t)device_state) & (align - 1)) return QFT_ERR_INVALID_ARG;
    for (size_t i = 0; i < plan->host.passes.size(); ++i) {
        cudaError_t e = qft_launch_pass(plan->host.passes[i], &plan->cache[i], device_state, device_state, (cudaStream_t)stream);
        if (e != cudaSuccess) return cuda_fail(e);
    }
    return QFT_OK;
}

qft_status_t qft_execute_oop(qft_plan_t plan, const void* device_in, void* device_out, void* stream) {
    if (!plan || !device_in || !device_out) return QFT_ERR_INVALID_ARG;
    if ((((uintptr_t)device_in) | ((uintptr_t)device_out)) & 15) return QFT_ERR_INVALID_ARG;
    if (device_in == device_out) return qft_execute(plan, device_out, stream);
    const size_t bytes = (size_t)8 << (plan->host.prm.n + plan->host.prm.batch_bits);
    const char *a = (const char*)device_in, *b = (const char*)device_out;
    if ((a < b && a + bytes > b) || (b < a && b + bytes > a)) return QFT_ERR_INVALID_ARG;  // partial overlap
    size_t first = 0;
    if (!plan->host.passes.empty() && qft_pass_reads_through_tensor_map(plan->host.passes[0])) {
        // the first pass reads its tiles from the input through the tensor map and stores them into the output
        cudaError_t e = qft_launch_pass(plan->host.passes[0], &plan->cache[0], (void*)device_in, device_out, (cudaStream_t)stream);
        if (e != cudaSuccess) return cuda_fail(e);
        first = 1;
    } else {
        cudaError_t e = cudaMemcpyAsync(device_out, device_in, bytes, cudaMemcpyDeviceToDevice, (cudaStream_t)stream);
        if (e != cudaSuccess) return cuda_fail(e);
    }
    for (size_t i = first; i < plan->host.passes.size(); ++i) {
        cudaError_t e = qft_launch_pass(plan->host.passes[i], &plan->cache[i], device_out, device_out, (cudaStream_t)stream);
        if (e != cudaSuccess) return cuda_fail(e);
    }
    return QFT_OK;
}

qft_status_t qft_plan_output_order(qft_plan_t plan, int* qubit_of_bit) {
    if (!plan || !qubit_of_bit) return QFT_ERR_INVALID_ARG;
    for (int a = 0; a < plan->host.prm.n; ++a) qubit_of_bit[a] = plan->host.out_qubit_at[a];
    return QFT_OK;
}

qft_status_t qft_execute_pass(qft_plan_t plan, int pass_index, void* device_state, void* stream) {
    if (!plan || !device_state || pass_index < 0 || pass_index >= (int)plan->host.passes.size())
        return QFT_ERR_INVALID_ARG;
    if (((uintptr_t)device_state) & 15) return QFT_ERR_INVALID_ARG;
    cudaError_t e = qft_launch_pass(plan->host.passes[pass_index], &plan->cache[pass_index], device_state, device_state,
                                    (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(e);
    return QFT_OK;
}

qft_status_t qft_plan_shard_info(qft_plan_t plan, int pass_index, int rank, int log2_ranks, long long* unit_lo,
                                 long long* unit_n, int* rank_bits_in_tile, long long* remote_bytes_each_way) {
    if (!plan || pass_index < 0 || pass_index >= (int)plan->host.passes.size() || !unit_lo || !unit_n || !rank_bits_in_tile ||
        !remote_bytes_each_way)
        return QFT_ERR_INVALID_ARG;
    std::string err;
    const int rc = qft_shard_range(plan->host, (size_t)pass_index, rank, log2_ranks, unit_lo, unit_n, rank_bits_in_tile, &err);
    if (rc != 0) {
        g_cuda_err = err;
        return (qft_status_t)rc;
    }
    const QftPassDesc& d = plan->host.passes[pass_index];
    const long long bytes = (*unit_n * (d.npair ? 2 : 1)) * ((long long)8 << (d.f + d.xt));  // this rank's share of the pass
    *remote_bytes_each_way = bytes - (bytes >> *rank_bits_in_tile);
    return QFT_OK;
}

qft_status_t qft_plan_shard_check(qft_plan_t plan, int log2_ranks) {
    if (!plan) return QFT_ERR_INVALID_ARG;
    std::string err;
    const int rc = qft_check_shard(plan->host, log2_ranks, &err);
    if (rc != 0) {
        g_cuda_err = err;
        return (qft_status_t)rc;
    }
    return QFT_OK;
}

qft_status_t qft_execute_pass_shard(qft_plan_t plan, int pass_index, void* state_base, int rank, int log2_ranks,
                                    void* stream) {
    if (!plan || !state_base || pass_index < 0 || pass_index >= (int)plan->host.passes.size()) return QFT_ERR_INVALID_ARG;
    if (((uintptr_t)state_base) & 15) return QFT_ERR_INVALID_ARG;
    long long lo, cnt;
    int g_in;
    std::string err;
    const int rc = qft_shard_range(plan->host, (size_t)pass_index, rank, log2_ranks, &lo, &cnt, &g_in, &err);
    if (rc != 0) {
        g_cuda_err = err;
        return (qft_status_t)rc;
    }
    QftPassDesc d = plan->host.passes[pass_index];
    d.unit_lo = (int32_t)lo;
    d.unit_n = (int32_t)cnt;
    cudaError_t e = qft_launch_pass(d, &plan->cache[pass_index], state_base, state_base, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(e);
    return QFT_OK;
}

qft_status_t qft_execute_host(qft_plan_t plan, void* host_state, void* stream) {
    if (!plan || !host_state) return QFT_ERR_INVALID_ARG;
    const size_t bytes = (size_t)8 << (plan->host.prm.n + plan->host.prm.batch_bits);
    cudaStream_t s = (cudaStream_t)stream;
    std::lock_guard<std::mutex> lock(plan->host_mu);
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e);
    if (!plan->dev_buf) {
        e = cudaMalloc(&plan->dev_buf, bytes);
        if (e != cudaSuccess) {
            plan->dev_buf = nullptr;
            g_cuda_err = cudaGetErrorString(e);
            return e == cudaErrorMemoryAllocation ? QFT_ERR_ALLOC : QFT_ERR_CUDA;
        }
        plan->dev_bytes = bytes;
        plan->dev_buf_device = dev;
    }
    if (plan->dev_buf_device != dev) return QFT_ERR_INVALID_ARG;  // the staging buffer lives on another device
    e = cudaMemcpyAsync(plan->dev_buf, host_state, bytes, cudaMemcpyHostToDevice, s);
    if (e != cudaSuccess) return cuda_fail(e);
    qft_status_t st = qft_execute(plan, plan->dev_buf, stream);
    if (st != QFT_OK) return st;
    e = cudaMemcpyAsync(host_state, plan->dev_buf, bytes, cudaMemcpyDeviceToHost, s);
    if (e != cudaSuccess) return cuda_fail(e);
    e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return cuda_fail(e);
    return QFT_OK;
}

qft_status_t qft_plan_destroy(qft_plan_t plan) {
    if (!plan) return QFT_OK;
    if (plan->dev_buf) cudaFree(plan->dev_buf);
    delete plan;
    return QFT_OK;
}

int qft_plan_num_passes(qft_plan_t plan) { return plan ? (int)plan->host.passes.size() : -1; }
int qft_plan_num_launches(qft_plan_t plan) { return plan ? (int)plan->host.passes.size() : -1; }

qft_status_t qft_plan_gate_counts(qft_plan_t plan, long long* n_h, long long* n_cr, long long* n_swap) {
    if (!plan || !n_h || !n_cr || !n_swap) return QFT_ERR_INVALID_ARG;
    *n_h = plan->host.n_h;
    *n_cr = plan->host.n_cr;
    *n_swap = plan->host.n_swap;
    return QFT_OK;
}

size_t qft_plan_describe_length(qft_plan_t plan) {
    if (!plan) return 0;
    try {
        return qft_describe_plan(plan->host).size() + 1;
    } catch (...) {
        return 0;
    }
}

qft_status_t qft_plan_describe(qft_plan_t plan, char* buf, size_t len) {
    if (!plan || !buf || len == 0) return QFT_ERR_INVALID_ARG;
    std::string s;
    try {
        s = qft_describe_plan(plan->host);
    } catch (...) {
        return QFT_ERR_ALLOC;
    }
    if (s.size() + 1 > len) return QFT_ERR_INVALID_ARG;
    std::memcpy(buf, s.c_str(), s.size() + 1);
    return QFT_OK;
}

qft_status_t qft_plan_self_check(qft_plan_t plan) {
    if (!plan) return QFT_ERR_INVALID_ARG;
    std::string err;
    int rc = qft_check_plan(plan->host, &err);
    if (rc != 0) {
        g_cuda_err = err;
        return QFT_ERR_INTERNAL;
    }
    return QFT_OK;
}

const char* qft_status_string(qft_status_t status) {
    switch (status) {
        case QFT_OK: return "ok";
        case QFT_ERR_INVALID_ARG: return "invalid argument";
        case QFT_ERR_UNSUPPORTED: return "unsupported";
        case QFT_ERR_ALLOC: return "allocation failed";
        case QFT_ERR_CUDA: return "CUDA error";
        case QFT_ERR_INTERNAL: return "internal planner error";
    }
    return "unknown status";
}

const char* qft_last_cuda_error(void) { return g_cuda_err.c_str(); }

unsigned long long qft_tensor_map_fallbacks(void) { return qft_launch_map_fallbacks(); }

#ifdef QFT_PHASE_TIMING
// profiling builds only: device buffer of 16 counters the TMA kernel of pass `pass_index` accumulates into
int qft_debug_set_phase_buffer(qft_plan_t plan, int pass_index, void* device_counters) {
    if (!plan || pass_index < 0 || pass_index >= (int)plan->host.passes.size()) return 1;
    plan->host.passes[pass_index].dbg = (unsigned long long*)device_counters;
    return 0;
}
#endif

}  // extern "C"
