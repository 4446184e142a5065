// qft_metrics_static.cu -- qft_fidelity_batched_static (include/qft.h): the fidelity reduction of qft_metrics.cu
// for a batch of states, for callers that cannot allocate device memory.
//
// Who that is: a process that handed all of its HBM to one pool up front (a serving framework's arena, or an
// application whose state vectors were sized to fill the card -- one n = 33 state is 64 GiB -- so that a later
// cudaMalloc has nothing left to give), and a caller inside a latency-critical loop that must not take the
// device-wide stall an allocation or a free can bring.  qft_fidelity allocates its 32-byte accumulator buffer
// with cudaMalloc at the first call on a device; this entry point never does.  Its accumulators live in a
// device array that is part of the library image: every GPU that loads libqft.so holds its 128 KiB
// (QFT_STATIC_MAX_BATCH states x 4 doubles) until the process exits, whether or not this function is ever called.
//
// Consequences the caller has to know (also in qft.h):
//   * at most QFT_STATIC_MAX_BATCH states per call; more is refused (QFT_ERR_UNSUPPORTED), never truncated;
//   * every call on a device uses the SAME array, which still holds the previous call's sums: each call clears
//     the part it uses on its stream before the reduction, and two calls whose work overlaps on the GPU
//     (different streams, different threads) race on it -- order them;
//   * the first call on each device looks the array's device address up (one runtime call, which may also load
//     the module); make that first call before starting any stream capture.
// The file calls no allocating or freeing runtime routine; tests/test_zz_no_alloc.py checks the source for that.
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>
#include <string>

#include "../../include/qft.h"

// The scratch: sums[4 b + 0..3] = sum |a|^2, sum |b|^2, Re and Im of sum conj(a) b over state b of the batch.
// In host code this name is only a handle for cudaGetSymbolAddress, never a pointer a kernel may be given.
static __device__ __align__(256) double qft_static_sums[QFT_STATIC_MAX_BATCH * 4];

namespace {

// grid = (CTAs per state, batch): CTA (x, y) strides over the pairs of amplitudes of state y.  Same arithmetic
// as qft_reduce4 in qft_metrics.cu (products of fp32 numbers are exact in fp64; fp64 accumulation).
__global__ void __launch_bounds__(256) qft_reduce4_batched(const float4* __restrict__ a, const float4* __restrict__ b,
                                                           unsigned long long npairs, double* __restrict__ sums) {
    const float4* __restrict__ as = a + (unsigned long long)blockIdx.y * npairs;
    const float4* __restrict__ bs = b + (unsigned long long)blockIdx.y * npairs;
    double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < npairs; i += stride) {
        const float4 u = as[i];
        const float4 v = bs[i];
        s0 += (double)u.x * u.x + (double)u.y * u.y + (double)u.z * u.z + (double)u.w * u.w;
        s1 += (double)v.x * v.x + (double)v.y * v.y + (double)v.z * v.z + (double)v.w * v.w;
        s2 += (double)u.x * v.x + (double)u.y * v.y + (double)u.z * v.z + (double)u.w * v.w;
        s3 += (double)u.x * v.y - (double)u.y * v.x + (double)u.z * v.w - (double)u.w * v.z;
    }
    __shared__ double sh[4][8];
    double s[4] = {s0, s1, s2, s3};
#pragma unroll
    for (int j = 0; j < 4; ++j) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s[j] += __shfl_xor_sync(0xffffffffu, s[j], o);
        if ((threadIdx.x & 31) == 0) sh[j][threadIdx.x >> 5] = s[j];
    }
    __syncthreads();
    if (threadIdx.x < 4) {
        double t = 0.0;
        for (int w = 0; w < 8; ++w) t += sh[threadIdx.x][w];
        atomicAdd(&sums[4 * blockIdx.y + threadIdx.x], t);
    }
}

// out[b] = |<a_b, b_b>|^2 / (||a_b||^2 ||b_b||^2); 0/0 = NaN for a zero state (there is no host to refuse it)
__global__ void qft_fidelity_finish(const double* __restrict__ sums, int batch, double* __restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < batch) {
        const double* s = sums + 4 * i;
        out[i] = (s[2] * s[2] + s[3] * s[3]) / (s[0] * s[1]);
    }
}

// Set-up, once per device, with that device current: the array's address ON THAT DEVICE and the grid size.
constexpr int kMaxDevices = 64;
struct DevSetup {
    double* sums = nullptr;  // device address of qft_static_sums on this device
    int ctas = 0;            // 8 CTAs per SM
};
DevSetup g_setup[kMaxDevices];
std::mutex g_setup_mu;

thread_local std::string g_static_err;

qft_status_t fail(qft_status_t st, const std::string& why) {
    g_static_err = why;
    return st;
}

}  // namespace

extern "C" {

qft_status_t qft_fidelity_batched_static(const void* device_a, const void* device_b, int n_qubits, int batch,
                                         double* device_fidelity_out, void* stream) {
    // arguments first: nothing below touches a device before they are accepted
    if (!device_a || !device_b || !device_fidelity_out)
        return fail(QFT_ERR_INVALID_ARG, "qft_fidelity_batched_static: null pointer");
    if ((((uintptr_t)device_a) | ((uintptr_t)device_b)) & 15)
        return fail(QFT_ERR_INVALID_ARG, "qft_fidelity_batched_static: states must be 16-byte aligned");
    if (((uintptr_t)device_fidelity_out) & 7)
        return fail(QFT_ERR_INVALID_ARG, "qft_fidelity_batched_static: device_fidelity_out must be 8-byte aligned");
    if (n_qubits < 1 || n_qubits > QFT_MAX_QUBITS || batch < 1)
        return fail(QFT_ERR_INVALID_ARG, "qft_fidelity_batched_static: n_qubits outside 1..34 or batch < 1");
    if (batch > QFT_STATIC_MAX_BATCH)
        return fail(QFT_ERR_UNSUPPORTED,
                    "qft_fidelity_batched_static: batch " + std::to_string(batch) + " exceeds QFT_STATIC_MAX_BATCH = " +
                        std::to_string(QFT_STATIC_MAX_BATCH) +
                        " (the built-in scratch array holds no more; split the batch, or use qft_fidelity)");
    if ((unsigned long long)batch > ((1ull << QFT_MAX_QUBITS) >> n_qubits))
        return fail(QFT_ERR_INVALID_ARG, "qft_fidelity_batched_static: batch * 2^n_qubits exceeds 2^34 amplitudes");

    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= kMaxDevices)
        return fail(QFT_ERR_CUDA, std::string("qft_fidelity_batched_static: no usable current device: ") +
                                      (e != cudaSuccess ? cudaGetErrorString(e) : "device ordinal >= 64"));
    double* sums = nullptr;
    int ctas = 0;
    {
        std::lock_guard<std::mutex> lock(g_setup_mu);
        DevSetup& su = g_setup[dev];
        if (!su.sums) {
            // the first call on this device: ask the runtime where the array lives here
            double* p = nullptr;
            e = cudaGetSymbolAddress((void**)&p, qft_static_sums);
            if (e != cudaSuccess || !p)
                return fail(QFT_ERR_CUDA, std::string("qft_fidelity_batched_static: cudaGetSymbolAddress failed: ") +
                                              cudaGetErrorString(e));
            int sms = 0;
            if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) sms = 148;
            su.ctas = sms * 8;
            su.sums = p;
        }
        sums = su.sums;
        ctas = su.ctas;
    }

    cudaStream_t s = (cudaStream_t)stream;
    // the array still holds the last call's sums: clear this call's part, in stream order
    e = cudaMemsetAsync(sums, 0, (size_t)batch * 4 * sizeof(double), s);
    if (e != cudaSuccess)
        return fail(QFT_ERR_CUDA, std::string("qft_fidelity_batched_static: clearing the scratch failed: ") + cudaGetErrorString(e));
    const unsigned long long npairs = (1ull << n_qubits) / 2;
    unsigned long long per_state = (npairs + 255) / 256;
    const unsigned long long share = (unsigned long long)(ctas / batch > 0 ? ctas / batch : 1);
    if (per_state > share) per_state = share;
    qft_reduce4_batched<<<dim3((unsigned)per_state, (unsigned)batch), 256, 0, s>>>((const float4*)device_a,
                                                                                   (const float4*)device_b, npairs, sums);
    e = cudaGetLastError();
    if (e == cudaSuccess) {
        qft_fidelity_finish<<<(batch + 255) / 256, 256, 0, s>>>(sums, batch, device_fidelity_out);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess)
        return fail(QFT_ERR_CUDA, std::string("qft_fidelity_batched_static: launch failed: ") + cudaGetErrorString(e));
    return QFT_OK;
}

const char* qft_static_last_error(void) { return g_static_err.c_str(); }

}  // extern "C"
