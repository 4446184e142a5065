// qft_metrics.cu -- the steps either side of the circuit: input encoding
// (divide by scale_in = ||x||_2), output decoding (one rescale) and the
// paper's accuracy metrics (fidelity and top-bin leakage), as HBM-bound device reductions
// with double-precision accumulation.  These calls return a number to the host and therefore synchronise.
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>

#include "../../include/qft.h"

namespace {

// sums[0] = sum |a|^2, sums[1] = sum |b|^2, sums[2] + i sums[3] = sum conj(a) b   (b may be null)
__global__ void __launch_bounds__(256) qft_reduce4(const float4* __restrict__ a, const float4* __restrict__ b,
                                                   unsigned long long npairs, double* __restrict__ sums) {
    double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < npairs; i += stride) {
        const float4 u = a[i];  // two amplitudes
        // the squares and products of two fp32 numbers are exact in fp64
        s0 += (double)u.x * u.x + (double)u.y * u.y + (double)u.z * u.z + (double)u.w * u.w;
        if (b) {
            const float4 v = b[i];
            s1 += (double)v.x * v.x + (double)v.y * v.y + (double)v.z * v.z + (double)v.w * v.w;
            s2 += (double)u.x * v.x + (double)u.y * v.y + (double)u.z * v.z + (double)u.w * v.w;
            s3 += (double)u.x * v.y - (double)u.y * v.x + (double)u.z * v.w - (double)u.w * v.z;
        }
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
        atomicAdd(&sums[threadIdx.x], t);
    }
}

__global__ void __launch_bounds__(256) qft_scale_kernel(float4* __restrict__ a, unsigned long long npairs, float s) {
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < npairs; i += stride) {
        float4 u = a[i];
        u.x *= s; u.y *= s; u.z *= s; u.w *= s;
        a[i] = u;
    }
}

// One 32-byte sums buffer per device, allocated at the first call on that device and kept for the life of the
// process; a call holds its device's lock until the sums are back on the host (the calls synchronise anyway).
constexpr int kMaxDevices = 64;
struct DevScratch {
    std::mutex mu;
    double* sums = nullptr;
    int grid = 0;  // 8 CTAs per SM of that device
};
DevScratch g_scratch[kMaxDevices];

int grid_for(int dev) {
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) sms = 148;
    return sms * 8;
}

qft_status_t reduce4(const void* a, const void* b, int n, cudaStream_t s, double out[4]) {
    if (!a || n < 1 || n > 34 || (((uintptr_t)a) & 15) || (b && (((uintptr_t)b) & 15))) return QFT_ERR_INVALID_ARG;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return QFT_ERR_CUDA;
    DevScratch& sc = g_scratch[dev];
    std::lock_guard<std::mutex> lock(sc.mu);
    if (!sc.sums) {
        if (cudaMalloc(&sc.sums, 4 * sizeof(double)) != cudaSuccess) { sc.sums = nullptr; return QFT_ERR_ALLOC; }
        sc.grid = grid_for(dev);
    }
    if (cudaMemsetAsync(sc.sums, 0, 4 * sizeof(double), s) != cudaSuccess) return QFT_ERR_CUDA;
    const unsigned long long npairs = (1ull << n) / 2;  // n >= 1: at least one pair
    unsigned long long blocks = (npairs + 255) / 256;
    if (blocks > (unsigned long long)sc.grid) blocks = sc.grid;
    qft_reduce4<<<(unsigned)blocks, 256, 0, s>>>((const float4*)a, (const float4*)b, npairs, sc.sums);
    if (cudaGetLastError() != cudaSuccess) return QFT_ERR_CUDA;
    if (cudaMemcpyAsync(out, sc.sums, 4 * sizeof(double), cudaMemcpyDeviceToHost, s) != cudaSuccess) return QFT_ERR_CUDA;
    if (cudaStreamSynchronize(s) != cudaSuccess) return QFT_ERR_CUDA;
    return QFT_OK;
}

}  // namespace

extern "C" {

qft_status_t qft_norm_sq(const void* device_state, int n_qubits, double* norm_sq_out, void* stream) {
    if (!norm_sq_out) return QFT_ERR_INVALID_ARG;
    double s[4];
    qft_status_t st = reduce4(device_state, nullptr, n_qubits, (cudaStream_t)stream, s);
    if (st == QFT_OK) *norm_sq_out = s[0];
    return st;
}

qft_status_t qft_rescale(void* device_state, int n_qubits, double factor, void* stream) {
    if (!device_state || n_qubits < 1 || n_qubits > 34 || (((uintptr_t)device_state) & 15)) return QFT_ERR_INVALID_ARG;
    const unsigned long long npairs = (1ull << n_qubits) / 2;
    unsigned long long blocks = (npairs + 255) / 256;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return QFT_ERR_CUDA;
    const unsigned long long cap = (unsigned long long)grid_for(dev);
    if (blocks > cap) blocks = cap;
    qft_scale_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>((float4*)device_state, npairs, (float)factor);
    return cudaGetLastError() == cudaSuccess ? QFT_OK : QFT_ERR_CUDA;
}

qft_status_t qft_encode(void* device_state, int n_qubits, double* scale_in_out, void* stream) {
    if (!scale_in_out) return QFT_ERR_INVALID_ARG;
    double n2 = 0.0;
    qft_status_t st = qft_norm_sq(device_state, n_qubits, &n2, stream);
    if (st != QFT_OK) return st;
    if (!(n2 > 0.0)) return QFT_ERR_INVALID_ARG;  // the zero vector has no encoding
    const double scale_in = sqrt(n2);
    *scale_in_out = scale_in;
    return qft_rescale(device_state, n_qubits, 1.0 / scale_in, stream);
}

int qft_num_qubits_for(unsigned long long length) {
    if (length == 0 || length > (1ull << 34)) return -1;
    int n = 0;
    while ((1ull << n) < length) ++n;
    return n < 1 ? 1 : n;
}

qft_status_t qft_encode_padded(void* device_state, int n_qubits, const void* device_x, unsigned long long length,
                               double* scale_in_out, void* stream) {
    if (!device_state || !device_x || !scale_in_out || n_qubits < 1 || n_qubits > 34 || length == 0 ||
        length > (1ull << n_qubits) || (((uintptr_t)device_state) & 15))
        return QFT_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    if (device_x != device_state) {
        // the copy below is undefined for overlapping ranges: the source is the state itself or disjoint from it
        const char *x0 = (const char*)device_x, *x1 = x0 + 8ull * length;
        const char *s0 = (const char*)device_state, *s1 = s0 + (8ull << n_qubits);
        if (x0 < s1 && s0 < x1) return QFT_ERR_INVALID_ARG;
    }
    if (device_x != device_state &&
        cudaMemcpyAsync(device_state, device_x, 8ull * length, cudaMemcpyDeviceToDevice, s) != cudaSuccess)
        return QFT_ERR_CUDA;
    const unsigned long long total = 1ull << n_qubits;
    if (length < total &&
        cudaMemsetAsync((char*)device_state + 8ull * length, 0, 8ull * (total - length), s) != cudaSuccess)
        return QFT_ERR_CUDA;
    return qft_encode(device_state, n_qubits, scale_in_out, stream);
}

qft_status_t qft_fidelity(const void* device_a, const void* device_b, int n_qubits, double* fidelity_out, void* stream) {
    if (!fidelity_out || !device_b) return QFT_ERR_INVALID_ARG;
    double s[4];
    qft_status_t st = reduce4(device_a, device_b, n_qubits, (cudaStream_t)stream, s);
    if (st != QFT_OK) return st;
    if (!(s[0] > 0.0) || !(s[1] > 0.0)) return QFT_ERR_INVALID_ARG;
    *fidelity_out = (s[2] * s[2] + s[3] * s[3]) / (s[0] * s[1]);
    return QFT_OK;
}

qft_status_t qft_leakage(const void* device_state, int n_qubits, unsigned long long bin, double* leakage_out,
                         void* stream) {
    if (!leakage_out || n_qubits < 1 || n_qubits > 34 || bin >= (1ull << n_qubits)) return QFT_ERR_INVALID_ARG;
    double s[4];
    qft_status_t st = reduce4(device_state, nullptr, n_qubits, (cudaStream_t)stream, s);
    if (st != QFT_OK) return st;
    if (!(s[0] > 0.0)) return QFT_ERR_INVALID_ARG;
    float2 v;
    if (cudaMemcpyAsync(&v, (const float2*)device_state + bin, sizeof v, cudaMemcpyDeviceToHost, (cudaStream_t)stream) !=
            cudaSuccess ||
        cudaStreamSynchronize((cudaStream_t)stream) != cudaSuccess)
        return QFT_ERR_CUDA;
    *leakage_out = 1.0 - ((double)v.x * v.x + (double)v.y * v.y) / s[0];
    return QFT_OK;
}

}  // extern "C"
