// qft_launch.h -- the launcher's interface to the C ABI (qft_api.cu).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include <mutex>

#include "qft_plan.h"

// Per-pass launch state the plan owns: which device the kernel's attributes were set on, and the tensor
// maps already encoded for this pass (keyed by state pointer and device), so that a repeated qft_execute
// on the same buffer does no driver call besides the launch itself.
struct QftPassCache {
    std::mutex mu;
    int attr_dev = -1;
    int next = 0;
    struct Entry {
        void* ptr = nullptr;
        int dev = -1;
        CUtensorMap map;
    } maps[4];
};

// Enqueue one pass: tiles are loaded from `src` and stored to `state` (the same buffer for an in-place pass; a
// different one only if qft_pass_reads_through_tensor_map(d), else cudaErrorNotSupported).
cudaError_t qft_launch_pass(const QftPassDesc& d, QftPassCache* cache, void* src, void* state, cudaStream_t stream);
bool qft_pass_reads_through_tensor_map(const QftPassDesc& d);
// Pass launches so far (this process, any plan) that fell back to the generic kernel because no tensor map was granted.
unsigned long long qft_launch_map_fallbacks();
