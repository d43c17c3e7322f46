// fake_cuda_runtime.h -- TEST INFRASTRUCTURE.  Stands in for <cuda_runtime.h> when the product's HOST code
// (paper_2607_04067_b200/csrc/hough_api.cu: handle management, planner, launch set-up, hough_run_host's staging) is
// compiled by g++ together with the kernel source under the SIMT shim (host_emu.cpp).  "Device" memory is host memory
// whose END sits on a guard page; copies and memsets are immediate; streams are ignored (everything is synchronous);
// a kernel launch runs the kernel under the emulator, cluster after cluster.  Only what hough_api.cu calls exists.
#pragma once
#include <map>

#include "simt_shim.h"

typedef int cudaError_t;
enum : int { cudaSuccess = 0, cudaErrorInvalidValue = 1, cudaErrorMemoryAllocation = 2 };
struct FakeStream;
typedef FakeStream* cudaStream_t;
enum cudaMemcpyKind { cudaMemcpyHostToHost = 0, cudaMemcpyHostToDevice = 1, cudaMemcpyDeviceToHost = 2, cudaMemcpyDeviceToDevice = 3 };
enum cudaFuncAttribute { cudaFuncAttributeMaxDynamicSharedMemorySize = 8, cudaFuncAttributeNonPortableClusterSizeAllowed = 11 };
enum cudaLaunchAttributeID { cudaLaunchAttributeClusterDimension = 4 };
struct cudaLaunchAttributeValue { struct { unsigned x, y, z; } clusterDim; };
struct cudaLaunchAttribute { cudaLaunchAttributeID id; cudaLaunchAttributeValue val; };
struct cudaLaunchConfig_t {
    dim3 gridDim, blockDim;
    size_t dynamicSmemBytes = 0;
    cudaStream_t stream = nullptr;
    cudaLaunchAttribute* attrs = nullptr;
    unsigned numAttrs = 0;
};
struct cudaDeviceProp {
    char name[256];
    int major, minor, multiProcessorCount;
    size_t sharedMemPerBlockOptin;
};

namespace fake_cuda {
// the emulated device: a B200 as the planner sees it (148 SMs, 227 KB of shared memory per CTA after opt-in, 228 KB per SM)
constexpr int SM_COUNT = 148;
constexpr size_t SMEM_OPTIN = 232448, SMEM_PER_SM = 233472, SMEM_RESERVED_PER_CTA = 1024;
inline std::map<void*, emu::Guarded> allocations;
inline std::map<const void*, int> smem_limit;        // cudaFuncAttributeMaxDynamicSharedMemorySize per kernel
inline std::map<const void*, int> nonportable;
inline long long n_malloc = 0, n_free = 0, n_launch = 0;
}  // namespace fake_cuda

inline const char* cudaGetErrorString(cudaError_t e) { return e == cudaSuccess ? "no error" : e == cudaErrorMemoryAllocation ? "out of memory (fake)" : "invalid value (fake)"; }
inline cudaError_t cudaGetLastError() { return cudaSuccess; }
inline cudaError_t cudaGetDeviceCount(int* n) { *n = 1; return cudaSuccess; }
inline cudaError_t cudaGetDevice(int* d) { *d = 0; return cudaSuccess; }
inline cudaError_t cudaGetDeviceProperties(cudaDeviceProp* p, int) {
    memset(p, 0, sizeof(*p));
    strcpy(p->name, "SIMT emulator (B200 shape)");
    p->major = 10; p->minor = 0; p->multiProcessorCount = fake_cuda::SM_COUNT; p->sharedMemPerBlockOptin = fake_cuda::SMEM_OPTIN;
    return cudaSuccess;
}
inline cudaError_t cudaMalloc(void** p, size_t n) {
    emu::Guarded g;
    g.alloc((n + 15) / 16 * 16 + 16);                  // 16-byte aligned like every real allocation; ends at a guard page
    memset(g.ptr, 0xA5, g.bytes);                      // device memory starts as garbage
    *p = g.ptr;
#ifdef EMU_RACE
    emu::race::track(g.ptr, g.bytes, false, -1, "global");
#endif
    fake_cuda::allocations[g.ptr] = g;
    ++fake_cuda::n_malloc;
    return cudaSuccess;
}
template <class T> inline cudaError_t cudaMalloc(T** p, size_t n) { return cudaMalloc((void**)p, n); }
inline cudaError_t cudaFree(void* p) {
    if (!p) return cudaSuccess;
    auto it = fake_cuda::allocations.find(p);
    if (it == fake_cuda::allocations.end()) return cudaErrorInvalidValue;
#ifdef EMU_RACE
    emu::race::untrack(p);
#endif
    it->second.release();
    fake_cuda::allocations.erase(it);
    ++fake_cuda::n_free;
    return cudaSuccess;
}
inline cudaError_t cudaMemcpyAsync(void* d, const void* s, size_t n, cudaMemcpyKind, cudaStream_t);
inline cudaError_t cudaMemcpy(void* d, const void* s, size_t n, cudaMemcpyKind k) { return cudaMemcpyAsync(d, s, n, k, nullptr); }
inline cudaError_t cudaMemcpyAsync(void* d, const void* s, size_t n, cudaMemcpyKind, cudaStream_t) {
#ifdef EMU_RACE
    emu::race::host_write(d, n);                       // what a copy wrote counts as written for the initcheck
#endif
    memcpy(d, s, n);
    return cudaSuccess;
}
inline cudaError_t cudaMemsetAsync(void* d, int v, size_t n, cudaStream_t) {
#ifdef EMU_RACE
    emu::race::host_write(d, n);
#endif
    memset(d, v, n);
    return cudaSuccess;
}
inline cudaError_t cudaStreamSynchronize(cudaStream_t) { return cudaSuccess; }
inline cudaError_t cudaFuncSetAttribute(const void* fn, cudaFuncAttribute a, int v) {
    if (a == cudaFuncAttributeMaxDynamicSharedMemorySize) {
        if (v < 0 || (size_t)v > fake_cuda::SMEM_OPTIN) return cudaErrorInvalidValue;
        fake_cuda::smem_limit[fn] = v;
    } else {
        fake_cuda::nonportable[fn] = v;
    }
    return cudaSuccess;
}
inline cudaError_t cudaOccupancyMaxActiveBlocksPerMultiprocessor(int* n, const void*, int threads, size_t smem) {
    const int by_smem = (int)(fake_cuda::SMEM_PER_SM / (smem + fake_cuda::SMEM_RESERVED_PER_CTA)), by_threads = 2048 / threads;
    *n = by_smem < by_threads ? by_smem : by_threads;
    return cudaSuccess;
}
inline cudaError_t cudaOccupancyMaxActiveClusters(int* n, const void* fn, const cudaLaunchConfig_t* cfg) {
    const int C = cfg->numAttrs ? (int)cfg->attrs[0].val.clusterDim.x : 1;
    if (C > 8 && !fake_cuda::nonportable[fn]) return cudaErrorInvalidValue;
    int per_sm = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, (int)cfg->blockDim.x, cfg->dynamicSmemBytes);
    *n = per_sm * (fake_cuda::SM_COUNT / C);           // (clusters never straddle GPCs here: an upper bound is enough for the planner)
    return cudaSuccess;
}
// defined in host_emu.cpp, after the kernel source
cudaError_t cudaLaunchKernelExC(const cudaLaunchConfig_t* cfg, const void* fn, void** args);
cudaError_t cudaLaunchKernel(const void* fn, dim3 grid, dim3 block, void** args, size_t smem, cudaStream_t stream);
