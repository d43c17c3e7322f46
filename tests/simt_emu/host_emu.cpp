// host_emu.cpp -- TEST INFRASTRUCTURE.  The product's C ABI on the CPU: paper_2607_04067_b200/csrc/hough_api.cu -- the
// real host code: handles, options, planner, launch set-up, hough_run_host's staging and pointer arithmetic --
// compiled by g++ against fake_cuda_runtime.h, with every kernel launch executed by the SIMT emulator (simt_shim.h)
// on the kernel source.  Built as libhough_hostemu.so by tests/simt_emu/__init__.py and loaded by the CPU tests only:
// they call the same entry points, with host pointers standing in for device pointers, and compare with the oracle.
// Nothing in the product builds, loads or links this.
#include "fake_cuda_runtime.h"

#ifndef HOUGH_HOST_EMU
#error "build with -DHOUGH_HOST_EMU (tests/simt_emu/__init__.py)"
#endif
#ifdef HOUGH_KERNEL_HEADER
#error "mutants are built with emu_main.cpp"
#endif
#include "../../paper_2607_04067_b200/csrc/hough_api.cu"

namespace {
const void* g_fn = nullptr;
void* g_arg = nullptr;
void entry_event() { ((void (*)(hough::KParams))g_fn)(*(const hough::KParams*)g_arg); }
void entry_circles() { ((void (*)(hough::CParams))g_fn)(*(const hough::CParams*)g_arg); }

// a bulk copy that starts inside an emulated device allocation must end inside it (memory the fake runtime did not
// allocate -- a caller's own array in the dry run of the GPU tests -- cannot be judged)
bool inside_one_allocation(const void* p, size_t n) {
    for (auto& kv : fake_cuda::allocations) {
        const unsigned char* lo = kv.second.ptr;
        if ((const unsigned char*)p >= lo && (const unsigned char*)p < lo + kv.second.bytes) return (const unsigned char*)p + n <= lo + kv.second.bytes;
    }
    return true;
}

cudaError_t run_grid(const void* fn, void* arg, int grid, int C, int threads, size_t smem, void (*entry)()) {
    if (threads <= 0 || threads > 1024 || threads % 32 || grid <= 0 || C <= 0 || grid % C) return cudaErrorInvalidValue;
    const auto lim = fake_cuda::smem_limit.find(fn);
    if (smem > 48 * 1024 && (lim == fake_cuda::smem_limit.end() || smem > (size_t)lim->second)) return cudaErrorInvalidValue;   // opt-in missing
    if (C > 8 && !fake_cuda::nonportable[fn]) return cudaErrorInvalidValue;
    g_fn = fn; g_arg = arg;
    emu::bulk_range_ok = inside_one_allocation;
    ++fake_cuda::n_launch;
#ifdef EMU_RACE
    emu::race::new_launch();
#endif
    const int n_clusters = grid / C;
    emu::next_unlaunched = 0;                 // (scheduler mode 1: a running CTA takes not-yet-launched CTAs out of the grid)
    while (emu::next_unlaunched < n_clusters) {
        const int c = emu::next_unlaunched++;
        emu::g.n_clusters_ = n_clusters;
        emu::run_cluster(c, n_clusters, C, threads, smem ? smem : 16, entry);
    }
    return cudaSuccess;
}
}  // namespace

cudaError_t cudaLaunchKernelExC(const cudaLaunchConfig_t* cfg, const void* fn, void** args) {
    int C = 1;
    for (unsigned i = 0; i < cfg->numAttrs; ++i)
        if (cfg->attrs[i].id == cudaLaunchAttributeClusterDimension) C = (int)cfg->attrs[i].val.clusterDim.x;
    return run_grid(fn, args[0], (int)cfg->gridDim.x, C, (int)cfg->blockDim.x, cfg->dynamicSmemBytes, entry_event);
}

cudaError_t cudaLaunchKernel(const void* fn, dim3 grid, dim3 block, void** args, size_t smem, cudaStream_t) {
    return run_grid(fn, args[0], (int)grid.x, 1, (int)block.x, smem, entry_circles);
}

// "device" memory for the tests' own buffers (guard page behind the end, 16-byte aligned, known to the race check):
// upload = a host-to-device copy (the bytes count as written), poke = the same bytes without that mark (poison that
// the kernel is not supposed to read), download = device to host
// (not counted: the malloc / free counters are the LIBRARY's allocations)
extern "C" void* hough_hostemu_malloc(long long n) {
    void* p = nullptr;
    if (cudaMalloc(&p, (size_t)(n > 0 ? n : 1)) != cudaSuccess) return nullptr;
    --fake_cuda::n_malloc;
    return p;
}
extern "C" void hough_hostemu_free(void* p) { if (p && cudaFree(p) == cudaSuccess) --fake_cuda::n_free; }
extern "C" void hough_hostemu_upload(void* d, const void* s, long long n) { cudaMemcpyAsync(d, s, (size_t)n, cudaMemcpyHostToDevice, nullptr); }
extern "C" void hough_hostemu_poke(void* d, const void* s, long long n) { memcpy(d, s, (size_t)n); }
extern "C" void hough_hostemu_download(void* d, const void* s, long long n) { memcpy(d, s, (size_t)n); }

// what the tests ask the emulated device: {allocations made, freed, kernel launches, race / initcheck reports so far}
extern "C" void hough_hostemu_counters(long long out[4]) {
    out[0] = fake_cuda::n_malloc; out[1] = fake_cuda::n_free; out[2] = fake_cuda::n_launch;
#ifdef EMU_RACE
    out[3] = (long long)emu::race::n_reports;
#else
    out[3] = -1;
#endif
}
