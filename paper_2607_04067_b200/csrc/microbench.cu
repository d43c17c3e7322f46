// microbench.cu -- measurement aids behind hough_bench_shared_atomics()
// (include/hough.h).  They give the denominators of the vote roofline
// (DESIGN.md "Roofline"): the SM's conflict-free shared-atomic rate and the
// issue-slot bound of the voting loop's instruction mix.
#include <cstdio>

#include "hough_kernel.cuh"

namespace {


// variants 0-2: nothing but shared atomics.  8 atomics per loop trip.
template <int VARIANT>
__global__ void __launch_bounds__(1024, 1) atomics_kernel(long long iters, unsigned* sink) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int ROWS = 256;   // 256 rows x 32 banks x 4 B = 32 KB
    unsigned* a = (unsigned*)smem;
    for (int i = threadIdx.x; i < ROWS * 32; i += blockDim.x) a[i] = 0;
    __syncthreads();
    const unsigned lane = threadIdx.x & 31;
    const unsigned base = (unsigned)__cvta_generic_to_shared(a);
    unsigned x = threadIdx.x * 2654435761u + blockIdx.x * 40503u + 12345u;
    const unsigned reg_inc = 0x10000u + (unsigned)(iters >> 62);   // a register value, not the literal 1
    for (long long it = 0; it < iters; ++it) {
        x = x * 1664525u + 1013904223u;
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            unsigned row = ((x >> (3 * q)) + 37u * q) & (ROWS - 1);
            unsigned addr;
            if (VARIANT == 2) {
                unsigned bank = (x >> (2 * q + 5)) & 31u;           // pseudo-random bank per lane
                addr = base + ((row << 5) + bank) * 4u;
            } else {
                addr = base + ((row << 5) + lane) * 4u;             // lane == bank: conflict-free
            }
            if (VARIANT == 1) hough::red_shared_add(addr, reg_inc);
            else hough::red_shared_add(addr, 1u);
        }
    }
    __syncthreads();
    if (sink && threadIdx.x == 0) sink[blockIdx.x] = a[lane];
}

// variant 5: the ATOMS pipe alone -- eight fixed, conflict-free addresses per thread (lane == bank), no address
// arithmetic in the loop.  This is the denominator of the vote roofline.
__global__ void __launch_bounds__(1024, 1) atomics_peak_kernel(long long iters, unsigned* sink) {
    extern __shared__ __align__(128) unsigned char smem[];
    unsigned* a = (unsigned*)smem;
    for (int i = threadIdx.x; i < 8192; i += blockDim.x) a[i] = 0;
    __syncthreads();
    const unsigned s = (unsigned)__cvta_generic_to_shared(a) + (threadIdx.x & 31) * 4u;
    const unsigned a0 = s, a1 = s + 128 * 3, a2 = s + 128 * 7, a3 = s + 128 * 12, a4 = s + 128 * 17, a5 = s + 128 * 21,
                   a6 = s + 128 * 30, a7 = s + 128 * 33;
    for (long long it = 0; it < iters; ++it) {
        asm volatile(
            "red.shared.add.u32 [%0],1; red.shared.add.u32 [%1],1; red.shared.add.u32 [%2],1; red.shared.add.u32 [%3],1; "
            "red.shared.add.u32 [%4],1; red.shared.add.u32 [%5],1; red.shared.add.u32 [%6],1; red.shared.add.u32 [%7],1;" ::
                "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(a4), "r"(a5), "r"(a6), "r"(a7));
    }
    __syncthreads();
    if (sink && threadIdx.x == 0) sink[blockIdx.x] = a[threadIdx.x & 31];
}

// variants 3-4 and 6-8: the voting loop's instruction mix over a synthetic (u,v) buffer
// (180 x 256 u16 geometry: 3 groups of 64 columns), with or without the atomics, scalar or packed
// (fp32x2) arithmetic, row pitch 384 B (IMAD addressing) or 512 B (shift-add addressing).
template <bool ATOMICS, bool PACKED, int PITCH>
__global__ void __launch_bounds__(1024, 1) votemix_kernel(long long iters, unsigned* sink) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int N_RHO = 256, NHITS = 1024;
    unsigned char* acc = smem;                               // (256 + 1 trash) rows
    float2* hb = (float2*)(smem + (N_RHO + 1) * PITCH);      // 8 KB
    for (int i = threadIdx.x; i < (N_RHO + 1) * PITCH / 4; i += blockDim.x) ((unsigned*)acc)[i] = 0;
    for (int i = threadIdx.x; i < NHITS; i += blockDim.x) {
        float r = 200.0f + 600.0f * (float)((i * 37) % 48) / 47.0f, phi = 0.0061359f * (float)i;
        float x = r * cosf(phi), y = r * sinf(phi);
        hb[i] = hough::conformal(make_float2(x, y), 1.0f);
    }
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const int g = warp % 3, stripe = warp / 3, n_stripes = nwarps / 3;
    const int j0 = 64 * g + lane, j1 = j0 + 32;
    const float th0 = 3.14159265f * j0 / 180.0f, th1 = 3.14159265f * j1 / 180.0f;
    const float c0 = cosf(th0), c1 = cosf(th1), s0 = sinf(th0), s1 = sinf(th1);
    const float rho_max = 1.0f / 334.0f, inv = 42752.0f;
    const unsigned pitch = PITCH, limit = N_RHO * PITCH;
    const unsigned lc0 = 4u * (g * 32 + lane) - HOUGH_MAGIC_BITS * pitch, lc1 = lc0;
    const unsigned acc_s = (unsigned)__cvta_generic_to_shared(acc);
    const unsigned trash = limit + 4u * (g * 32 + lane);
    const hough::ull C2 = hough::pack2(c0, c1), S2 = hough::pack2(s0, s1);
    unsigned chk = 0;
    if (stripe < n_stripes) {
        for (long long it = 0; it < iters; ++it) {
#pragma unroll 4
            for (int i = stripe; i < NHITS; i += n_stripes) {
                const float2 uv = hb[i];
                unsigned b0, b1;
                if (PACKED) {
                    hough::bin_bits2(uv.x, uv.y, C2, S2, rho_max, inv, b0, b1);
                } else {
                    b0 = hough::bin_bits(uv.x, uv.y, c0, s0, rho_max, inv);
                    b1 = hough::bin_bits(uv.x, uv.y, c1, s1, rho_max, inv);
                }
                const unsigned rel0 = b0 * pitch + lc0, rel1 = b1 * pitch + lc1;
                if (ATOMICS) {
                    hough::vote_add(acc_s + min(rel0, trash), 1u);
                    hough::vote_add(acc_s + min(rel1, trash), 0x10000u);
                } else {
                    chk += (rel0 < limit ? rel0 : 0u) ^ (rel1 < limit ? rel1 : 0u);
                }
            }
        }
    }
    __syncthreads();
    if (sink && (chk == 0x12345u || threadIdx.x == 0)) sink[blockIdx.x] = ((unsigned*)acc)[lane] + chk;
}

}  // namespace

extern "C" int hough_bench_shared_atomics(int variant, int ctas_per_sm, int threads, long long iters, double* out_rate) {
    if (variant < 0 || variant > 8 || ctas_per_sm < 1 || threads < 32 || threads > 1024 || (threads & 31) || iters < 1 || !out_rate)
        return HOUGH_ERR_INVALID_ARG;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return HOUGH_ERR_CUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return HOUGH_ERR_CUDA;
    const int grid = sms * ctas_per_sm;
    unsigned* sink = nullptr;
    if (cudaMalloc(&sink, sizeof(unsigned) * grid) != cudaSuccess) return HOUGH_ERR_NOMEM;
    size_t smem = (variant <= 2 || variant == 5) ? 32768 : (257 * (variant == 8 ? 512 : 384) + 8192);
    const void* fn = nullptr;
    switch (variant) {
        case 0: fn = (const void*)&atomics_kernel<0>; break;
        case 1: fn = (const void*)&atomics_kernel<1>; break;
        case 2: fn = (const void*)&atomics_kernel<2>; break;
        case 3: fn = (const void*)&votemix_kernel<false, false, 384>; break;
        case 4: fn = (const void*)&votemix_kernel<true, false, 384>; break;
        case 6: fn = (const void*)&votemix_kernel<false, true, 384>; break;
        case 7: fn = (const void*)&votemix_kernel<true, true, 384>; break;
        case 8: fn = (const void*)&votemix_kernel<true, true, 512>; break;
        default: fn = (const void*)&atomics_peak_kernel; break;
    }
    cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaEvent_t ev0, ev1;
    cudaEventCreate(&ev0); cudaEventCreate(&ev1);
    void* args[2] = {(void*)&iters, (void*)&sink};
    float ms = 0.0f;
    for (int rep = 0; rep < 3 && e == cudaSuccess; ++rep) {   // 2 warm-ups, the third is timed
        if (rep == 2) cudaEventRecord(ev0, 0);
        e = cudaLaunchKernel(fn, dim3(grid), dim3(threads), args, smem, 0);
        if (rep == 2) cudaEventRecord(ev1, 0);
    }
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e == cudaSuccess) cudaEventElapsedTime(&ms, ev0, ev1);
    cudaEventDestroy(ev0); cudaEventDestroy(ev1);
    cudaFree(sink);
    if (e != cudaSuccess) return HOUGH_ERR_CUDA;
    double per_thread = (variant <= 2 || variant == 5) ? 8.0 * (double)iters : 0.0;
    double total;
    if (variant <= 2 || variant == 5) {
        total = per_thread * (double)threads * (double)grid;
    } else {
        const int nwarps = threads / 32, n_stripes = nwarps / 3;
        total = (double)iters * 1024.0 * 192.0 * (double)grid * (n_stripes > 0 ? 1.0 : 0.0);   // lane-votes incl. padded lanes
    }
    *out_rate = total / ((double)ms * 1e-3);
    return HOUGH_OK;
}
