// hough_kernel.cuh -- the fused per-event kernel (sm_100a).
//
// One CTA (or one thread-block cluster of C CTAs that split the theta columns)
// per event: the launch has n_events * C CTAs and the hardware block scheduler
// deals them to the SM slots (no scratch, re-entrant across streams; the event
// loop below only iterates beyond 2^31 CTAs).  Per event:
//   H0/H1 stage hits -> conformal (u,v) in shared memory   PAPER.md:52-57 Eq. (1)
//   H2/H3 vote: lane = CPL theta columns, warp-uniform hit
//   H4    threshold + 3x3 local maximum -> peak bitmap
//   H5    raster-order peak list
//   H6    hit selection against the dilated peak bitmap
//   H7    stable compaction
// The exact fp32 operation order is DESIGN.md S1/S2 (one rounding per
// operation, no FMA contraction).  This file shares nothing with oracle/.
//
// Accumulator layout in shared memory: rho-major,
// A[k][word], so that a warp that owns 32 (or 64) adjacent theta columns hits
// 32 distinct banks whatever the rho bins are: votes are conflict-free by
// construction.  Local column jl = 64 G + 32 h + l  (pair G, half h, lane l):
//   u16: word G*32 + l of row k holds columns (h=0 | h=1) in its (low | high) half
//   u32: word (2G+h)*32 + l of row k
// Row n_rho is a trash row (one full pitch) that swallows the out-of-range votes and those of the padding columns.
// In the vote phase a warp owns a group of 32*CPL adjacent columns (CPL = 2, 4 or 6 per lane) and a
// stripe of the hits: one broadcast LDS.64 of (u,v) feeds CPL votes per lane.
//
// HOUGH_HOST_EMU (tests/simt_emu only): the same source is compiled by g++ against a SIMT shim (fibers, barriers, warp
// collectives, a per-CTA shared-memory buffer) so that the CPU tests can execute the kernel's LOGIC -- indexing, phase
// order, bounds -- against the oracle without a GPU.  The shim supplies the CUDA names; only the inline PTX below has
// a host restatement.  It is test infrastructure: nothing in the product path is built with it.
#pragma once
#ifndef HOUGH_HOST_EMU
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#define HOUGH_DYN_SMEM(name) extern __shared__ __align__(128) unsigned char name[]
#endif
#include <stdint.h>

#include "../../include/hough.h"

namespace hough {
namespace cg = cooperative_groups;

typedef unsigned long long ull;

// 1.5 * 2^23: adding it with round-toward-minus-infinity leaves floor(t) in the
// low mantissa bits for |t| < 2^22 (exact: the sum is representable up to the
// rounding that IS the floor).
#define HOUGH_MAGIC_F 12582912.0f
#define HOUGH_MAGIC_BITS 0x4B400000u
#define HOUGH_SEL_ROUND_BLOCKS 32   // clustered selection: hit blocks per CTA per round

// -DHOUGH_DEBUG_BOUNDS (libhough_b200_dbg.so, paper_2607_04067_b200/build.py): every shared-memory offset of the
// vote, H4, H5, H6 and H7 phases (and the compaction's global index) is checked against the plan's region sizes
// before use.  A violating access is SKIPPED (never performed, never traps) and the event's d_counts entry becomes
// {HOUGH_DBG_SENTINEL, phase}.  The release build compiles the checks away.
#define HOUGH_DBG_SENTINEL (-2)
enum { HB_STAGE = 1, HB_VOTE_FAST = 2, HB_VOTE_SLOW = 3, HB_H4 = 4, HB_H5 = 5, HB_H6_SETUP = 6, HB_KEEP = 7, HB_H7 = 8 };
#ifdef HOUGH_DEBUG_BOUNDS
#define HB_CHK(ok, phase) ((ok) ? true : ((dbg_viol = dbg_viol ? dbg_viol : (phase)), false))
#else
#define HB_CHK(ok, phase) (true)
#endif

struct KParams {
    const float2* xy;
    const int* off;
    int n_events;
    unsigned char* keep;
    hough_peak* peaks;
    int* counts;
    float2* kept_xy;
    int* kept_idx;
    unsigned* accum_dump;
    const float* cos_t;
    const float* sin_t;
    int n_theta, n_rho, threshold, window, max_peaks;
    float rho_max, inv, scale;
    float tame_bound;     // a hit is "tame" iff (|u|+|v|) <= tame_bound (then |t| < 2^17 at every column) ...
    float ftz_min;        // ... and u, v are each 0 or >= ftz_min in magnitude (then no product u*c, v*s is subnormal)
    int force_slow;       // 1: literal slow path for every hit
#ifdef HOUGH_DIAG
    int diag;             // bench-only build: 2 = skip the vote loops, 3 = skip everything after voting (outputs undefined)
#endif
    int csize;            // CTAs per event (cluster size)
    int cols_per_cta;     // theta columns owned by one CTA
    int n_groups;         // groups of 32*CPL columns per CTA
    int n_stripes;        // warps per group in the vote phase
    unsigned rcp_groups;  // (warp * rcp_groups) >> 16 == warp / n_groups for warp < 32 (checked by the planner)
    unsigned rcp_2s;      // (m * rcp_2s) >> 20 == m / (2 * n_stripes) for m <= chunk (checked by the planner)
    int vpr;              // uint4 vectors per accumulator row = pitch_b / 16
    int pitch_b;          // bytes per rho row of the accumulator (multiple of 128)
    int wpr;              // 32-bit words per bitmap row = ceil(n_rho / 32)
    int chunk;            // hits staged per pass
    int region_bytes;     // accumulator region (also reused after peak extraction)
    int pbm_off;          // peak bitmap [cols_per_cta][wpr]
    int pbm_bytes;
    int hb_off;           // hit buffer float2[chunk]
    int misc_off;         // 64 ints
    // post-extraction layout inside the accumulator region (byte offsets)
    int w8_off, w8_pitch, mcf_off, msf_off, colq_off, stash_off, cnt_off, gcnt_off;
    // options of the extended instantiation (EXT = true; readings Q18-Q20).
    // The default instantiation (EXT = false) never reads them.
    int peak_mode;        // 0: threshold + 3x3 local maximum; 1: relative threshold + iterative NMS
    int rel_permille;     // NMS: candidates need a >= ceil(rel_permille * A_max / 1000) (and >= threshold)
    int nms_radius;       // NMS: half-width of the suppressed neighbourhood
    int theta_wrap;       // column -1 is column n_theta-1 with the rho index mirrored
    int keep_mode;        // 0: (theta, rho) window; 1: distance to the candidate circle
    int circ_cap;         // distance filter: circles staged in the dead accumulator region
    int stage_mode;       // 0: coalesced float2 loads; 1: one cp.async.bulk per chunk into the hit buffer (north_star (1))
    int select_mode;      // H6: 0 scan of the marked columns per hit; 1 dense (window mask in the accumulator, vote mapping); 2 dense when many columns are marked
    int sched_mode;       // 0: one CTA per event; 1: a resident CTA steals not-yet-launched CTAs' events (cluster launch control)
    double keep_tol;      // distance filter tolerance, units of the hit coordinates
};

// Candidate circle of a peak (Eq. (2), with the conformal scale s of reading Q1; DESIGN.md readings
// Q14, Q15): rho_c = (k + 0.5) / inv - rho_max at the centre of the bin, centre = s (c_j, s_j) / (2 rho_c),
// r_c = s / (2 |rho_c|); fp64, one rounding per operation (the TU is built with -fmad=false), IEEE division.
__device__ __forceinline__ double rho_centre(int k, float inv, float rho_max) {
    return __dsub_rn(__ddiv_rn(__dadd_rn((double)k, 0.5), (double)inv), (double)rho_max);
}
__device__ __forceinline__ void circle_of(float cj, float sj, int k, float inv, float rho_max, float scale, double& x_c, double& y_c, double& r_c) {
    const double den = __dmul_rn(2.0, rho_centre(k, inv, rho_max)), s = (double)scale;
    x_c = __ddiv_rn(__dmul_rn(s, (double)cj), den);
    y_c = __ddiv_rn(__dmul_rn(s, (double)sj), den);
    r_c = __ddiv_rn(s, fabs(den));
}

// ---------------------------------------------------------------- small helpers
#ifdef HOUGH_HOST_EMU
inline void red_shared_add(unsigned saddr, unsigned v) { __atomic_fetch_add((unsigned*)emu::shared_ptr(saddr), v, __ATOMIC_RELAXED); }
inline void vote_add(unsigned saddr, unsigned v) { __atomic_fetch_add((unsigned*)emu::shared_ptr(saddr), v, __ATOMIC_RELAXED); }
inline void red_shared_or(unsigned saddr, unsigned v) { __atomic_fetch_or((unsigned*)emu::shared_ptr(saddr), v, __ATOMIC_RELAXED); }
#else
__device__ __forceinline__ void red_shared_add(unsigned saddr, unsigned v) {
    asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(saddr), "r"(v) : "memory");
}
// The vote proper.  No "memory" clobber: ordering against the zeroing stores and the later scan is
// given by the __syncthreads() around the vote phase, and the compiler stays free to hoist the
// hit loads of the next iterations above it.
__device__ __forceinline__ void vote_add(unsigned saddr, unsigned v) {
    asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(saddr), "r"(v));
}
__device__ __forceinline__ void red_shared_or(unsigned saddr, unsigned v) {
    asm volatile("red.shared.or.b32 [%0], %1;" ::"r"(saddr), "r"(v) : "memory");
}
#endif

// Bulk-copy staging (EXT, stage_mode 1; north_star subsystem (1), SURVEY.md section 7 "Bulk-copy alignment"): one
// cp.async.bulk (TMA engine, SASS UBLKCP) per chunk of hits, completion on an mbarrier.  `bar` and `dst` are
// shared-window addresses, `bytes` a multiple of 16, `src` 16-byte aligned.
#ifdef HOUGH_HOST_EMU
inline void mbar_init(unsigned, unsigned) {}
inline void fence_proxy_async() {}
inline void mbar_expect_tx(unsigned, unsigned) {}
EMU_NOSAN inline void bulk_copy_g2s(unsigned dst, const void* src, unsigned bytes, unsigned bar) {
    emu::bulk_check(dst, src, bytes);
    memcpy(emu::shared_ptr(dst), src, bytes);
    emu::mbar_complete(bar);
    emu::async_write(emu::shared_ptr(dst), bytes, bar);      // race check: written by the copy engine, visible through `bar`
}
inline bool mbar_try_wait(unsigned bar, unsigned parity) { return emu::mbar_wait_parity(bar, parity); }
inline void prefetch_l2_bulk(const void*, unsigned) {}
// cluster launch control: the emulator hands out the not-yet-launched CTAs of the grid (emu::clc_steal)
EMU_NOSAN inline void clc_try_cancel(unsigned resp, unsigned bar) {
    int* r = (int*)emu::shared_ptr(resp);
    const int id = emu::clc_steal();
    r[0] = id; r[1] = 0; r[2] = 0; r[3] = id >= 0 ? 1 : 0;
    emu::mbar_complete(bar);
    emu::async_write(r, 16, bar);                            // race check: written by the hardware, visible through `bar`
}
inline int clc_query(unsigned resp) {        // the stolen CTA's blockIdx.x, or -1 when nothing was left to steal
    const int* r = (const int*)emu::shared_ptr(resp);
    return r[3] ? r[0] : -1;
}
#else
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_copy_g2s(unsigned dst, const void* src, unsigned bytes, unsigned bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// L2 prefetch of a 16-byte aligned global range (a hint: no destination, no completion to wait for)
__device__ __forceinline__ void prefetch_l2_bulk(const void* src, unsigned bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}
// Blackwell cluster launch control (PTX ISA 8.6, sm_100): ask the hardware to cancel the launch of a CTA of this grid
// that has not started yet; the 16-byte answer lands in shared memory and completes 16 bytes on the mbarrier.
__device__ __forceinline__ void clc_try_cancel(unsigned resp, unsigned bar) {
    asm volatile("clusterlaunchcontrol.try_cancel.async.shared::cta.mbarrier::complete_tx::bytes.b128 [%0], [%1];"
                 ::"r"(resp), "r"(bar) : "memory");
}
// Decodes the answer: the cancelled CTA's blockIdx.x (this CTA now owns its work), or -1 when no CTA was left.
__device__ __forceinline__ int clc_query(unsigned resp) {
    unsigned ok, x;
    asm volatile("{\n\t.reg .pred p;\n\t.reg .b128 r;\n\tld.shared.b128 r, [%2];\n\t"
                 "clusterlaunchcontrol.query_cancel.is_canceled.pred.b128 p, r;\n\tselp.u32 %0, 1, 0, p;\n\tmov.u32 %1, 0;\n\t"
                 "@p clusterlaunchcontrol.query_cancel.get_first_ctaid::x.b32.b128 %1, r;\n\t}"
                 : "=r"(ok), "=r"(x) : "r"(resp) : "memory");
    return ok ? (int)x : -1;
}
__device__ __forceinline__ bool mbar_try_wait(unsigned bar, unsigned parity) {
    unsigned ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
#endif

// S1: d = fl(fl(x*x)+fl(y*y)); u = scale*fl(x/d); v = scale*fl(y/d).  Eq. (1).
__device__ __forceinline__ float2 conformal(float2 h, float scale) {
    float d = __fadd_rn(__fmul_rn(h.x, h.x), __fmul_rn(h.y, h.y));
    return make_float2(__fmul_rn(scale, __fdiv_rn(h.x, d)), __fmul_rn(scale, __fdiv_rn(h.y, d)));
}

// S2 for one (hit, theta column) pair, one rounding per operation, intrinsics that ptxas never contracts:
//   rho = fl(fl(u*c) + fl(v*s)); t = fl(fl(rho + rho_max) * inv); y = t + 1.5*2^23 rounded toward -inf.
// Returns the raw bits of y: (bits - HOUGH_MAGIC_BITS) as unsigned is < n_rho  <=>  0 <= t < n_rho, and
// then it IS floor(t) -- for every input, including NaN/inf/huge.
// This scalar form is exact for ANY hit; selection (H6) uses it.  The voting loop uses the packed form below,
// which takes the same number of issue slots (a packed fp32x2 instruction occupies two,
// profiles/r01_microbench_voteloop.md) but half the instructions and registers.
__device__ __forceinline__ unsigned bin_bits(float u, float v, float c, float s, float rho_max, float inv) {
    const float rho = __fadd_rn(__fmul_rn(u, c), __fmul_rn(v, s));
    const float t = __fmul_rn(__fadd_rn(rho, rho_max), inv);
    return __float_as_uint(__fadd_rd(t, HOUGH_MAGIC_F));
}

// Two columns at once with the packed fp32x2 instructions of sm_100 (FMUL2 / FADD2): the same six
// roundings per column as bin_bits, one instruction per PAIR of columns.  Every operation carries an
// explicit rounding mode.  The two products are computed with .ftz: ptxas contracts a plain
// mul.rn.f32x2 feeding an add.rn.f32x2 into FFMA2 (one rounding instead of two, seen with CUDA 12.9
// even under --fmad=false), and it cannot do so when the flush modes differ.  The flush itself never
// acts: the fast path only takes hits whose products with every non-zero table entry are normal
// (KParams::ftz_min); build.py rejects any FFMA2 in the SASS.
#ifdef HOUGH_HOST_EMU
inline ull pack2(float lo, float hi) { return (ull)__float_as_uint(lo) | ((ull)__float_as_uint(hi) << 32); }
// host restatement of the packed sequence, lane by lane, INCLUDING the flush-to-zero of the two products' inputs and
// results, so that a non-tame hit on the fast path would show up as a mismatch against the oracle
inline void bin_bits2(float u, float v, ull c2, ull s2, float rho_max, float inv, unsigned& b0, unsigned& b1) {
    unsigned out[2];
    for (int h = 0; h < 2; ++h) {
        const float c = __uint_as_float((unsigned)(c2 >> (32 * h))), s = __uint_as_float((unsigned)(s2 >> (32 * h)));
        const float p1 = emu::ftz(__fmul_rn(emu::ftz(u), emu::ftz(c))), p2 = emu::ftz(__fmul_rn(emu::ftz(v), emu::ftz(s)));
        const float t = __fmul_rn(__fadd_rn(__fadd_rn(p1, p2), rho_max), inv);
        out[h] = __float_as_uint(__fadd_rd(t, HOUGH_MAGIC_F));
    }
    b0 = out[0];
    b1 = out[1];
}
#else
__device__ __forceinline__ ull pack2(float lo, float hi) {
    ull r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void bin_bits2(float u, float v, ull c2, ull s2, float rho_max, float inv, unsigned& b0, unsigned& b1) {
    const ull u2 = pack2(u, u), v2 = pack2(v, v), rm2 = pack2(rho_max, rho_max), inv2 = pack2(inv, inv);
    const ull mg2 = pack2(HOUGH_MAGIC_F, HOUGH_MAGIC_F);
    ull p1, p2, rho, sh, t, y;
    asm("mul.rn.ftz.f32x2 %0, %1, %2;" : "=l"(p1) : "l"(u2), "l"(c2));
    asm("mul.rn.ftz.f32x2 %0, %1, %2;" : "=l"(p2) : "l"(v2), "l"(s2));
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(rho) : "l"(p1), "l"(p2));
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(sh) : "l"(rho), "l"(rm2));
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(t) : "l"(sh), "l"(inv2));
    asm("add.rm.f32x2 %0, %1, %2;" : "=l"(y) : "l"(t), "l"(mg2));
    asm("mov.b64 {%0, %1}, %2;" : "=r"(b0), "=r"(b1) : "l"(y));
}
#endif

// S2, scalar and literal (the slow exact path and the reference for the trick).  Returns k or -1.
__device__ __forceinline__ int bin_exact(float u, float v, float c, float s, float rho_max, float inv, int n_rho) {
    float rho = __fadd_rn(__fmul_rn(u, c), __fmul_rn(v, s));
    float t = __fmul_rn(__fadd_rn(rho, rho_max), inv);
    if (t >= 0.0f && t < (float)n_rho) return (int)t;
    return -1;
}

// Exclusive scan of one int per thread over the CTA; `total` is returned to every thread.
// wsum: 33 ints of shared scratch.  Contains two __syncthreads(); may be called back to back.
__device__ __forceinline__ int block_exscan(int v, int* wsum, int& total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = (blockDim.x + 31) >> 5;
    int inc = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        int o = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += o;
    }
    __syncwarp();                        // a previous call's reads of wsum[warp] by this warp's lanes come before the write
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        int w = lane < nwarps ? wsum[lane] : 0;
        int winc = w;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            int o = __shfl_up_sync(0xffffffffu, winc, d);
            if (lane >= d) winc += o;
        }
        wsum[lane] = winc - w;
        if (lane == 31) wsum[32] = winc;
    }
    __syncthreads();
    total = wsum[32];
    int r = wsum[warp] + inc - v;
    return r;
}

template <bool ACC16>
__device__ __forceinline__ unsigned cell_word_off(int jl) {   // word index within a rho row
    int g = jl >> 6, h = (jl >> 5) & 1, l = jl & 31;
    return ACC16 ? (unsigned)(g * 32 + l) : (unsigned)((2 * g + h) * 32 + l);
}

template <bool ACC16>
__device__ __forceinline__ unsigned cell_from(const unsigned char* acc, int pitch_b, int jl, int k) {
    unsigned w = *(const unsigned*)(acc + (size_t)k * pitch_b + 4u * cell_word_off<ACC16>(jl));
    if (ACC16) return (w >> (16 * ((jl >> 5) & 1))) & 0xFFFFu;
    return w;
}

// ---------------------------------------------------------------- the kernel
template <bool ACC16, bool CL, int CPL, bool EXT = false>
__global__ void __launch_bounds__(1024, 1) hough_event_kernel(const __grid_constant__ KParams p) {
    HOUGH_DYN_SMEM(smem);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nthreads = blockDim.x, nwarps = nthreads >> 5;

    unsigned rank = 0;
    if (CL) rank = cg::this_cluster().block_rank();
    const int C = p.csize;
    int cluster_id = blockIdx.x, n_clusters = gridDim.x;
    if (CL) {   // the hardware's own cluster index: no division by the run-time cluster size
#ifdef HOUGH_HOST_EMU
        cluster_id = emu::cluster_id();
        n_clusters = emu::n_clusters();
#else
        asm("mov.u32 %0, %%clusterid.x;" : "=r"(cluster_id));
        asm("mov.u32 %0, %%nclusterid.x;" : "=r"(n_clusters));
#endif
    }

    unsigned char* acc = smem;                                  // accumulator region
    unsigned* pbm = (unsigned*)(smem + p.pbm_off);              // peak bitmap [cols_per_cta][wpr]
    float2* const hb0 = (float2*)(smem + p.hb_off);             // staged (u,v); H4 reuses its tail as the candidate list
    float2* hb = hb0;                                           // (bulk staging shifts it by one hit for odd event starts)
    int* misc = (int*)(smem + p.misc_off);                      // [0..32] scan scratch, [40] peak total, [41] marked count, [42] candidates
    const unsigned acc_s = (unsigned)__cvta_generic_to_shared(acc);

    const int col0 = (int)rank * p.cols_per_cta;
    int ncols = p.n_theta - col0;
    if (ncols > p.cols_per_cta) ncols = p.cols_per_cta;
    if (ncols < 0) ncols = 0;

    // ---- vote-phase lane constants: this lane owns local columns 32*(g*CPL+q) + lane, q < CPL, of group g
    const int stripe = (int)(((unsigned)warp * p.rcp_groups) >> 16), g = warp - stripe * p.n_groups;
    const unsigned pitch = (unsigned)p.pitch_b;
    const unsigned limit = (unsigned)p.n_rho * pitch;
    // Word of (k, column q of this lane) = k*pitch + wbase + stride*(q or q/2): one base register, the rest is an
    // immediate of the ATOMS.  u16: columns q, q+1 share a word (low | high half), words of a lane are 128 B apart;
    // u32: one word per column, 128 B apart.  Out-of-range bins (including every wrapped negative) are clamped to
    // the lane's word of the trash row BEFORE the immediate is added, so they stay inside the trash row.
    const unsigned wbase = ACC16 ? (unsigned)(g * (CPL / 2) * 128 + 4 * lane) : (unsigned)(g * CPL * 128 + 4 * lane);
    const unsigned lc0 = wbase - HOUGH_MAGIC_BITS * pitch;     // rel = bits * pitch + lc0
    const unsigned trash0 = limit + wbase;
    ull c2q[CPL / 2], s2q[CPL / 2];
#pragma unroll
    for (int q = 0; q < CPL; q += 2) {
        const int j0 = 32 * (g * CPL + q) + lane, j1 = j0 + 32;
        // a padding column gets a NaN table entry: its t is NaN at every hit and its votes end in the trash row
        const float qnan = __uint_as_float(0x7FC00000u);
        const float c0 = j0 < ncols ? p.cos_t[col0 + j0] : qnan, s0 = j0 < ncols ? p.sin_t[col0 + j0] : qnan;
        const float c1 = j1 < ncols ? p.cos_t[col0 + j1] : qnan, s1 = j1 < ncols ? p.sin_t[col0 + j1] : qnan;
        c2q[q / 2] = pack2(c0, c1);
        s2q[q / 2] = pack2(s0, s1);
    }
    const float rho_max = p.rho_max, inv = p.inv;

    const int zero_vec = (p.region_bytes + p.pbm_bytes) >> 4;   // pbm follows the region; both 16-B multiples

    // EXT, bulk staging: the hit buffer keeps two spare slots (a chunk's source range is aligned down and up by one hit)
    const bool bulk = EXT && p.stage_mode == 1;
    const int chunk = bulk ? p.chunk - 2 : p.chunk;
    const unsigned bar_s = (unsigned)__cvta_generic_to_shared(misc + 52), hb0_s = (unsigned)__cvta_generic_to_shared(hb0);
    const int total_hits = (bulk || (EXT && !CL && p.sched_mode == 1)) ? __shfl_sync(0xffffffffu, p.off[p.n_events], 0) : 0;
    unsigned bar_phase = 0;
    if (bulk) {
        if (tid == 0) mbar_init(bar_s, 1u);
        __syncthreads();
    }
    // Issues the copy of chunk [cbeg, cbeg + m) of the event that starts at hit `beg` (thread 0 only).  The 16-byte
    // aligned source range starts at the even hit index at or below the chunk's first hit and holds an even number of
    // hits; it may include one hit of a neighbouring event on either side, but never reaches past the batch's last hit:
    // there the odd last hit is left to a plain load (tail_plain).  Returns the bytes in flight.
    auto bulk_issue = [&](int beg, int cbeg, int m, int& hshift, bool& tail_plain) -> unsigned {
        const int g0 = beg + cbeg;
        hshift = g0 & 1;
        int cnt = (hshift + m + 1) & ~1;
        tail_plain = false;
        if (g0 - hshift + cnt > total_hits) { cnt -= 2; tail_plain = true; }
        const unsigned bytes = 8u * (unsigned)cnt;
        if (tid == 0 && cnt > 0 && cnt <= p.chunk) {      // (cnt <= m + 2 <= p.chunk by construction)
            fence_proxy_async();           // earlier generic-proxy accesses of the buffer are ordered before the async write
            mbar_expect_tx(bar_s, bytes);
            bulk_copy_g2s(hb0_s, (const void*)(p.xy + (g0 - hshift)), bytes, bar_s);
        }
        return bytes;
    };

    // EXT, scheduler mode 1 (one CTA per event only): persistent CTAs with hardware work stealing.  The launch is the same
    // one-CTA-per-event grid; a resident CTA asks, at the start of every event, to cancel the launch of a CTA that has not
    // started yet (cluster launch control) and, when its own event is done, takes over the cancelled CTA's event: the
    // per-CTA prologue above (table loads, lane constants) then runs once per resident CTA, the block scheduler still
    // balances the events, and no scratch memory or counter is needed (the handle stays re-entrant).  The answer arrives
    // long before it is needed; when it names a next event, that event's hits are prefetched into L2 while this event's
    // H4-H7 run.  A failed request (nothing left to launch) ends the loop: no request may follow a failed one.
    const bool steal = EXT && !CL && p.sched_mode == 1;
    const unsigned clc_bar_s = (unsigned)__cvta_generic_to_shared(misc + 56), clc_resp_s = (unsigned)__cvta_generic_to_shared(misc + 60);
    unsigned clc_phase = 0;
    if (steal) {
        if (tid == 0) mbar_init(clc_bar_s, 1u);
        __syncthreads();
    }
    auto next_event = [&](int e) -> int {
        if (!steal) return e + n_clusters;
        __syncthreads();                           // every thread is done with event e (and with the previous answer)
        if (tid == 0) {
            bool done = false;
            for (int spin = 0; spin < (1 << 24) && !done; ++spin) done = mbar_try_wait(clc_bar_s, clc_phase);   // bounded: never a hang
            misc[54] = done ? clc_query(clc_resp_s) : -1;
        }
        clc_phase ^= 1u;
        __syncthreads();
        const int nxt = misc[54];
        return nxt >= 0 ? nxt : p.n_events;        // p.n_events ends the loop
    };

    for (int e = cluster_id; e < p.n_events; e = next_event(e)) {
        if (steal && tid == 0) {                   // this event's request: answered while the event is processed
            fence_proxy_async();                   // the previous answer was read through the generic proxy
            mbar_expect_tx(clc_bar_s, 16u);
            clc_try_cancel(clc_resp_s, clc_bar_s);
        }
        // shfl from lane 0 = "this value is warp-uniform" for ptxas (keeps the event loop in uniform control flow)
        const int beg = __shfl_sync(0xffffffffu, p.off[e], 0);
        const int n = __shfl_sync(0xffffffffu, p.off[e + 1], 0) - beg;
        if (ACC16 && n > 65535) {   // a u16 cell could wrap: refuse the event (uniform over the cluster)
            if (rank == 0 && tid == 0) { p.counts[2 * e] = -1; p.counts[2 * e + 1] = -1; }
            continue;
        }

        const bool single = n <= chunk;      // the whole event is staged at once: (u,v) stay in hb until selection
        int dbg_viol = 0;                    // HOUGH_DEBUG_BOUNDS: first phase whose offset check failed (else unused)
        (void)dbg_viol;
        const unsigned acc_end = (unsigned)(p.n_rho + 1) * (unsigned)p.pitch_b;   // accumulator incl. the trash row
        (void)acc_end;

        // the first two hits of this thread are requested before the zeroing stores, which then overlap the latency
        float2 pre0 = make_float2(1.0f, 0.0f), pre1 = pre0;
        if (!bulk && tid < n) pre0 = __ldg(&p.xy[beg + tid]);
        if (!bulk && tid + nthreads < n) pre1 = __ldg(&p.xy[beg + tid + nthreads]);
        // bulk staging: the first chunk's copy is in flight while the accumulator is zeroed
        int hshift = 0;
        bool tail_plain = false;
        unsigned in_flight = 0;
        if (bulk && n > 0) in_flight = bulk_issue(beg, 0, min(chunk, n), hshift, tail_plain);

        // ---- zero accumulator + peak bitmap
        {
            uint4* z = (uint4*)smem;
            const uint4 zz = make_uint4(0, 0, 0, 0);
            for (int i = tid; i < zero_vec; i += nthreads) z[i] = zz;
            if (tid == 0) { misc[42] = 0; misc[33] = 1; }      // [33]: every chunk of the event took the packed fast path so far
        }

        // ---- H0-H3: stage, transform, vote (chunked)
        for (int cbeg = 0; cbeg < n; cbeg += chunk) {
            const int m = min(chunk, n - cbeg);
            int tame = 1;
            if (bulk) {
                if (cbeg > 0) in_flight = bulk_issue(beg, cbeg, m, hshift, tail_plain);   // (the previous chunk ended with a barrier)
                hb = hb0 + hshift;               // raw hit i of the chunk lands in slot hshift + i: converted in place below
                if (in_flight) {
                    bool done = false;
                    for (int spin = 0; spin < (1 << 24) && !done; ++spin) done = mbar_try_wait(bar_s, bar_phase);   // bounded: never a hang
                    bar_phase ^= 1u;
                    if (!done) tail_plain = true, in_flight = 0;      // give up on the copy: every hit comes from a plain load
                }
            }
            for (int i = tid; i < m; i += nthreads) {
                float2 h;
                if (bulk) h = (in_flight && !(tail_plain && i == m - 1)) ? hb[i] : __ldg(&p.xy[beg + cbeg + i]);
                else if (cbeg == 0 && i == tid) h = pre0;
                else if (cbeg == 0 && i == tid + nthreads) h = pre1;
                else h = __ldg(&p.xy[beg + cbeg + i]);
                float2 uv = conformal(h, p.scale);
                if (HB_CHK(hshift + i < p.chunk, HB_STAGE)) hb[i] = uv;
                const float au = fabsf(uv.x), av = fabsf(uv.y);
                tame &= (__fadd_rn(au, av) <= p.tame_bound) ? 1 : 0;                        // false for NaN/inf
                tame &= ((au >= p.ftz_min || au == 0.0f) && (av >= p.ftz_min || av == 0.0f)) ? 1 : 0;
            }
            const int all_tame = __shfl_sync(0xffffffffu, __syncthreads_and(tame) && !p.force_slow, 0);
            if (tid == 0 && !all_tame) misc[33] = 0;      // (kept in shared memory: a register live across the voting loop costs it a reload)
            // Every warp votes (nwarps == n_groups * n_stripes).  Hits are dealt in rounds of 2*S:
            // the full rounds have a warp-uniform trip count, which keeps the loop in uniform
            // control flow (shared-window base in a uniform register, ATOMS [R+UR] addressing).
            const int S = p.n_stripes;
            const int R = (int)(((unsigned)m * p.rcp_2s) >> 20);   // m / (2 * S)
#ifdef HOUGH_DIAG
            if (p.diag == 2) {
            } else
#endif
            if (all_tame) {
                // out-of-range votes (rel >= limit, including every wrapped negative) land in the lane's own
                // word of the trash row: no predicate, no branch, no conflict
                auto vote_hit = [&](const float2 uv) {
#pragma unroll
                    for (int q = 0; q < CPL; q += 2) {
                        unsigned b0, b1;
                        bin_bits2(uv.x, uv.y, c2q[q / 2], s2q[q / 2], rho_max, inv, b0, b1);
                        const unsigned rel0 = min(b0 * pitch + lc0, trash0);
                        const unsigned rel1 = min(b1 * pitch + lc0, trash0);
                        if (ACC16) {
                            if (HB_CHK(rel0 + 128 * (q / 2) + 4 <= acc_end, HB_VOTE_FAST)) atomicAdd((unsigned*)(acc + rel0 + 128 * (q / 2)), 1u);
                            if (HB_CHK(rel1 + 128 * (q / 2) + 4 <= acc_end, HB_VOTE_FAST)) atomicAdd((unsigned*)(acc + rel1 + 128 * (q / 2)), 0x10000u);
                        } else {
                            if (HB_CHK(rel0 + 128 * q + 4 <= acc_end, HB_VOTE_FAST)) atomicAdd((unsigned*)(acc + rel0 + 128 * q), 1u);
                            if (HB_CHK(rel1 + 128 * (q + 1) + 4 <= acc_end, HB_VOTE_FAST)) atomicAdd((unsigned*)(acc + rel1 + 128 * (q + 1)), 1u);
                        }
                    }
                };
                for (int r = 0; r < R; ++r) {
                    const float2 uv0 = hb[(2 * r) * S + stripe], uv1 = hb[(2 * r + 1) * S + stripe];
                    vote_hit(uv0);
                    vote_hit(uv1);
                }
                for (int i = 2 * R * S + stripe; i < m; i += S) vote_hit(hb[i]);
            } else {
                // exact slow path: literal S2 with float compares (degenerate hits: NaN, inf, r < ~0.3 mm)
                for (int i = stripe; i < m; i += S) {
                    const float2 uv = hb[i];
                    for (int q = 0; q < CPL; ++q) {
                        const int jl = 32 * (g * CPL + q) + lane;
                        if (jl >= ncols) continue;
                        const int k = bin_exact(uv.x, uv.y, p.cos_t[col0 + jl], p.sin_t[col0 + jl], p.rho_max, p.inv, p.n_rho);
                        if (k >= 0 && HB_CHK((unsigned)k * pitch + 4u * cell_word_off<ACC16>(jl) + 4 <= limit, HB_VOTE_SLOW))
                            red_shared_add(acc_s + (unsigned)k * pitch + 4u * cell_word_off<ACC16>(jl), (ACC16 && (q & 1)) ? 0x10000u : 1u);
                    }
                }
            }
            __syncthreads();
        }
        if (n == 0) __syncthreads();         // no staging barrier ran: order the zeroing before the scan
        if (CL) cg::this_cluster().sync();   // (A) every CTA's columns are complete

        // scheduler mode 1: if the answer to this event's request is already there, pull the next event's hits into L2
        // now, under this event's H4-H7 (a hint only; the 16-byte aligned range never reaches past the batch's last hit)
        if (steal && tid == 0 && mbar_try_wait(clc_bar_s, clc_phase)) {
            const int nxt = clc_query(clc_resp_s);
            if (nxt >= 0 && nxt < p.n_events) {
                const int b0 = p.off[nxt] & ~1, b1 = min((p.off[nxt + 1] + 1) & ~1, total_hits & ~1);
                if (b1 > b0) prefetch_l2_bulk((const void*)(p.xy + b0), 8u * (unsigned)(b1 - b0));
            }
        }

#ifdef HOUGH_DIAG
        if (p.diag == 3) { __syncthreads(); continue; }
#endif

        // ---- optional accumulator dump (parity / debugging; never timed)
        if (p.accum_dump) {
            unsigned* dst = p.accum_dump + ((size_t)e * p.n_theta + col0) * p.n_rho;
            const int cells = ncols * p.n_rho;
            for (int idx = tid; idx < cells; idx += nthreads) {
                int jl = idx / p.n_rho, k = idx - jl * p.n_rho;
                if (HB_CHK((unsigned)k * pitch + 4u * cell_word_off<ACC16>(jl) + 4 <= limit, HB_H4)) dst[idx] = cell_from<ACC16>(acc, p.pitch_b, jl, k);
            }
        }

        int n_stored;
        if (EXT && p.peak_mode == 1) {
            // ---- N2: threshold relative to the global maximum + iterative "extract the most
            // significant peak, suppress its neighbourhood" (reading Q18).
            // rowkey[k] = best cell of this CTA's columns in rho row k as (votes << 32) | (0xFFFF - j) << 16 | (0xFFFF - k):
            // the maximum over keys is the largest count and, among equals, the raster-first cell.  All warps build the
            // row keys; the extraction loop costs a few hundred cycles per peak (2R+1 rows to refresh).
            ull* rowkey = (ull*)pbm;      // the peak bitmap is unused in this mode; the planner sizes it for n_rho keys
            auto warp_max = [&](ull best) -> ull {
#pragma unroll
                for (int d = 16; d >= 1; d >>= 1) {
                    const ull o = __shfl_xor_sync(0xffffffffu, best, d);
                    if (o > best) best = o;
                }
                return best;
            };
            auto row_best = [&](int k) -> ull {
                ull best = 0;
                for (int jl = lane; jl < ncols; jl += 32) {
                    if (!HB_CHK((unsigned)k * pitch + 4u * cell_word_off<ACC16>(jl) + 4 <= limit, HB_H4)) continue;
                    const unsigned a = cell_from<ACC16>(acc, p.pitch_b, jl, k);
                    const ull key = ((ull)a << 32) | ((ull)(0xFFFFu - (unsigned)(col0 + jl)) << 16) | (ull)(0xFFFFu - (unsigned)k);
                    if (a != 0u && key > best) best = key;
                }
                return warp_max(best);
            };
            for (int k = warp; k < p.n_rho; k += nwarps) {
                const ull b = row_best(k);
                if (lane == 0 && HB_CHK(8 * k + 8 <= p.pbm_bytes, HB_H4)) rowkey[k] = b;
            }
            __syncthreads();
            auto local_best = [&]() -> ull {      // whole warp: best key over this CTA's rows
                ull best = 0;
                for (int k = lane; k < p.n_rho; k += 32)
                    if (HB_CHK(8 * k + 8 <= p.pbm_bytes, HB_H4)) { const ull b = rowkey[k]; if (b > best) best = b; }
                return warp_max(best);
            };
            const int R = p.nms_radius, side = 2 * R + 1;
            // whole warp: zero the (2R+1)^2 neighbourhood of (j, k) -- the cells this CTA owns -- and refresh the keys of
            // the rows that changed (and of their mirrors when the neighbourhood crosses the theta seam)
            auto suppress = [&](int j, int k) {
                for (int idx = lane; idx < side * side; idx += 32) {
                    int jj = j + idx / side - R, kk = k + idx % side - R;
                    if (kk < 0 || kk >= p.n_rho) continue;
                    if (jj < 0 || jj >= p.n_theta) {
                        if (!p.theta_wrap) continue;
                        while (jj < 0) { jj += p.n_theta; kk = p.n_rho - 1 - kk; }
                        while (jj >= p.n_theta) { jj -= p.n_theta; kk = p.n_rho - 1 - kk; }
                    }
                    const int jl = jj - col0;
                    if (jl < 0 || jl >= ncols) continue;       // another CTA of the cluster owns this column
                    const unsigned woff = (unsigned)kk * pitch + 4u * cell_word_off<ACC16>(jl);
                    if (!HB_CHK(woff + 4 <= limit, HB_H4)) continue;
                    const unsigned mask = ACC16 ? (0xFFFFu << (16 * ((jl >> 5) & 1))) : 0xFFFFFFFFu;
                    atomicAnd((unsigned*)(acc + woff), ~mask);     // two columns share a u16 word: clear one half atomically
                }
                const bool seam = p.theta_wrap && (j - R < 0 || j + R >= p.n_theta);
                __syncwarp();
                for (int kk = k - R; kk <= k + R; ++kk) {
                    if (kk < 0 || kk >= p.n_rho) continue;
                    const ull b = row_best(kk);
                    if (lane == 0) rowkey[kk] = b;
                    if (seam) {
                        const ull bm = row_best(p.n_rho - 1 - kk);
                        if (lane == 0) rowkey[p.n_rho - 1 - kk] = bm;
                    }
                }
                __syncwarp();
            };
            auto thr_of = [&](ull first_best) -> ull {      // reading Q18: max(threshold, ceil(permille * A_max / 1000))
                const ull rel = ((ull)p.rel_permille * (ull)(unsigned)(first_best >> 32) + 999ull) / 1000ull;
                return (ull)p.threshold > rel ? (ull)p.threshold : rel;
            };
            int n_found = 0;
            if (!CL) {
                // one CTA holds the whole accumulator: warp 0 runs the extraction loop alone, no block barrier per peak
                if (warp == 0) {
                    ull best = local_best();
                    const ull thr_eff = thr_of(best);
                    for (;;) {
                        const unsigned a = (unsigned)(best >> 32);
                        if (a == 0u || (ull)a < thr_eff) break;
                        const int j = 0xFFFF - (int)((best >> 16) & 0xFFFFull), k = 0xFFFF - (int)(best & 0xFFFFull);
                        if (lane == 0 && n_found < p.max_peaks) {
                            hough_peak pk;
                            pk.theta_bin = (uint16_t)j; pk.rho_bin = (uint16_t)k; pk.votes = a;
                            p.peaks[(size_t)e * p.max_peaks + n_found] = pk;
                        }
                        ++n_found;
                        suppress(j, k);
                        best = local_best();
                    }
                    if (lane == 0) misc[43] = n_found;
                }
                __syncthreads();
                n_found = misc[43];
            } else {
                // theta columns are split over the cluster: every iteration each CTA's warp 0 publishes its local best
                // (double-buffered slot), one cluster.sync, every CTA reduces the C slots over DSMEM to the SAME global
                // best and takes the same decision; each CTA suppresses the cells it owns.  One cluster barrier per peak.
                ull* slot = (ull*)(misc + 44);      // [2] local best of this CTA, by iteration parity (remote-readable)
                ull* gbest = (ull*)(misc + 48);     // [2] the cluster's best, by iteration parity
                ull thr_eff = 0;
                for (int it = 0;; ++it) {
                    if (warp == 0) {
                        const ull lb = local_best();
                        if (lane == 0) slot[it & 1] = lb;
                    }
                    cg::this_cluster().sync();
                    if (warp == 0) {
                        ull v = 0;
                        if (lane < C) v = *(const ull*)cg::this_cluster().map_shared_rank((void*)&slot[it & 1], lane);
                        v = warp_max(v);
                        if (lane == 0) gbest[it & 1] = v;
                    }
                    __syncthreads();
                    const ull best = gbest[it & 1];
                    if (it == 0) thr_eff = thr_of(best);
                    const unsigned a = (unsigned)(best >> 32);
                    if (a == 0u || (ull)a < thr_eff) break;      // the same value in every thread of every CTA
                    const int j = 0xFFFF - (int)((best >> 16) & 0xFFFFull), k = 0xFFFF - (int)(best & 0xFFFFull);
                    if (rank == 0 && tid == 0 && n_found < p.max_peaks) {
                        hough_peak pk;
                        pk.theta_bin = (uint16_t)j; pk.rho_bin = (uint16_t)k; pk.votes = a;
                        p.peaks[(size_t)e * p.max_peaks + n_found] = pk;
                    }
                    ++n_found;
                    if (warp == 0) suppress(j, k);
                }
                __threadfence();
                cg::this_cluster().sync();   // rank 0's stored peaks are visible cluster-wide; no CTA leaves while its slot may be read
            }
            if (rank == 0 && tid == 0) p.counts[2 * e] = n_found;
            n_stored = min(n_found, p.max_peaks);
        } else {
        // ---- H4: threshold + 3x3 local maximum -> peak bitmap (reading Q8)
        {
            // 3x3 test of one cell (reading Q8).  Branch-free: every neighbour is loaded from a clamped (always
            // valid) address and replaced by 0 when it lies outside the array, so the eight loads are independent.
            auto test_peak = [&](int jl, int k, unsigned a) {
                const int j = col0 + jl;
                const int km = max(k - 1, 0), kp1 = min(k + 1, p.n_rho - 1);
                const bool vkm = k > 0, vkp = k + 1 < p.n_rho;
                unsigned nb[3][3];
#pragma unroll
                for (int dj = -1; dj <= 1; ++dj) {
                    int jj = j + dj;
                    bool vj = jj >= 0 && jj < p.n_theta;
                    bool mir = false;       // EXT, theta wrap (reading Q19): column -1 is column n_theta-1 read upside down
                    if (EXT && p.theta_wrap && !vj) { jj += jj < 0 ? p.n_theta : -p.n_theta; mir = true; vj = true; }
                    const int jc = min(max(jj, 0), p.n_theta - 1);
                    const unsigned char* base = acc;
                    int jcl = jc;
                    if (CL) {
                        const int owner = jc / p.cols_per_cta;
                        jcl = jc - owner * p.cols_per_cta;
                        if (owner != (int)rank) base = (const unsigned char*)cg::this_cluster().map_shared_rank((void*)acc, owner);
                    }
                    const unsigned char* colp = base + 4u * cell_word_off<ACC16>(jcl);
                    const int sh = ACC16 ? 16 * ((jcl >> 5) & 1) : 0;
                    const int r0 = (EXT && mir) ? p.n_rho - 1 - km : km, r1 = (EXT && mir) ? p.n_rho - 1 - k : k,
                              r2 = (EXT && mir) ? p.n_rho - 1 - kp1 : kp1;
                    const bool in = HB_CHK(jcl >= 0 && jcl < p.cols_per_cta && min(r0, r2) >= 0 && max(r0, r2) < p.n_rho &&
                                           (unsigned)max(r0, r2) * pitch + 4u * cell_word_off<ACC16>(jcl) + 4 <= limit, HB_H4);
                    const unsigned w0 = in ? *(const unsigned*)(colp + (size_t)r0 * p.pitch_b) : 0u;
                    const unsigned w1 = in ? *(const unsigned*)(colp + (size_t)r1 * p.pitch_b) : 0u;
                    const unsigned w2 = in ? *(const unsigned*)(colp + (size_t)r2 * p.pitch_b) : 0u;
                    const unsigned msk = ACC16 ? 0xFFFFu : 0xFFFFFFFFu;
                    nb[dj + 1][0] = (vj && vkm) ? ((w0 >> sh) & msk) : 0u;
                    nb[dj + 1][1] = vj ? ((w1 >> sh) & msk) : 0u;
                    nb[dj + 1][2] = (vj && vkp) ? ((w2 >> sh) & msk) : 0u;
                }
                // strictly greater than the neighbours that precede in raster order, >= those that follow
                const bool ok = a > nb[0][0] && a > nb[0][1] && a > nb[0][2] && a > nb[1][0] &&
                                a >= nb[1][2] && a >= nb[2][0] && a >= nb[2][1] && a >= nb[2][2];
                if (ok && HB_CHK(jl >= 0 && k >= 0 && 4 * (jl * p.wpr + (k >> 5)) + 4 <= p.pbm_bytes, HB_H4))
                    red_shared_or((unsigned)__cvta_generic_to_shared(&pbm[jl * p.wpr + (k >> 5)]), 1u << (k & 31));
            };
            // Pass 1 streams the accumulator as uint4 and lists the VECTORS that hold a cell >= threshold (the list
            // lives in the part of the hit buffer without staged (u,v)); pass 2 gives every cell of a listed vector
            // its own thread.  A vector that does not fit the list is handled on the spot, so the list size never
            // decides the result.
            unsigned* vlist = (unsigned*)(hb + (single ? n : 0));
            const int vcap = 2 * (chunk - (single ? n : 0));
            const unsigned thr = (unsigned)p.threshold;
            const int vpr = p.vpr;
            constexpr int CELLS = ACC16 ? 8 : 4;               // cells per uint4
            auto test_cell = [&](int v, int c) {
                const int k = v / vpr, wv = v - k * vpr;
                const int wi = 4 * wv + (ACC16 ? (c >> 1) : c);  // word index within the row
                if (!HB_CHK(v >= 0 && k < p.n_rho && (unsigned)k * pitch + 4u * wi + 4 <= limit, HB_H4)) return;
                const unsigned word = *(const unsigned*)(acc + (size_t)k * p.pitch_b + 4u * wi);
                // u16: word G*32 + l holds columns 64G + l (low half) and 64G + 32 + l (high half); u32: word index IS the column
                const int jl = ACC16 ? 64 * (wi >> 5) + (wi & 31) + 32 * (c & 1) : wi;
                const unsigned a = ACC16 ? ((word >> (16 * (c & 1))) & 0xFFFFu) : word;
                if (a >= thr && jl < ncols) test_peak(jl, k, a);   // padding columns never hold votes; belt and braces
            };
            const int n_vec = p.n_rho * vpr;
            const uint4* acc4 = (const uint4*)acc;
            const unsigned thr2 = thr | (thr << 16);
            const bool thr_fits = !ACC16 || thr <= 0xFFFFu;     // a u16 cell can never reach a larger threshold
            // does any cell of the vector reach the threshold?  (u16: packed 3-input max, then one packed compare)
            auto vec_any = [&](const uint4& w) -> bool {
                if (ACC16) {
                    bool hi, lo;
                    const unsigned mx = __vimax3_u16x2(__vimax3_u16x2(w.x, w.y, w.z), w.w, 0u);
                    (void)__vibmax_u16x2(mx, thr2, &hi, &lo);   // hi/lo: that half of mx is >= thr
                    return (hi || lo) && thr_fits;
                }
                return __vimax3_u32(__vimax3_u32(w.x, w.y, w.z), w.w, 0u) >= thr;
            };
            auto scan_vec = [&](int v, const uint4& w) {
                if (!vec_any(w)) return;
                const int pos = atomicAdd(&misc[42], 1);
                if (pos < vcap) {
                    if (HB_CHK((hshift + (single ? n : 0)) * 8 + 4 * pos + 4 <= 8 * p.chunk, HB_H4)) vlist[pos] = (unsigned)v;
                    return;
                }
#pragma unroll 1
                for (int c = 0; c < CELLS; ++c) test_cell(v, c);
            };
            int v = tid;
            for (; v + 3 * nthreads < n_vec; v += 4 * nthreads) {   // four vectors per trip, one test
                if (!HB_CHK(16u * (unsigned)(v + 3 * nthreads + 1) <= limit, HB_H4)) continue;
                const uint4 w0 = acc4[v], w1 = acc4[v + nthreads], w2 = acc4[v + 2 * nthreads], w3 = acc4[v + 3 * nthreads];
                bool any4;                                         // max over the 16 words: eight 3-input max, one compare
                if (ACC16) {
                    unsigned m = __vimax3_u16x2(w0.x, w0.y, w0.z);
                    m = __vimax3_u16x2(m, w0.w, w1.x); m = __vimax3_u16x2(m, w1.y, w1.z); m = __vimax3_u16x2(m, w1.w, w2.x);
                    m = __vimax3_u16x2(m, w2.y, w2.z); m = __vimax3_u16x2(m, w2.w, w3.x); m = __vimax3_u16x2(m, w3.y, w3.z);
                    m = __vimax3_u16x2(m, w3.w, 0u);
                    bool hi, lo;
                    (void)__vibmax_u16x2(m, thr2, &hi, &lo);
                    any4 = (hi || lo) && thr_fits;
                } else {
                    unsigned m = __vimax3_u32(w0.x, w0.y, w0.z);
                    m = __vimax3_u32(m, w0.w, w1.x); m = __vimax3_u32(m, w1.y, w1.z); m = __vimax3_u32(m, w1.w, w2.x);
                    m = __vimax3_u32(m, w2.y, w2.z); m = __vimax3_u32(m, w2.w, w3.x); m = __vimax3_u32(m, w3.y, w3.z);
                    any4 = __vimax3_u32(m, w3.w, 0u) >= thr;
                }
                if (any4) {
                    scan_vec(v, w0); scan_vec(v + nthreads, w1); scan_vec(v + 2 * nthreads, w2); scan_vec(v + 3 * nthreads, w3);
                }
            }
            for (; v < n_vec; v += nthreads)
                if (HB_CHK(16u * (unsigned)(v + 1) <= limit, HB_H4)) scan_vec(v, acc4[v]);
            __syncthreads();
            const int n_items = min(misc[42], vcap) * CELLS;
            for (int i = tid; i < n_items; i += nthreads)
                if (HB_CHK((hshift + (single ? n : 0)) * 8 + 4 * (i / CELLS) + 4 <= 8 * p.chunk, HB_H4)) test_cell((int)vlist[i / CELLS], i % CELLS);
        }
        __syncthreads();

        // ---- H5: raster-order peak list.  pbm is [jl][k/32]: ascending word index is raster order.
        const int W = ncols * p.wpr;
        const int span = (W + nthreads - 1) / nthreads;
        const int w_lo = min(tid * span, W), w_hi = min(w_lo + span, W);
        int my_peaks = 0;
        for (int w = w_lo; w < w_hi; ++w)
            if (HB_CHK(4 * w + 4 <= p.pbm_bytes, HB_H5)) my_peaks += __popc(pbm[w]);
        int cta_peaks;
        int pos = block_exscan(my_peaks, misc, cta_peaks);
        int base = 0, n_peaks = cta_peaks;
        if (CL) {
            if (tid == 0) misc[40] = cta_peaks;
            cg::this_cluster().sync();   // (B) all scans done (accumulators no longer read remotely); totals visible
            n_peaks = 0;
            for (int r = 0; r < C; ++r) {
                int t = *(const int*)cg::this_cluster().map_shared_rank((void*)&misc[40], r);
                if (r < (int)rank) base += t;
                n_peaks += t;
            }
        }
        pos += base;
        for (int w = w_lo; w < w_hi && pos < p.max_peaks; ++w) {
            unsigned bits = HB_CHK(4 * w + 4 <= p.pbm_bytes, HB_H5) ? pbm[w] : 0u;
            const int jl = w / p.wpr, kb = (w - jl * p.wpr) << 5;
            while (bits && pos < p.max_peaks) {
                const int k = kb + __ffs(bits) - 1;
                bits &= bits - 1;
                if (!HB_CHK(jl < ncols && k < p.n_rho && pos >= 0, HB_H5)) continue;
                hough_peak pk;
                pk.theta_bin = (uint16_t)(col0 + jl);
                pk.rho_bin = (uint16_t)k;
                pk.votes = cell_from<ACC16>(acc, p.pitch_b, jl, k);
                p.peaks[(size_t)e * p.max_peaks + pos] = pk;
                ++pos;
            }
        }
        if (rank == 0 && tid == 0) p.counts[2 * e] = n_peaks;
        n_stored = min(n_peaks, p.max_peaks);
        if (CL) {
            __threadfence();
            cg::this_cluster().sync();   // (C) stored peaks visible cluster-wide; accumulator region is dead
        } else {
            __syncthreads();
        }
        }   // peak mode

        // ---- H6 set-up.  Marked columns = theta columns inside some stored peak's window; they get consecutive
        // indices q.  W8[q/8][k] is a byte whose bit (q%8) says "bin k of marked column q lies in a stored peak's
        // window" (= the union of the windows, S5).  Byte n_rho of a row stays 0: the clamp target of invalid bins.
        unsigned char* W8 = acc + p.w8_off;
        float* mcf = (float*)(acc + p.mcf_off);
        float* msf = (float*)(acc + p.msf_off);
        int* colq = (int*)(acc + p.colq_off);
        int n_marked = 0, n_g8 = 0, n_circ = 0;
        double* circ = (double*)(acc + p.w8_off);   // EXT, distance filter: (x_c, y_c, r_c) of the first circ_cap stored peaks
        // ---- H6 dense mode (EXT, HOUGH_OPT_SELECT_MODE).  When most theta columns are marked, the scan
        // below costs more than the voting phase (every hit x every marked column, one thread per hit).  Here the dead
        // accumulator is rewritten as the window mask -- cell (j, k) non-zero iff some stored peak has |j - j_p| <= w and
        // |k - k_p| <= w, S5's union of windows -- and every hit is tested at ALL columns with the voting loop's own
        // mapping and address arithmetic, a load where the vote had its atomic: bins outside the grid read the trash
        // row (zero).  One ballot per hit; the keep flags (one bit per hit of the event) live in the dead peak bitmap.
        const int ev_tame_d = (EXT && p.select_mode != 0) ? misc[33] : 0;
        unsigned* kf = pbm;
        bool dense = false;
        if (EXT && !CL && p.select_mode != 0 && p.keep_mode == 0 && n_stored > 0 && n > 0 && (long long)n <= 8LL * p.pbm_bytes &&
            (p.select_mode == 1 || 2LL * n_stored * (2 * p.window + 1) > p.n_theta)) {
            dense = true;
            {
                uint4* z = (uint4*)smem;
                const uint4 zz = make_uint4(0, 0, 0, 0);
                for (int i = tid; i < zero_vec; i += nthreads) z[i] = zz;      // accumulator, trash row, peak bitmap (= flags)
            }
            __syncthreads();
            for (int q = tid; q < n_stored; q += nthreads) {
                const hough_peak pk = p.peaks[(size_t)e * p.max_peaks + q];
                for (int dj = -p.window; dj <= p.window; ++dj) {
                    int j = (int)pk.theta_bin + dj, kref = (int)pk.rho_bin;
                    if (j < 0 || j >= p.n_theta) {
                        if (!p.theta_wrap) continue;
                        while (j < 0) { j += p.n_theta; kref = p.n_rho - 1 - kref; }       // reading Q19: mirrored across the seam
                        while (j >= p.n_theta) { j -= p.n_theta; kref = p.n_rho - 1 - kref; }
                    }
                    const unsigned half = ACC16 ? (1u << (16 * ((j >> 5) & 1))) : 1u;
                    for (int k = max(0, kref - p.window); k <= min(p.n_rho - 1, kref + p.window); ++k) {
                        const unsigned woff = (unsigned)k * pitch + 4u * cell_word_off<ACC16>(j);
                        if (HB_CHK(j < ncols && woff + 4 <= limit, HB_H6_SETUP)) atomicOr((unsigned*)(acc + woff), half);
                    }
                }
            }
            __syncthreads();
            const int S = p.n_stripes;
            for (int cbeg = 0; cbeg < n; cbeg += chunk) {
                const int m = min(chunk, n - cbeg);
                if (!single) {                    // the staged (u, v) of a chunked event are gone: stage this chunk again
                    for (int i = tid; i < m; i += nthreads)
                        if (HB_CHK(i < p.chunk, HB_STAGE)) hb0[i] = conformal(__ldg(&p.xy[beg + cbeg + i]), p.scale);
                    __syncthreads();
                }
                const float2* src = single ? hb : hb0;
                for (int i = stripe; i < m; i += S) {
                    const float2 uv = src[i];
                    unsigned any = 0;
                    if (ev_tame_d) {
#pragma unroll
                        for (int q = 0; q < CPL; q += 2) {
                            unsigned b0, b1;
                            bin_bits2(uv.x, uv.y, c2q[q / 2], s2q[q / 2], rho_max, inv, b0, b1);
                            const unsigned rel0 = min(b0 * pitch + lc0, trash0) + (ACC16 ? 128 * (q / 2) : 128 * q);
                            const unsigned rel1 = min(b1 * pitch + lc0, trash0) + (ACC16 ? 128 * (q / 2) : 128 * (q + 1));
                            const unsigned w0 = HB_CHK(rel0 + 4 <= acc_end, HB_KEEP) ? *(const unsigned*)(acc + rel0) : 0u;
                            const unsigned w1 = HB_CHK(rel1 + 4 <= acc_end, HB_KEEP) ? *(const unsigned*)(acc + rel1) : 0u;
                            any |= ACC16 ? ((w0 & 0xFFFFu) | (w1 >> 16)) : (w0 | w1);
                        }
                    } else {                      // degenerate hits somewhere in the event: the literal S2, as on the slow vote path
                        for (int q = 0; q < CPL; ++q) {
                            const int jl = 32 * (g * CPL + q) + lane;
                            if (jl >= ncols) continue;
                            const int k = bin_exact(uv.x, uv.y, p.cos_t[col0 + jl], p.sin_t[col0 + jl], p.rho_max, p.inv, p.n_rho);
                            if (k < 0) continue;
                            const unsigned woff = (unsigned)k * pitch + 4u * cell_word_off<ACC16>(jl);
                            const unsigned wv = HB_CHK(woff + 4 <= limit, HB_KEEP) ? *(const unsigned*)(acc + woff) : 0u;
                            any |= ACC16 ? ((wv >> (16 * ((jl >> 5) & 1))) & 0xFFFFu) : wv;
                        }
                    }
                    const unsigned bal = __ballot_sync(0xffffffffu, any != 0u);
                    if (lane == 0 && bal && HB_CHK(4 * ((cbeg + i) >> 5) + 4 <= p.pbm_bytes, HB_KEEP))
                        atomicOr(&kf[(cbeg + i) >> 5], 1u << ((cbeg + i) & 31));       // the column groups of one hit are different warps
                }
                __syncthreads();                  // flags complete / hb0 free for the next chunk
            }
        }
        if (dense) {
        } else if (EXT && p.keep_mode == 1) {
            // ---- N4b set-up (reading Q20): the stored peaks' candidate circles, Eq. (2)
            n_circ = min(n_stored, p.circ_cap);
            for (int q = tid; q < n_circ; q += nthreads) {
                const hough_peak pk = p.peaks[(size_t)e * p.max_peaks + q];
                double xc, yc, rc;
                circle_of(p.cos_t[pk.theta_bin], p.sin_t[pk.theta_bin], (int)pk.rho_bin, p.inv, p.rho_max, p.scale, xc, yc, rc);
                if (HB_CHK(p.w8_off + 24 * (q + 1) <= (CL ? p.stash_off : p.region_bytes), HB_H6_SETUP)) {
                    circ[3 * q] = xc; circ[3 * q + 1] = yc; circ[3 * q + 2] = rc;
                }
            }
            __syncthreads();
        } else {
        {
            long long cols_ub = (long long)n_stored * (2LL * p.window + 1);
            if (cols_ub > p.n_theta) cols_ub = p.n_theta;
            const int w8_vec = (int)((cols_ub + 7) >> 3) * (p.w8_pitch >> 4);
            uint4* z = (uint4*)W8;
            const uint4 zz = make_uint4(0, 0, 0, 0);
            for (int i = tid; i < w8_vec; i += nthreads)
                if (HB_CHK(p.w8_off + 16 * (i + 1) <= p.mcf_off, HB_H6_SETUP)) z[i] = zz;
            for (int j = tid; j < p.n_theta; j += nthreads)
                if (HB_CHK(p.colq_off + 4 * (j + 1) <= p.region_bytes, HB_H6_SETUP)) colq[j] = 0;
            if (tid == 0) misc[41] = 0;
        }
        __syncthreads();
        for (int q = tid; q < n_stored; q += nthreads) {
            const hough_peak pk = p.peaks[(size_t)e * p.max_peaks + q];
            if (EXT && p.theta_wrap) {     // reading Q19: window columns beyond a border fold onto the other end
                for (int dj = -p.window; dj <= p.window; ++dj) {
                    int j = ((int)pk.theta_bin + dj) % p.n_theta;
                    if (j < 0) j += p.n_theta;
                    if (HB_CHK(j >= 0 && j < p.n_theta, HB_H6_SETUP)) atomicOr(&colq[j], 1);
                }
                continue;
            }
            // (atomic: the windows of two peaks overlap, and two plain stores of the same 1 are still a write-write hazard)
            const int jlo = max(0, (int)pk.theta_bin - p.window), jhi = min(p.n_theta - 1, (int)pk.theta_bin + p.window);
            for (int j = jlo; j <= jhi; ++j)
                if (HB_CHK(j >= 0 && j < p.n_theta, HB_H6_SETUP)) atomicOr(&colq[j], 1);
        }
        __syncthreads();
        // number the marked columns (order irrelevant for the OR of S5)
        for (int jb = 0; jb < p.n_theta; jb += nthreads) {
            const int j = jb + tid;
            const bool any = j < p.n_theta && colq[j] != 0;
            const unsigned bal = __ballot_sync(0xffffffffu, any);
            int wbase = 0;
            if (lane == 0 && bal) wbase = atomicAdd(&misc[41], __popc(bal));
            wbase = __shfl_sync(0xffffffffu, wbase, 0);
            if (any) {
                const int q = wbase + __popc(bal & ((1u << lane) - 1u));
                if (HB_CHK(q >= 0 && q < p.n_theta, HB_H6_SETUP)) {
                    mcf[q] = p.cos_t[j];
                    msf[q] = p.sin_t[j];
                    colq[j] = q;
                }
            }
        }
        __syncthreads();
        n_marked = misc[41];
        n_g8 = (n_marked + 7) >> 3;
        if (tid < 8 * n_g8 - n_marked && HB_CHK(n_marked + tid < p.n_theta + 8, HB_H6_SETUP)) {   // pad the last group with columns whose bits are never set
            mcf[n_marked + tid] = 0.0f;
            msf[n_marked + tid] = 0.0f;
        }
        for (int q = tid; q < n_stored; q += nthreads) {
            const hough_peak pk = p.peaks[(size_t)e * p.max_peaks + q];
            // sets bit (cq % 8) of bytes klo..khi of marked column j's row
            auto fill = [&](int j, int klo, int khi) {
                const int cq = colq[j];
                if (!HB_CHK(cq >= 0 && cq < n_marked && ((cq >> 3) + 1) * p.w8_pitch <= p.mcf_off - p.w8_off && (khi | 3) < p.w8_pitch, HB_H6_SETUP)) return;
                const unsigned bit4 = (1u << (cq & 7)) * 0x01010101u;
                const unsigned row_s = (unsigned)__cvta_generic_to_shared(W8 + (cq >> 3) * p.w8_pitch);
                for (int wd = klo >> 2; wd <= khi >> 2; ++wd) {
                    const int a = max(klo, wd << 2) & 3, b = min(khi, (wd << 2) + 3) & 3;
                    const unsigned bytes = (0xFFFFFFFFu >> (8 * (3 - b))) & (0xFFFFFFFFu << (8 * a));
                    red_shared_or(row_s + 4u * wd, bit4 & bytes);
                }
            };
            if (EXT && p.theta_wrap) {     // a folded column is compared with the MIRRORED peak bin (once per fold)
                for (int dj = -p.window; dj <= p.window; ++dj) {
                    int j = (int)pk.theta_bin + dj, kref = (int)pk.rho_bin;
                    while (j < 0) { j += p.n_theta; kref = p.n_rho - 1 - kref; }
                    while (j >= p.n_theta) { j -= p.n_theta; kref = p.n_rho - 1 - kref; }
                    fill(j, max(0, kref - p.window), min(p.n_rho - 1, kref + p.window));
                }
                continue;
            }
            const int jlo = max(0, (int)pk.theta_bin - p.window), jhi = min(p.n_theta - 1, (int)pk.theta_bin + p.window);
            const int klo = max(0, (int)pk.rho_bin - p.window), khi = min(p.n_rho - 1, (int)pk.rho_bin + p.window);
            for (int j = jlo; j <= jhi; ++j) fill(j, klo, khi);
        }
        __syncthreads();
        }   // keep mode

        // ---- H6 keep test of one hit: OR over the marked columns q of bit q of W8[.][bin(i, column q)]  (== S5)
        const unsigned n_rho_u = (unsigned)p.n_rho;
        const int ev_tame = misc[33];      // CTA-uniform; written before the chunk's closing barrier
        auto keep_test = [&](float2 uv, float2 h, bool valid) -> bool {
            if (EXT && p.keep_mode == 1) {
                // N4b: keep iff | ||hit - centre|| - r_c | < tol for some stored peak (fp64, one rounding per operation)
                bool kp = false;
                if (valid) {
                    const double x = (double)h.x, y = (double)h.y;
                    for (int q = 0; q < n_stored && !kp; ++q) {
                        double xc, yc, rc;
                        if (q < n_circ) {
                            xc = circ[3 * q]; yc = circ[3 * q + 1]; rc = circ[3 * q + 2];
                        } else {                 // more stored peaks than staged circles: straight from the peak list
                            const hough_peak pk = p.peaks[(size_t)e * p.max_peaks + q];
                            circle_of(p.cos_t[pk.theta_bin], p.sin_t[pk.theta_bin], (int)pk.rho_bin, p.inv, p.rho_max, p.scale, xc, yc, rc);
                        }
                        const double dx = __dsub_rn(x, xc), dy = __dsub_rn(y, yc);
                        const double d = sqrt(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)));
                        if (fabs(__dsub_rn(d, rc)) < p.keep_tol) kp = true;
                    }
                }
                return kp;
            }
            unsigned hitbits = 0;
            for (int g8 = 0; g8 < n_g8; ++g8) {
                if (!HB_CHK(8 * g8 + 8 <= p.n_theta + 8 && (g8 + 1) * p.w8_pitch <= p.mcf_off - p.w8_off && p.n_rho < p.w8_pitch, HB_KEEP)) break;
                const float4 ca = *(const float4*)(mcf + 8 * g8), cb = *(const float4*)(mcf + 8 * g8 + 4);
                const float4 sa = *(const float4*)(msf + 8 * g8), sb = *(const float4*)(msf + 8 * g8 + 4);
                const unsigned char* row = W8 + g8 * p.w8_pitch;
                const float cc[8] = {ca.x, ca.y, ca.z, ca.w, cb.x, cb.y, cb.z, cb.w};
                const float ss[8] = {sa.x, sa.y, sa.z, sa.w, sb.x, sb.y, sb.z, sb.w};
                if (ev_tame) {
                    // two marked columns per packed instruction, as in the voting loop: same six roundings per column,
                    // same bins for tame hits, 3 FP instructions per column instead of 6
#pragma unroll
                    for (int i = 0; i < 8; i += 2) {
                        unsigned b0, b1;
                        bin_bits2(uv.x, uv.y, pack2(cc[i], cc[i + 1]), pack2(ss[i], ss[i + 1]), rho_max, inv, b0, b1);
                        const unsigned k0 = min(b0 - HOUGH_MAGIC_BITS, n_rho_u), k1 = min(b1 - HOUGH_MAGIC_BITS, n_rho_u);
                        hitbits |= ((unsigned)row[k0] & (1u << i)) | ((unsigned)row[k1] & (2u << i));
                    }
                } else {
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const unsigned k = min(bin_bits(uv.x, uv.y, cc[i], ss[i], rho_max, inv) - HOUGH_MAGIC_BITS, n_rho_u);
                        hitbits |= (unsigned)row[k] & (1u << i);
                    }
                }
                if (__all_sync(0xffffffffu, hitbits != 0u || !valid)) break;
            }
            return hitbits != 0u && valid;
        };

        // ---- H6 + H7
        if (!CL) {
            int kept_base = 0;
            for (int b0i = 0; b0i < n; b0i += nthreads) {
                const int i = b0i + tid;
                const bool valid = i < n;
                float2 uv = make_float2(0.0f, 0.0f);
                if (valid) uv = single ? hb[i] : conformal(__ldg(&p.xy[beg + i]), p.scale);
                float2 hxy = make_float2(0.0f, 0.0f);
                if (EXT && p.keep_mode == 1 && valid) hxy = __ldg(&p.xy[beg + i]);
                const bool kp = (EXT && dense) ? (valid && ((kf[i >> 5] >> (i & 31)) & 1u) != 0u) : keep_test(uv, hxy, valid);
                int blk_total;
                const int ppos = block_exscan(kp ? 1 : 0, misc, blk_total);
                if (valid) {
                    p.keep[beg + i] = kp ? 1 : 0;
                    if (kp && HB_CHK(kept_base + ppos >= 0 && kept_base + ppos <= i, HB_H7)) {
                        if (p.kept_xy) p.kept_xy[beg + kept_base + ppos] = __ldg(&p.xy[beg + i]);
                        if (p.kept_idx) p.kept_idx[beg + kept_base + ppos] = i;
                    }
                }
                kept_base += blk_total;
            }
            if (tid == 0) p.counts[2 * e + 1] = kept_base;
            __syncthreads();   // D / lists are dead: the region may be zeroed for the next event
        } else {
            // clustered: hit blocks are dealt round-robin to the CTAs; two passes per round
            unsigned* stash = (unsigned*)(acc + p.stash_off);   // [round block][warp] ballots
            int* cnt = (int*)(acc + p.cnt_off);                 // my blocks' kept counts (remote-readable)
            int* gcnt = (int*)(acc + p.gcnt_off);               // exclusive bases of this round's blocks
            const int n_blocks = (n + nthreads - 1) / nthreads;
            const int round_blocks = HOUGH_SEL_ROUND_BLOCKS * C;
            int kept_base = 0;
            for (int rb = 0; rb < n_blocks; rb += round_blocks) {
                const int rnb = min(round_blocks, n_blocks - rb);
                for (int bl = 0; rb + bl * C + (int)rank < rb + rnb; ++bl) {
                    const int i = (rb + bl * C + (int)rank) * nthreads + tid;
                    const bool valid = i < n;
                    float2 uv = make_float2(0.0f, 0.0f);
                    if (valid) uv = single ? hb[i] : conformal(__ldg(&p.xy[beg + i]), p.scale);
                    float2 hxy = make_float2(0.0f, 0.0f);
                    if (EXT && p.keep_mode == 1 && valid) hxy = __ldg(&p.xy[beg + i]);
                    const bool kp = keep_test(uv, hxy, valid);
                    const unsigned bal = __ballot_sync(0xffffffffu, kp);
                    if (lane == 0 && HB_CHK(bl < HOUGH_SEL_ROUND_BLOCKS, HB_H7)) stash[bl * nwarps + warp] = bal;
                    if (valid) p.keep[beg + i] = kp ? 1 : 0;
                    const int tot = __syncthreads_count(kp);
                    if (tid == 0 && HB_CHK(bl < HOUGH_SEL_ROUND_BLOCKS, HB_H7)) cnt[bl] = tot;
                }
                cg::this_cluster().sync();   // (D) counts of this round visible
                // exclusive bases of the round's blocks (every CTA computes all; tiny)
                if (warp == 0) {
                    int run = kept_base;
                    for (int b = 0; b < rnb; b += 32) {
                        const int bb = b + lane;
                        int v = 0;
                        if (bb < rnb && HB_CHK(bb / C < HOUGH_SEL_ROUND_BLOCKS, HB_H7)) v = *(const int*)cg::this_cluster().map_shared_rank((void*)&cnt[bb / C], bb % C);
                        int incl = v;
#pragma unroll
                        for (int d = 1; d < 32; d <<= 1) {
                            int o = __shfl_up_sync(0xffffffffu, incl, d);
                            if (lane >= d) incl += o;
                        }
                        if (bb < rnb) gcnt[bb] = run + incl - v;
                        run += __shfl_sync(0xffffffffu, incl, 31);
                    }
                    if (lane == 0) gcnt[rnb] = run;
                }
                __syncthreads();
                for (int bl = 0; rb + bl * C + (int)rank < rb + rnb; ++bl) {
                    const int bb = bl * C + (int)rank;
                    const int i = (rb + bb) * nthreads + tid;
                    const unsigned bal = stash[bl * nwarps + warp];
                    if ((bal >> lane) & 1u) {
                        int ppos = gcnt[bb] + __popc(bal & ((1u << lane) - 1u));
                        for (int w2 = 0; w2 < warp; ++w2) ppos += __popc(stash[bl * nwarps + w2]);
                        if (!HB_CHK(ppos >= 0 && ppos <= i && bb <= HOUGH_SEL_ROUND_BLOCKS * C, HB_H7)) continue;
                        if (p.kept_xy) p.kept_xy[beg + ppos] = __ldg(&p.xy[beg + i]);
                        if (p.kept_idx) p.kept_idx[beg + ppos] = i;
                    }
                }
                kept_base = gcnt[rnb];
                cg::this_cluster().sync();   // (E) remote reads of cnt done before it is rewritten / zeroed
            }
            if (rank == 0 && tid == 0) p.counts[2 * e + 1] = kept_base;
        }
#ifdef HOUGH_DEBUG_BOUNDS
        {   // report skipped accesses: {HOUGH_DBG_SENTINEL, bit mask of the phases that violated}
            if (CL) cg::this_cluster().sync();   // after rank 0's regular count writes
            const int m = __syncthreads_or(dbg_viol ? (1 << dbg_viol) : 0);
            if (m && tid == 0) { p.counts[2 * e] = HOUGH_DBG_SENTINEL; p.counts[2 * e + 1] = m; }
        }
#endif
    }
}


// ---------------------------------------------------------------- N1: candidate circles and track parameters
// SURVEY.md 8(f) NEXT-1; Eq. (2), pT and phi0 PAPER.md:150-158; readings Q14-Q17.
// One CTA per event, one warp per stored peak: the lanes stride over the event's hits, count the hits ASSOCIATED with
// the peak (own bin at the peak's column within the keep window) and on which side of the centre direction they lie
// (fp32 cross product c_j y - s_j x, one rounding per operation); lane 0 then writes the circle in fp64.
struct CParams {
    const float2* xy;
    const int* off;
    int n_events;
    const hough_peak* peaks;
    const int* counts;
    hough_circle* out;
    const float* cos_t;
    const float* sin_t;
    int n_theta, n_rho, window, max_peaks;
    float rho_max, inv, scale;
    double b_field;
};

__global__ void __launch_bounds__(256) hough_circles_kernel(const __grid_constant__ CParams p) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const double pi = 3.14159265358979323846;
    for (int e = blockIdx.x; e < p.n_events; e += gridDim.x) {
        const int beg = p.off[e], n = p.off[e + 1] - beg;
        const int n_peaks = p.counts[2 * e];
        const int n_stored = n_peaks < p.max_peaks ? n_peaks : p.max_peaks;   // a refused event (-1) stores nothing
        for (int q = warp; q < n_stored; q += nwarps) {
            const hough_peak pk = p.peaks[(size_t)e * p.max_peaks + q];
            const int j = pk.theta_bin, k = pk.rho_bin;
            const float cj = p.cos_t[j], sj = p.sin_t[j];
            const double rc = rho_centre(k, p.inv, p.rho_max);
            int n_pos = 0, n_neg = 0, n_assoc = 0;
            for (int i = lane; i < n; i += 32) {
                const float2 h = __ldg(&p.xy[beg + i]);
                const float2 uv = conformal(h, p.scale);
                const int kb = bin_exact(uv.x, uv.y, cj, sj, p.rho_max, p.inv, p.n_rho);
                if (kb < 0) continue;
                const int dk = kb > k ? kb - k : k - kb;
                if (dk > p.window) continue;
                ++n_assoc;
                float z = __fsub_rn(__fmul_rn(cj, h.y), __fmul_rn(sj, h.x));
                if (rc < 0.0) z = -z;
                if (z > 0.0f) ++n_pos;
                else if (z < 0.0f) ++n_neg;
            }
#pragma unroll
            for (int d = 16; d >= 1; d >>= 1) {
                n_pos += __shfl_xor_sync(0xffffffffu, n_pos, d);
                n_neg += __shfl_xor_sync(0xffffffffu, n_neg, d);
                n_assoc += __shfl_xor_sync(0xffffffffu, n_assoc, d);
            }
            if (lane == 0) {
                hough_circle c;
                circle_of(cj, sj, k, p.inv, p.rho_max, p.scale, c.x_c, c.y_c, c.r_c);
                c.pt = __dmul_rn(__dmul_rn(0.0003, p.b_field), c.r_c);
                c.charge = n_neg > n_pos ? 1 : (n_pos > n_neg ? -1 : 0);
                c.n_hits = n_assoc;
                double phi_c = __ddiv_rn(__dmul_rn((double)j, pi), (double)p.n_theta);
                if (rc < 0.0) phi_c = __dadd_rn(phi_c, pi);
                double phi0 = __dsub_rn(phi_c, __dmul_rn((double)c.charge, pi / 2.0));
                if (phi0 < 0.0) phi0 = __dadd_rn(phi0, 2.0 * pi);
                if (phi0 >= 2.0 * pi) phi0 = __dsub_rn(phi0, 2.0 * pi);
                c.phi0 = phi0;
                p.out[(size_t)e * p.max_peaks + q] = c;
            }
        }
    }
}

}  // namespace hough
