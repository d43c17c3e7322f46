// simt_shim.h -- TEST INFRASTRUCTURE.  A small single-OS-thread SIMT emulator that lets g++ compile
// paper_2607_04067_b200/csrc/hough_kernel.cuh (with -DHOUGH_HOST_EMU) and execute it on the CPU: every CUDA
// thread of a cluster is a fiber (ucontext); __syncthreads, cluster.sync and the full-mask warp collectives are
// barriers at which a fiber yields; shared memory is one guarded buffer per CTA; shared atomics are plain
// read-modify-writes (fibers never run concurrently).  It checks the kernel's LOGIC (indexing, phase order,
// bounds) against the oracle without a GPU; it says nothing about PTX semantics or speed.
//
// Race check (the hough_emu_race build: this file compiled with -fsanitize=thread but linked WITHOUT ThreadSanitizer's
// runtime).  The compiler's instrumentation calls __tsan_read<N> / __tsan_write<N> / __tsan_atomic* for every memory
// access of the kernel; the hooks at the end of this file implement a detector made for CUDA's synchronisation: every
// barrier is all-inclusive at its scope (warp: __syncwarp; CTA: __syncthreads*; cluster: cluster.sync), so an earlier
// access A happens before a later access B exactly when B's thread has passed more barriers of a scope both share
// than A's thread had when it made A.  Every thread counts the barriers it has passed, every byte of shared memory
// (of all CTAs of the cluster) and of the global output buffers remembers its last plain write, its last atomics and
// the reads since; two accesses of different threads to the same byte, at least one a write and not both atomic,
// that no barrier orders, are reported with both code addresses.  cp.async.bulk / launch-control writes are "async"
// writes: ordered after what the issuing thread did before, and before a reader only through the mbarrier phase it
// waited for.  Threads of different clusters of one launch are never ordered.  This is what compute-sanitizer's
// racecheck reports for shared memory, extended to DSMEM and global memory.  The same shadow state gives an initcheck:
// a read or atomic of a byte that nothing has written since the CTA started (shared) / since the first launch (outputs).  (Warp shuffles and votes order nothing.
// The emulator's own bookkeeping is excluded from the instrumentation: EMU_NOSAN.)
#pragma once
#include <sys/mman.h>
#include <ucontext.h>
#include <unistd.h>

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <utility>
#include <vector>

#if defined(__SANITIZE_THREAD__)
#define EMU_RACE 1
#define EMU_NOSAN __attribute__((no_sanitize("thread")))
#else
#define EMU_NOSAN
#endif

#define __global__
#define __device__
#define __host__
#define __forceinline__ inline
#define __launch_bounds__(...)
#define __grid_constant__
#define __align__(n) alignas(n)

struct float2 { float x, y; };
struct float4 { float x, y, z, w; };
struct alignas(16) uint4 { unsigned x, y, z, w; };
struct dim3 {
    unsigned x, y, z;
    dim3(unsigned x_ = 1, unsigned y_ = 1, unsigned z_ = 1) : x(x_), y(y_), z(z_) {}
};
inline float2 make_float2(float x, float y) { return float2{x, y}; }
inline uint4 make_uint4(unsigned x, unsigned y, unsigned z, unsigned w) { return uint4{x, y, z, w}; }

namespace emu {

[[noreturn]] inline void die(const char* msg) {
    fprintf(stderr, "simt_emu: %s\n", msg);
    fflush(stderr);
    _exit(3);
}

// A buffer whose END sits on a page boundary followed by an inaccessible page, and whose start is preceded by one:
// an access past the end faults at once, one before the start faults within a page.
struct Guarded {
    unsigned char* base = nullptr;   // mmap base
    size_t map_bytes = 0;
    unsigned char* ptr = nullptr;    // user pointer
    size_t bytes = 0;
    void alloc(size_t n) {
        const size_t pg = (size_t)sysconf(_SC_PAGESIZE);
        bytes = n;
        const size_t body = (n + pg - 1) / pg * pg;
        map_bytes = body + 2 * pg;
        base = (unsigned char*)mmap(nullptr, map_bytes, PROT_READ | PROT_WRITE, MAP_PRIVATE | MAP_ANONYMOUS, -1, 0);
        if (base == MAP_FAILED) die("mmap failed");
        mprotect(base, pg, PROT_NONE);
        mprotect(base + pg + body, pg, PROT_NONE);
        ptr = base + pg + body - n;               // n is a multiple of 16 for shared memory, so ptr is 16-byte aligned there
    }
    void release() { if (base) munmap(base, map_bytes); base = nullptr; }
};

struct Barrier {
    int expected = 0, arrived = 0;
    unsigned gen = 0;
    int acc_and = 1, acc_or = 0, acc_cnt = 0;
    int res_and = 1, res_or = 0, res_cnt = 0;
    int line = 0;                    // synccheck: the source line of the barrier call the first thread of this generation made
};

struct Warp {
    int arrived = 0;
    unsigned gen = 0;
    unsigned vals[2][32];
};

struct Cta {
    unsigned mbar_phases[2] = {0, 0};   // completed phases of the CTA's mbarriers (bulk-copy staging, launch control)
    unsigned mbar_addr[2] = {0, 0};
    int steals_left = 0;             // launch control: how many more events this CTA may take over (emu::clc_steal)
    Guarded smem;
    int rank = 0;
    dim3 bidx;
    Barrier bar;
    std::vector<Warp> warps;
};

struct Fiber {
    ucontext_t ctx;
    unsigned char* stack = nullptr;  // a slice of run_cluster's one stack block
    dim3 tidx;
    Cta* cta = nullptr;
    bool done = false;
    // race check: who this is, and how many barriers of each scope it has passed (see the header comment)
    unsigned fid = 0, cta_uid = 0, cl_gen = 0, cta_gen = 0, warp_gen = 0, mbar_seen[2] = {0, 0};
    unsigned long progress = 0;      // bumped whenever the fiber gets past a wait
};

struct Grid {
    dim3 bdim, gdim;
    int csize = 1, cluster = 0, n_clusters_ = 1;
    std::vector<Cta> ctas;           // the CTAs of the cluster being run
    Barrier cluster_bar;
    ucontext_t sched;
    void (*entry)() = nullptr;
};

inline Grid g;
inline Fiber* cur = nullptr;

#ifdef EMU_RACE
// ---------------------------------------------------------------- race check: shadow state and the ordering rule
namespace race {

enum Kind : unsigned char { NONE = 0, READ = 1, WRITE = 2, ATOMIC = 3, ASYNC = 4, PRIOR = 5 };   // PRIOR: written by an earlier launch
struct Rec {                                   // one remembered access of one byte
    unsigned fid = 0, cl = 0, cta = 0, wg = 0, pc = 0, mphase = 0;
    unsigned short cta_uid = 0;
    unsigned char kind = NONE, mslot = 0;
};
struct Shadow { Rec w, a[2], r[3]; };          // last plain / async write, last atomics (two threads), reads since (three threads)
struct Region {
    unsigned char* lo = nullptr;
    size_t bytes = 0;
    bool shared = false;
    int rank = 0;
    const char* name = "";
    std::vector<Shadow> sh;
};
inline std::vector<Region> regions;
// HOUGH_EMU_PROFILE=1: how often each code address touched tracked memory, per access kind (dumped by emu_main at exit):
// a count of the kernel's shared / global memory operations per source line, thread by thread
inline bool profile_on = getenv("HOUGH_EMU_PROFILE") != nullptr;
inline std::map<unsigned long long, unsigned long long> profile;      // (pc << 8 | shared << 4 | kind) -> thread-level accesses
inline unsigned long n_reports = 0;
inline std::vector<unsigned long long> seen_pairs;

EMU_NOSAN inline void track(void* p, size_t bytes, bool shared, int rank, const char* name = "shared") {
    regions.emplace_back();
    Region& r = regions.back();
    r.lo = (unsigned char*)p; r.bytes = bytes; r.shared = shared; r.rank = rank; r.name = name;
    r.sh.assign(bytes, Shadow());
}
EMU_NOSAN inline void untrack_shared() {       // shared memory dies with its cluster
    for (size_t i = regions.size(); i-- > 0;)
        if (regions[i].shared) regions.erase(regions.begin() + (long)i);
}
EMU_NOSAN inline void untrack(void* p) {
    for (size_t i = regions.size(); i-- > 0;)
        if (regions[i].lo == (unsigned char*)p) regions.erase(regions.begin() + (long)i);
}
EMU_NOSAN inline void host_write(void* p, size_t n) {      // a copy or memset between launches: the bytes count as written
    unsigned char* a = (unsigned char*)p;
    for (auto& r : regions)
        if (a >= r.lo && a < r.lo + r.bytes)
            for (size_t i = 0; i < n && (size_t)(a - r.lo) + i < r.bytes; ++i) {
                Shadow& s = r.sh[(size_t)(a - r.lo) + i];
                s = Shadow();
                s.w.kind = PRIOR;
            }
}
EMU_NOSAN inline void new_launch() {           // a kernel boundary orders everything: forget the history, keep "was written"
    for (auto& r : regions)
        for (auto& s : r.sh) {
            const bool written = s.w.kind != NONE || s.a[0].kind != NONE || s.a[1].kind != NONE;
            s = Shadow();
            if (written) s.w.kind = PRIOR;
        }
}

// does the remembered access `p` happen before whatever the current thread does now?
EMU_NOSAN inline bool ordered(const Rec& p) {
    const Fiber* c = cur;
    if (p.kind == PRIOR) return true;
    const unsigned csz = (unsigned)g.csize;
    if (p.cta_uid / csz != c->cta_uid / csz) return false;                    // another cluster of the launch: never
    const bool same_cta = p.cta_uid == c->cta_uid;
    if (p.kind == ASYNC) return same_cta && c->mbar_seen[p.mslot] >= p.mphase;   // only the mbarrier phase orders an async write
    if (p.fid == c->fid) return true;                                         // program order
    if (p.cl < c->cl_gen) return true;
    if (same_cta && p.cta < c->cta_gen) return true;
    if (same_cta && (p.fid >> 5) == (c->fid >> 5) && p.wg < c->warp_gen) return true;   // (block sizes are multiples of 32)
    return false;
}

EMU_NOSAN inline void report(const Region& rg, size_t off, unsigned char kind, unsigned pc, const Rec& p) {
    const unsigned long long key = ((unsigned long long)pc << 32) | p.pc;
    for (auto k : seen_pairs) if (k == key) return;
    seen_pairs.push_back(key);
    ++n_reports;
    static const char* names[] = {"none", "read", "write", "atomic", "async-write"};
    const unsigned th = (unsigned)g.bdim.x;
    fprintf(stderr, "RACE %s+%zu (cta rank %d's): %s by cta %u thread %u pc 0x%x  <->  earlier %s by cta %u thread %u pc 0x%x\n",
            rg.name, off, rg.rank, names[kind], cur->cta_uid, cur->fid % th, pc, names[p.kind], (unsigned)p.cta_uid, p.fid % th, p.pc);
}

EMU_NOSAN inline void access(const void* addr, size_t size, unsigned char kind, const void* ret_pc, unsigned mslot = 0, unsigned mphase = 0) {
    static bool busy = false;      // the containers used below are instrumented library code: their accesses are not the kernel's
    if (!cur || busy) return;                                                  // (!cur: host code -- set-up, read-back)
    busy = true;
    struct Done { ~Done() { busy = false; } } done;
    const unsigned char* a = (const unsigned char*)addr;
    Region* rg = nullptr;
    for (auto& r : regions)
        if (a >= r.lo && a < r.lo + r.bytes) { rg = &r; break; }
    if (!rg) return;                                                           // stack, parameters, read-only inputs
    const unsigned pc = (unsigned)(size_t)ret_pc - 1;
    if (profile_on) ++profile[((unsigned long long)pc << 8) | (rg->shared ? 16u : 0u) | kind];
    Rec me;
    me.fid = cur->fid; me.cl = cur->cl_gen; me.cta = cur->cta_gen; me.wg = cur->warp_gen; me.pc = pc;
    me.cta_uid = (unsigned short)cur->cta_uid; me.kind = kind; me.mslot = (unsigned char)mslot; me.mphase = mphase;
    for (size_t i = 0; i < size && (size_t)(a - rg->lo) + i < rg->bytes; ++i) {
        const size_t off = (size_t)(a - rg->lo) + i;
        Shadow& s = rg->sh[off];
        // initcheck: a read (or a read-modify-write) of a byte that nothing has written since the launch / since the CTA
        // started -- shared memory starts as garbage, the output buffers hold whatever the caller left there
        if (kind != WRITE && kind != ASYNC && s.w.kind == NONE && s.a[0].kind == NONE && s.a[1].kind == NONE) {
            const unsigned long long key = ((unsigned long long)pc << 32) | 1u;
            bool seen = false;
            for (auto k : seen_pairs) if (k == key) { seen = true; break; }
            if (!seen) {
                seen_pairs.push_back(key);
                ++n_reports;
                fprintf(stderr, "UNINIT %s+%zu (cta rank %d's): %s of a never-written byte by cta %u thread %u pc 0x%x\n", rg->name, off,
                        rg->rank, kind == READ ? "read" : "atomic", cur->cta_uid, cur->fid % (unsigned)g.bdim.x, pc);
            }
        }
        // a plain or async write conflicts with everything; a read with writes and atomics; an atomic with plain accesses
        if (s.w.kind != NONE && !ordered(s.w)) report(*rg, off, kind, pc, s.w);
        if (kind != ATOMIC)
            for (auto& q : s.a) if (q.kind != NONE && !ordered(q)) report(*rg, off, kind, pc, q);
        if (kind != READ)
            for (auto& q : s.r) if (q.kind != NONE && !ordered(q)) report(*rg, off, kind, pc, q);
        if (kind == READ) {
            // remember this read: replace my own older one or one that is ordered before me (then it is ordered before
            // every later access too); else take a free slot; else keep reads of different warps
            Rec* slot = nullptr;
            for (auto& q : s.r) if (q.kind != NONE && (q.fid == me.fid || ordered(q))) { slot = &q; break; }
            if (!slot) for (auto& q : s.r) if (q.kind == NONE) { slot = &q; break; }
            if (!slot && (s.r[0].fid >> 5) == (s.r[1].fid >> 5) && (s.r[0].fid >> 5) != (me.fid >> 5)) slot = &s.r[1];
            if (!slot && (s.r[1].fid >> 5) == (s.r[2].fid >> 5) && (s.r[1].fid >> 5) != (me.fid >> 5)) slot = &s.r[2];
            if (slot) *slot = me;
        } else if (kind == ATOMIC) {
            Rec* slot = nullptr;
            for (auto& q : s.a) if (q.kind != NONE && (q.fid == me.fid || ordered(q))) { slot = &q; break; }
            if (!slot) for (auto& q : s.a) if (q.kind == NONE) { slot = &q; break; }
            if (!slot) slot = &s.a[(me.fid >> 5) == (s.a[0].fid >> 5) ? 0 : 1];
            *slot = me;
            for (auto& q : s.r) q.kind = NONE;                                 // (checked above)
        } else {
            s.w = me;
            for (auto& q : s.a) q.kind = NONE;
            for (auto& q : s.r) q.kind = NONE;
        }
    }
}

}  // namespace race
#endif

EMU_NOSAN inline void yield() {
    Fiber* me = cur;
    swapcontext(&me->ctx, &g.sched);
}

// synccheck: every thread of a barrier generation must arrive from the SAME barrier call of the source (a barrier in
// divergent code pairs up calls that were never meant to meet; the hardware would count them all the same).  `line` is
// the call site (__builtin_LINE() in the default arguments of __syncthreads* / cluster.sync).
EMU_NOSAN inline void wait_barrier(Barrier& b, int pred, int& r_and, int& r_or, int& r_cnt, int scope = 1, int line = 0) {
    const unsigned gen = b.gen;
    if (b.arrived == 0) b.line = line;
    else if (b.line != line) {
        fprintf(stderr, "simt_emu: threads of one %s barrier generation arrive from different source lines: %d and %d\n",
                scope == 2 ? "cluster" : "CTA", b.line, line);
        die("divergent barrier");
    }
    b.acc_and &= pred ? 1 : 0;
    b.acc_or |= pred ? 1 : 0;
    b.acc_cnt += pred ? 1 : 0;
    if (++b.arrived == b.expected) {
        b.res_and = b.acc_and; b.res_or = b.acc_or; b.res_cnt = b.acc_cnt;
        b.acc_and = 1; b.acc_or = 0; b.acc_cnt = 0;
        b.arrived = 0;
        ++b.gen;
    } else {
        while (b.gen == gen) yield();
    }
    ++cur->progress;
    if (scope == 2) ++cur->cl_gen; else ++cur->cta_gen;      // counted on leaving: by then every thread of the scope has arrived
    r_and = b.res_and; r_or = b.res_or; r_cnt = b.res_cnt;
}

// full-mask warp collective: every lane deposits `v`, all wait, every lane may read any lane's value
EMU_NOSAN inline const unsigned* warp_exchange(unsigned v, bool orders_memory = false) {
    Cta* c = cur->cta;
    Warp& w = c->warps[cur->tidx.x >> 5];
    const unsigned gen = w.gen;
    unsigned* buf = w.vals[gen & 1];
    buf[cur->tidx.x & 31] = v;
    if (++w.arrived == 32) {
        w.arrived = 0;
        ++w.gen;
    } else {
        while (w.gen == gen) yield();
    }
    ++cur->progress;
    if (orders_memory) ++cur->warp_gen;                      // __syncwarp; shuffles and votes order nothing
    return buf;
}

constexpr unsigned SHARED_WINDOW = 0x01000000u;   // what __cvta_generic_to_shared returns for the first byte
EMU_NOSAN inline unsigned char* shared_ptr(unsigned saddr) {
    const unsigned off = saddr - SHARED_WINDOW;
    if ((size_t)off + 4 > cur->cta->smem.bytes) die("shared-window address outside the CTA's shared memory");
    return cur->cta->smem.ptr + off;
}
EMU_NOSAN inline unsigned char* dyn_smem() { return cur->cta->smem.ptr; }
EMU_NOSAN inline int cluster_id() { return g.cluster; }
EMU_NOSAN inline int n_clusters() { return g.n_clusters_; }

// bulk-copy staging: what a cp.async.bulk must satisfy (16-byte aligned source, destination and size; the source inside
// the hit array)
inline const unsigned char* bulk_lo = nullptr;
inline const unsigned char* bulk_hi = nullptr;
inline bool (*bulk_range_ok)(const void*, size_t) = nullptr;      // host emulation: "inside one device allocation"
EMU_NOSAN inline void bulk_check(unsigned dst, const void* src, unsigned bytes) {
    const unsigned char* s = (const unsigned char*)src;
    if (((size_t)s & 15) || (bytes & 15) || ((dst - SHARED_WINDOW) & 15)) die("cp.async.bulk: source, destination or size not 16-byte aligned");
    if (bulk_range_ok ? !bulk_range_ok(s, bytes) : (s < bulk_lo || s + bytes > bulk_hi)) die("cp.async.bulk: source range leaves the hit array");
    if ((size_t)(dst - SHARED_WINDOW) + bytes > cur->cta->smem.bytes) die("cp.async.bulk: destination leaves shared memory");
}

// The CTA's mbarrier: the emulated copy lands at issue time, which completes one phase; a waiter of parity p gets true
// once the phase of that parity has completed, else it yields (so a thread that runs ahead of the issuing thread really
// waits, as it does for the asynchronous copy on the device).
EMU_NOSAN inline unsigned& mbar_slot(unsigned bar) {
    Cta* c = cur->cta;
    for (int i = 0; i < 2; ++i) {
        if (c->mbar_addr[i] == bar) return c->mbar_phases[i];
        if (c->mbar_addr[i] == 0) { c->mbar_addr[i] = bar; return c->mbar_phases[i]; }
    }
    die("more than two mbarriers in one CTA");
}
EMU_NOSAN inline void mbar_complete(unsigned bar) { ++mbar_slot(bar); }
EMU_NOSAN inline bool mbar_wait_parity(unsigned bar, unsigned parity) {
    unsigned& ph = mbar_slot(bar);
    if ((ph & 1u) != (parity & 1u)) {
        cur->mbar_seen[&ph - cur->cta->mbar_phases] = ph;     // race check: async writes of the phases up to ph are visible now
        ++cur->progress;
        return true;
    }
    yield();
    return false;
}
// race check: a write made by the copy engine / the launch-control hardware on behalf of the current thread; readers see
// it through the completed phase of mbarrier `bar`
EMU_NOSAN inline void async_write(void* p, unsigned bytes, unsigned bar) {
#ifdef EMU_RACE
    unsigned& ph = mbar_slot(bar);
    race::access(p, bytes, race::ASYNC, __builtin_return_address(0), (unsigned)(&ph - cur->cta->mbar_phases), ph);
#else
    (void)p; (void)bytes; (void)bar;
#endif
}

// Cluster launch control: the CTAs of the grid that have not started yet are cluster ids next_unlaunched .. n-1 (the
// emulator runs one CTA after the other).  A request hands out the next of them -- the hardware then never launches it
// -- unless this CTA has used up its share (HOUGH_EMU_STEALS, default unlimited; a small number mixes stolen and
// regularly launched CTAs) or none is left; -1 = the request failed.
inline int next_unlaunched = 0;
EMU_NOSAN inline int clc_steal() {
    if (cur->cta->steals_left == 0 || next_unlaunched >= g.n_clusters_) return -1;
    if (cur->cta->steals_left > 0) --cur->cta->steals_left;
    return next_unlaunched++;
}

inline float ftz(float x) { return std::fpclassify(x) == FP_SUBNORMAL ? std::copysign(0.0f, x) : x; }

EMU_NOSAN inline void fiber_main() {
    g.entry();
    cur->done = true;
    swapcontext(&cur->ctx, &g.sched);
}

// Runs one cluster (csize CTAs of `threads` threads, `smem_bytes` each) to completion.
EMU_NOSAN inline void run_cluster(int cluster, int n_clusters, int csize, int threads, size_t smem_bytes, void (*entry)()) {
    g.bdim.x = (unsigned)threads;
    g.gdim.x = (unsigned)(n_clusters * csize);
    g.csize = csize; g.cluster = cluster; g.n_clusters_ = n_clusters; g.entry = entry;
    g.ctas.assign((size_t)csize, Cta());
    g.cluster_bar = Barrier();
    g.cluster_bar.expected = csize * threads;
    std::vector<Fiber> fibers((size_t)csize * threads);
#ifdef EMU_RACE
    const size_t stack_bytes = 128 * 1024;
#else
    const size_t stack_bytes = 32 * 1024;
#endif
    std::vector<unsigned char> stacks(fibers.size() * stack_bytes);     // one block: one mapping, not one per fiber
    for (int r = 0; r < csize; ++r) {
        Cta& c = g.ctas[r];
        c.smem.alloc(smem_bytes);
        memset(c.smem.ptr, 0xCD, smem_bytes);       // shared memory starts as garbage, as on the device
#ifdef EMU_RACE
        race::track(c.smem.ptr, smem_bytes, /*shared=*/true, r);
#endif
        c.rank = r;
        c.bidx.x = (unsigned)(cluster * csize + r);
        c.bar.expected = threads;
        c.warps.assign((size_t)threads / 32, Warp());
        c.steals_left = getenv("HOUGH_EMU_STEALS") ? atoi(getenv("HOUGH_EMU_STEALS")) : -1;
        for (int t = 0; t < threads; ++t) {
            Fiber& f = fibers[(size_t)r * threads + t];
            f.stack = stacks.data() + ((size_t)r * threads + t) * stack_bytes;
            f.fid = (unsigned)((cluster * csize + r) * threads + t);
            f.cta_uid = (unsigned)(cluster * csize + r);
            f.tidx.x = (unsigned)t;
            f.cta = &c;
            getcontext(&f.ctx);
            f.ctx.uc_stack.ss_sp = f.stack;
            f.ctx.uc_stack.ss_size = stack_bytes;
            f.ctx.uc_link = nullptr;
            makecontext(&f.ctx, (void (*)())fiber_main, 0);
        }
    }
    // Order in which the fibers get their turn in every scheduling pass.  A fiber runs until its next barrier or warp
    // collective, so the order decides which thread's phase runs first: code that is missing a barrier between a producer
    // and a consumer gives different results under different orders.  HOUGH_EMU_ORDER = forward (default) | reverse |
    // shuffle[:seed] (a fresh pseudo-random permutation per pass).
    const char* ord = getenv("HOUGH_EMU_ORDER");
    const bool reverse = ord && !strncmp(ord, "reverse", 7), shuffle = ord && !strncmp(ord, "shuffle", 7);
    unsigned long long rng = 0x9E3779B97F4A7C15ull ^ (shuffle && ord[7] == ':' ? strtoull(ord + 8, nullptr, 10) : 0ull) ^ (unsigned)cluster;
    std::vector<size_t> order(fibers.size());
    for (size_t i = 0; i < order.size(); ++i) order[i] = reverse ? order.size() - 1 - i : i;
    size_t live = fibers.size();
    while (live) {
        unsigned long before = 0, after = 0;
        for (auto& f : fibers) before += f.progress;
        size_t finished_now = 0;
        if (shuffle)
            for (size_t i = order.size() - 1; i > 0; --i) {
                rng = rng * 6364136223846793005ull + 1442695040888963407ull;
                std::swap(order[i], order[(size_t)((rng >> 33) % (i + 1))]);
            }
        for (size_t oi = 0; oi < order.size(); ++oi) {
            Fiber& f = fibers[order[oi]];
            if (f.done) continue;
            cur = &f;
            swapcontext(&g.sched, &f.ctx);
            if (f.done) { ++finished_now; --live; }
        }
        for (auto& f : fibers) after += f.progress;
        if (after == before && finished_now == 0) die("deadlock: a barrier or warp collective was not reached by every thread");
    }
    cur = nullptr;
#ifdef EMU_RACE
    race::untrack_shared();
#endif
    for (auto& c : g.ctas) c.smem.release();
}

}  // namespace emu

#ifdef EMU_RACE
// ---------------------------------------------------------------- what -fsanitize=thread makes the compiler call
extern "C" {
EMU_NOSAN void __tsan_init() {}
EMU_NOSAN void __tsan_func_entry(void*) {}
EMU_NOSAN void __tsan_func_exit() {}
EMU_NOSAN void __tsan_vptr_update(void**, void*) {}
EMU_NOSAN void __tsan_vptr_read(void**) {}
#define EMU_HOOK(N)                                                                                                              \
    EMU_NOSAN void __tsan_read##N(void* p) { emu::race::access(p, N, emu::race::READ, __builtin_return_address(0)); }            \
    EMU_NOSAN void __tsan_write##N(void* p) { emu::race::access(p, N, emu::race::WRITE, __builtin_return_address(0)); }          \
    EMU_NOSAN void __tsan_unaligned_read##N(void* p) { emu::race::access(p, N, emu::race::READ, __builtin_return_address(0)); }  \
    EMU_NOSAN void __tsan_unaligned_write##N(void* p) { emu::race::access(p, N, emu::race::WRITE, __builtin_return_address(0)); }
EMU_HOOK(1) EMU_HOOK(2) EMU_HOOK(4) EMU_HOOK(8) EMU_HOOK(16)
#undef EMU_HOOK
EMU_NOSAN void __tsan_read_range(void* p, unsigned long n) { emu::race::access(p, n, emu::race::READ, __builtin_return_address(0)); }
EMU_NOSAN void __tsan_write_range(void* p, unsigned long n) { emu::race::access(p, n, emu::race::WRITE, __builtin_return_address(0)); }
// the kernel's atomics (shim: __atomic builtins, relaxed) arrive here
#define EMU_ATOMIC(OP, EXPR)                                                                                                     \
    EMU_NOSAN unsigned __tsan_atomic32_fetch_##OP(volatile unsigned* p, unsigned v, int) {                                       \
        emu::race::access((const void*)p, 4, emu::race::ATOMIC, __builtin_return_address(0));                                    \
        const unsigned o = *p; *p = EXPR; return o;                                                                              \
    }
EMU_ATOMIC(add, o + v) EMU_ATOMIC(and, o & v) EMU_ATOMIC(or, o | v)
#undef EMU_ATOMIC
// host code compiled into the same unit (std::atomic counters, the guards of function-local statics): plain operations,
// the host side of the emulation runs on one thread
EMU_NOSAN unsigned char __tsan_atomic8_load(const volatile unsigned char* p, int) { return *p; }
EMU_NOSAN unsigned long long __tsan_atomic64_load(const volatile unsigned long long* p, int) { return *p; }
EMU_NOSAN unsigned long long __tsan_atomic64_fetch_add(volatile unsigned long long* p, unsigned long long v, int) { const unsigned long long o = *p; *p = o + v; return o; }
}
#endif

// ---------------------------------------------------------------- the CUDA names the kernel uses
#define threadIdx (emu::cur->tidx)
#define blockIdx (emu::cur->cta->bidx)
inline dim3& blockDim = emu::g.bdim;      // (objects, not macros: host code has struct members of these names)
inline dim3& gridDim = emu::g.gdim;
#define HOUGH_DYN_SMEM(name) unsigned char* name = emu::dyn_smem()

EMU_NOSAN inline void __syncthreads(int line = __builtin_LINE()) { int a, o, c; emu::wait_barrier(emu::cur->cta->bar, 1, a, o, c, 1, line); }
EMU_NOSAN inline int __syncthreads_and(int p, int line = __builtin_LINE()) { int a, o, c; emu::wait_barrier(emu::cur->cta->bar, p, a, o, c, 1, line); return a; }
EMU_NOSAN inline int __syncthreads_or(int p, int line = __builtin_LINE()) { int a, o, c; emu::wait_barrier(emu::cur->cta->bar, p, a, o, c, 1, line); return o; }
EMU_NOSAN inline int __syncthreads_count(int p, int line = __builtin_LINE()) { int a, o, c; emu::wait_barrier(emu::cur->cta->bar, p, a, o, c, 1, line); return c; }
inline void __threadfence() {}

EMU_NOSAN inline void need_full_mask(unsigned m) { if (m != 0xffffffffu) emu::die("only full-mask warp collectives are emulated"); }
EMU_NOSAN inline int __shfl_sync(unsigned m, int v, int src) { need_full_mask(m); return (int)emu::warp_exchange((unsigned)v)[src & 31]; }
EMU_NOSAN inline int __shfl_up_sync(unsigned m, int v, int d) {
    need_full_mask(m);
    const int lane = (int)(emu::cur->tidx.x & 31);
    const unsigned* b = emu::warp_exchange((unsigned)v);
    return lane >= d ? (int)b[lane - d] : v;
}
EMU_NOSAN inline unsigned __ballot_sync(unsigned m, int p) {
    need_full_mask(m);
    const unsigned* b = emu::warp_exchange(p ? 1u : 0u);
    unsigned r = 0;
    for (int l = 0; l < 32; ++l) r |= (b[l] & 1u) << l;
    return r;
}
EMU_NOSAN inline int __all_sync(unsigned m, int p) { return __ballot_sync(m, p) == 0xffffffffu; }
EMU_NOSAN inline int __shfl_xor_sync(unsigned m, int v, int d) {
    need_full_mask(m);
    const int lane = (int)(emu::cur->tidx.x & 31);
    return (int)emu::warp_exchange((unsigned)v)[(lane ^ d) & 31];
}
EMU_NOSAN inline unsigned long long __shfl_xor_sync(unsigned m, unsigned long long v, int d) {
    const unsigned lo = (unsigned)__shfl_xor_sync(m, (int)(unsigned)v, d), hi = (unsigned)__shfl_xor_sync(m, (int)(unsigned)(v >> 32), d);
    return (unsigned long long)lo | ((unsigned long long)hi << 32);
}
EMU_NOSAN inline void __syncwarp() { emu::warp_exchange(0u, true); }

inline unsigned atomicAdd(unsigned* p, unsigned v) { return __atomic_fetch_add(p, v, __ATOMIC_RELAXED); }
inline int atomicAdd(int* p, int v) { return __atomic_fetch_add(p, v, __ATOMIC_RELAXED); }
inline unsigned atomicAnd(unsigned* p, unsigned v) { return __atomic_fetch_and(p, v, __ATOMIC_RELAXED); }
inline int atomicOr(int* p, int v) { return __atomic_fetch_or(p, v, __ATOMIC_RELAXED); }
inline unsigned atomicOr(unsigned* p, unsigned v) { return __atomic_fetch_or(p, v, __ATOMIC_RELAXED); }
template <class T> inline T __ldg(const T* p) { return *p; }
EMU_NOSAN inline size_t __cvta_generic_to_shared(const void* p) {
    const ptrdiff_t off = (const unsigned char*)p - emu::cur->cta->smem.ptr;
    if (off < 0 || (size_t)off >= emu::cur->cta->smem.bytes) emu::die("cvta of a pointer outside the CTA's shared memory");
    return (size_t)emu::SHARED_WINDOW + (size_t)off;
}

inline unsigned __float_as_uint(float f) { unsigned u; memcpy(&u, &f, 4); return u; }
inline float __uint_as_float(unsigned u) { float f; memcpy(&f, &u, 4); return f; }
// one rounding per operation: this file is compiled with -ffp-contract=off and without fast-math
inline float __fmul_rn(float a, float b) { volatile float r = a * b; return r; }
inline float __fadd_rn(float a, float b) { volatile float r = a + b; return r; }
inline float __fdiv_rn(float a, float b) { volatile float r = a / b; return r; }
inline float __fsub_rn(float a, float b) { volatile float r = a - b; return r; }
inline double __dadd_rn(double a, double b) { volatile double r = a + b; return r; }
inline double __dsub_rn(double a, double b) { volatile double r = a - b; return r; }
inline double __dmul_rn(double a, double b) { volatile double r = a * b; return r; }
inline double __ddiv_rn(double a, double b) { volatile double r = a / b; return r; }
inline float __fadd_rd(float a, float b) {        // round toward minus infinity: exact in double, then step down if needed
    const double s = (double)a + (double)b;
    float r = (float)s;
    if (std::isfinite(r) && (double)r > s) r = std::nextafterf(r, -INFINITY);
    return r;
}
inline int __popc(unsigned x) { return __builtin_popcount(x); }
inline int __ffs(unsigned x) { return __builtin_ffs((int)x); }
inline unsigned umax3(unsigned a, unsigned b, unsigned c) { return a > b ? (a > c ? a : c) : (b > c ? b : c); }
inline unsigned __vimax3_u32(unsigned a, unsigned b, unsigned c) { return umax3(a, b, c); }
inline unsigned __vimax3_u16x2(unsigned a, unsigned b, unsigned c) {
    return umax3(a & 0xFFFFu, b & 0xFFFFu, c & 0xFFFFu) | (umax3(a >> 16, b >> 16, c >> 16) << 16);
}
inline unsigned __vibmax_u16x2(unsigned a, unsigned b, bool* hi, bool* lo) {   // per-half max; *hi / *lo: a's half is >= b's
    *lo = (a & 0xFFFFu) >= (b & 0xFFFFu);
    *hi = (a >> 16) >= (b >> 16);
    return ((*lo ? a : b) & 0xFFFFu) | ((*hi ? a : b) & 0xFFFF0000u);
}
template <class T> inline T min(T a, T b) { return a < b ? a : b; }
template <class T> inline T max(T a, T b) { return a > b ? a : b; }
inline unsigned min(unsigned a, int b) { return a < (unsigned)b ? a : (unsigned)b; }

namespace cooperative_groups {
struct cluster_group {
    EMU_NOSAN unsigned block_rank() const { return (unsigned)emu::cur->cta->rank; }
    EMU_NOSAN void sync(int line = __builtin_LINE()) const { int a, o, c; emu::wait_barrier(emu::g.cluster_bar, 1, a, o, c, 2, line); }
    EMU_NOSAN void* map_shared_rank(void* p, int rank) const {
        const ptrdiff_t off = (unsigned char*)p - emu::cur->cta->smem.ptr;
        if (off < 0 || (size_t)off >= emu::cur->cta->smem.bytes) emu::die("map_shared_rank of a pointer outside shared memory");
        if (rank < 0 || rank >= emu::g.csize) emu::die("map_shared_rank: bad rank");
        return emu::g.ctas[(size_t)rank].smem.ptr + off;
    }
};
inline cluster_group this_cluster() { return cluster_group(); }
}  // namespace cooperative_groups
