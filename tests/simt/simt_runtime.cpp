// simt_runtime.cpp — TEST INFRASTRUCTURE (see simt_host.h): the fiber scheduler that executes the CTAs of a
// kernel launch on the host, the rendezvous behind __syncthreads / the *_sync warp collectives, and a
// synchronous stand-in for the CUDA runtime calls the library makes.  x86-64 System V only.
#include "simt_host.h"

#include <stdio.h>
#include <stdlib.h>
#include <sys/mman.h>
#include <unistd.h>

#include <map>
#include <mutex>
#include <vector>

#if !defined(__x86_64__)
#error "the SIMT host emulation switches stacks with x86-64 assembly"
#endif

// void simt_switch(void **save_sp, void *new_sp): store the callee-saved state on the current stack, switch
asm(".text\n"
    ".globl simt_switch\n"
    ".type simt_switch,@function\n"
    "simt_switch:\n"
    "    pushq %rbp\n    pushq %rbx\n    pushq %r12\n    pushq %r13\n    pushq %r14\n    pushq %r15\n"
    "    movq %rsp, (%rdi)\n"
    "    movq %rsi, %rsp\n"
    "    popq %r15\n    popq %r14\n    popq %r13\n    popq %r12\n    popq %rbx\n    popq %rbp\n"
    "    ret\n"
    ".size simt_switch, .-simt_switch\n");
extern "C" void simt_switch(void **save_sp, void *new_sp);

namespace simt {

Builtins g_cur;
unsigned char *g_dyn_smem = nullptr;
unsigned long long g_counters[16] = {};
int g_trace = 0;
unsigned long long g_trace_stats[8] = {};

namespace {

constexpr size_t kStackBytes = 256 << 10;
constexpr int kMaxThreads = 1024;

struct Fiber {
    void *sp = nullptr;
    unsigned char *stack = nullptr;
    bool done = true;
    const volatile unsigned int *wait_gen = nullptr;     // blocked until *wait_gen != wait_val
    unsigned int wait_val = 0;
    uint3 tid;
};

struct WarpState {
    uint64_t deposit[32];
    uint32_t arrived = 0, alive = 0, need_mask = 0;
    volatile unsigned int gen = 0;
    WarpTable table[2];
};

struct CtaState {
    int n_threads = 0, n_alive = 0, arrived = 0;
    int acc_or = 0, acc_and = 1, acc_cnt = 0;
    int result[2] = { 0, 0 };
    volatile unsigned int gen = 0;
};

std::mutex g_launch_mutex;               // one launch at a time (the emulation is single-threaded by design)
std::vector<Fiber> g_fibers;
std::vector<WarpState> g_warps;
CtaState g_cta;
void *g_sched_sp = nullptr;
int g_running = -1;
KernelBody g_body;
dim3 g_bdim, g_gdim;
uint3 g_bid;

void yield_to_scheduler()
{
    Fiber &f = g_fibers[g_running];
    simt_switch(&f.sp, g_sched_sp);
    // resumed: restore the built-ins of this fiber
    g_cur.tid = f.tid; g_cur.bid = g_bid; g_cur.bdim = g_bdim; g_cur.gdim = g_gdim;
}

void complete_warp(WarpState &w)
{
    WarpTable &t = w.table[(w.gen + 1) & 1u];
    for (int l = 0; l < 32; ++l) t.v[l] = w.deposit[l];
    t.present = w.arrived;
    w.arrived = 0;
    w.need_mask = 0;
    w.gen = w.gen + 1;
}

void complete_cta()
{
    CtaState &c = g_cta;
    int *r = &c.result[(c.gen + 1) & 1u];
    r[0] = (c.acc_or ? 1 : 0) | (c.acc_and ? 2 : 0) | (c.acc_cnt << 2);
    c.arrived = 0; c.acc_or = 0; c.acc_and = 1; c.acc_cnt = 0;
    c.gen = c.gen + 1;
}

void fiber_main()
{
    g_body.fn(g_body.ctx);
    // the thread exits: it no longer takes part in any rendezvous, and pending ones may now be complete
    const int me = g_running;
    Fiber &f = g_fibers[me];
    WarpState &w = g_warps[me >> 5];
    w.alive &= ~(1u << (me & 31));
    if (w.arrived) {
        const uint32_t need = (w.need_mask ? w.need_mask : w.alive) & w.alive;
        if ((w.arrived & need) == need) complete_warp(w);
    }
    g_cta.n_alive--;
    if (g_cta.arrived > 0 && g_cta.arrived >= g_cta.n_alive) complete_cta();
    f.done = true;
    simt_switch(&f.sp, g_sched_sp);
    abort();                                  // never resumed
}

extern "C" void simt_fiber_entry() { fiber_main(); }

void prepare_fiber(Fiber &f)
{
    if (!f.stack) {
        void *m = mmap(nullptr, kStackBytes + 4096, PROT_READ | PROT_WRITE, MAP_PRIVATE | MAP_ANONYMOUS | MAP_STACK, -1, 0);
        if (m == MAP_FAILED) { perror("simt: mmap stack"); abort(); }
        mprotect(m, 4096, PROT_NONE);         // stack overflow guard
        f.stack = (unsigned char *)m + 4096;
    }
    uintptr_t top = ((uintptr_t)f.stack + kStackBytes) & ~(uintptr_t)15;
    uint64_t *s = (uint64_t *)top;
    *--s = 0;                                 // fake return address of the entry function
    *--s = (uint64_t)(uintptr_t)&simt_fiber_entry;
    for (int i = 0; i < 6; ++i) *--s = 0;     // rbp rbx r12 r13 r14 r15
    f.sp = s;
    f.done = false;
    f.wait_gen = nullptr;
}

void run_cta(size_t dyn_smem)
{
    const int n = (int)(g_bdim.x * g_bdim.y * g_bdim.z);
    if ((int)g_fibers.size() < n) g_fibers.resize(n);
    g_warps.assign((n + 31) / 32, WarpState());
    g_cta = CtaState();
    g_cta.n_threads = g_cta.n_alive = n;
    std::vector<unsigned char> smem(dyn_smem + 16, 0xCD);        // uninitialised on hardware: poison
    g_dyn_smem = smem.data();
    for (int t = 0; t < n; ++t) {
        Fiber &f = g_fibers[t];
        prepare_fiber(f);
        f.tid.x = (unsigned)t % g_bdim.x;
        f.tid.y = ((unsigned)t / g_bdim.x) % g_bdim.y;
        f.tid.z = (unsigned)t / (g_bdim.x * g_bdim.y);
        g_warps[t >> 5].alive |= 1u << (t & 31);
    }
    int remaining = n, cur = 0, idle_scan = 0;
    while (remaining > 0) {
        Fiber &f = g_fibers[cur];
        const bool runnable = !f.done && (!f.wait_gen || *f.wait_gen != f.wait_val);
        if (runnable) {
            idle_scan = 0;
            f.wait_gen = nullptr;
            g_running = cur;
            g_cur.tid = f.tid; g_cur.bid = g_bid; g_cur.bdim = g_bdim; g_cur.gdim = g_gdim;
            simt_switch(&g_sched_sp, f.sp);
            g_running = -1;
            if (f.done) --remaining;
        } else if (++idle_scan > n) {
            fprintf(stderr, "simt: deadlock in CTA (%u,%u,%u): every live thread waits at a barrier or warp collective "
                            "that the others never reach\n", g_bid.x, g_bid.y, g_bid.z);
            abort();
        }
        cur = cur + 1 == n ? 0 : cur + 1;
    }
    g_dyn_smem = nullptr;
}

}  // namespace

void launch_cta_grid(dim3 grid, dim3 block, size_t dyn_smem, KernelBody body)
{
    std::lock_guard<std::mutex> lock(g_launch_mutex);
    const unsigned long long n = (unsigned long long)block.x * block.y * block.z;
    if (n == 0 || n > kMaxThreads || grid.x == 0 || grid.y == 0 || grid.z == 0) {
        fprintf(stderr, "simt: invalid launch configuration grid (%u,%u,%u) block (%u,%u,%u)\n", grid.x, grid.y, grid.z,
                block.x, block.y, block.z);
        abort();                              // cudaErrorInvalidConfiguration on hardware: a bug in the caller
    }
    if (dyn_smem > (227u << 10)) { fprintf(stderr, "simt: %zu bytes of dynamic shared memory\n", dyn_smem); abort(); }
    g_body = body; g_bdim = block; g_gdim = grid;
    for (unsigned z = 0; z < grid.z; ++z)
        for (unsigned y = 0; y < grid.y; ++y)
            for (unsigned x = 0; x < grid.x; ++x) {
                g_bid.x = x; g_bid.y = y; g_bid.z = z;
                run_cta(dyn_smem);
            }
}

const WarpTable &warp_exchange(uint32_t mask, uint64_t value)
{
    const int me = g_running;
    WarpState &w = g_warps[me >> 5];
    const int lane = me & 31;
    if (mask != 0 && !(mask >> lane & 1u)) {
        fprintf(stderr, "simt: lane %d calls a *_sync collective with a mask (%08x) that does not name it\n", lane, mask);
        abort();
    }
    if (w.arrived && w.need_mask != mask) {
        fprintf(stderr, "simt: lanes of one warp meet in collectives with different masks (%08x vs %08x)\n", w.need_mask, mask);
        abort();
    }
    w.need_mask = mask;
    w.deposit[lane] = value;
    w.arrived |= 1u << lane;
    const unsigned int my_gen = w.gen;
    const uint32_t need = (mask ? mask : w.alive) & w.alive;
    if ((w.arrived & need) == need) complete_warp(w);
    else {
        Fiber &f = g_fibers[me];
        f.wait_gen = &w.gen; f.wait_val = my_gen;
        yield_to_scheduler();
    }
    return w.table[(my_gen + 1) & 1u];
}

// sampled: the lane takes a sample in this warp iteration; loads: it also loads the sample's 8 voxels (it may still hold them)
void trace_corner_loads(bool sampled, bool loads, const void *base, const void *p0, const void *p1, const void *p2, const void *p3)
{
    const void *ptr[4] = { p0, p1, p2, p3 };
    const int lane = g_running & 31;
    const uint64_t kIdle = ~0ull, kNoLoad = ~0ull - 1;
    for (int r = 0; r < 4; ++r) {
        const uint64_t off = !sampled ? kIdle : !loads ? kNoLoad : (uint64_t)((const char *)ptr[r] - (const char *)base);
        const WarpTable &t0 = warp_exchange(0u, off);                // every live lane of the warp arrives here
        WarpTable t = t0;
        int first = -1, n_smp = 0, n_ld = 0;
        for (int l = 0; l < 32; ++l) {
            if (!(t.present >> l & 1u) || t.v[l] == kIdle) { t.v[l] = ~0ull; continue; }
            if (first < 0) first = l;
            ++n_smp;
            if (t.v[l] == kNoLoad) t.v[l] = ~0ull; else ++n_ld;      // below, ~0 = takes no part in the loads
        }
        if (lane != first) continue;                                 // one lane does the counting
        if (r == 0) { g_trace_stats[0] += 1; g_trace_stats[1] += (unsigned long long)n_smp; g_trace_stats[7] += (unsigned long long)n_ld; }
        if (n_ld == 0) continue;
        for (int e = 0; e < 2; ++e) {                                // the loads of p and p + 1 element
            uint64_t lines[32], sectors[32];
            int nl = 0, ns = 0;
            for (int l = 0; l < 32; ++l) {
                if (!(t.present >> l & 1u) || t.v[l] == ~0ull) continue;
                const uint64_t a = t.v[l] + 4u * (unsigned)e, ln = a >> 7, sc = a >> 5;
                bool seen = false;
                for (int k = 0; k < nl; ++k) seen = seen || lines[k] == ln;
                if (!seen) lines[nl++] = ln;
                seen = false;
                for (int k = 0; k < ns; ++k) seen = seen || sectors[k] == sc;
                if (!seen) sectors[ns++] = sc;
            }
            g_trace_stats[2] += 1; g_trace_stats[3] += (unsigned long long)nl; g_trace_stats[4] += (unsigned long long)ns;
        }
        // what-if: ONE 16-byte load of the aligned quad that holds element p, plus a scalar load of p + 1 only for the
        // lanes whose p is the last element of its quad (the alternative to two scalar loads per row)
        for (int e = 0; e < 2; ++e) {
            uint64_t lines[32];
            int nl = 0, n_lanes = 0;
            for (int l = 0; l < 32; ++l) {
                if (!(t.present >> l & 1u) || t.v[l] == ~0ull) continue;
                const bool last = ((t.v[l] >> 2) & 3u) == 3u;
                if (e == 1 && !last) continue;
                ++n_lanes;
                const uint64_t ln = (e == 0 ? t.v[l] : t.v[l] + 4u) >> 7;
                bool seen = false;
                for (int k = 0; k < nl; ++k) seen = seen || lines[k] == ln;
                if (!seen) lines[nl++] = ln;
            }
            if (n_lanes) { g_trace_stats[5] += 1; g_trace_stats[6] += (unsigned long long)nl; }
        }
    }
}

int cta_barrier(int pred, int mode)
{
    const int me = g_running;
    CtaState &c = g_cta;
    c.arrived++;
    if (pred) { c.acc_or = 1; c.acc_cnt++; } else c.acc_and = 0;
    const unsigned int my_gen = c.gen;
    if (c.arrived >= c.n_alive) complete_cta();
    else {
        Fiber &f = g_fibers[me];
        f.wait_gen = &c.gen; f.wait_val = my_gen;
        yield_to_scheduler();
    }
    const int r = c.result[(my_gen + 1) & 1u];
    return mode == 0 ? 0 : mode == 1 ? (r & 1) : mode == 2 ? ((r >> 1) & 1) : (r >> 2);
}

}  // namespace simt

// ====================================================================== runtime API stand-in
namespace {

struct Alloc { size_t bytes; void *map; size_t map_bytes; int kind; };   // kind 1 host (pinned), 2 device
std::map<uintptr_t, Alloc> g_allocs;
std::mutex g_alloc_mutex;
size_t g_device_bytes = 0;
size_t g_device_capacity = (size_t)4 << 30;

// n bytes whose END sits against an inaccessible page (and whose start is preceded by one): reads or writes past
// either end of the allocation fault.  The start is 16-byte aligned (256 on hardware; the library needs 16).
void *guarded_alloc(size_t n, int kind)
{
    const size_t page = 4096, body = (n + page - 1) / page * page;
    const size_t total = body + 2 * page;
    unsigned char *m = (unsigned char *)mmap(nullptr, total, PROT_READ | PROT_WRITE, MAP_PRIVATE | MAP_ANONYMOUS, -1, 0);
    if (m == MAP_FAILED) return nullptr;
    mprotect(m, page, PROT_NONE);
    mprotect(m + page + body, page, PROT_NONE);
    const size_t slack = (body - n) & ~(size_t)15;
    unsigned char *p = m + page + slack;
    memset(m + page, 0xA5, body);                                    // not zero: uninitialised on hardware
    std::lock_guard<std::mutex> lock(g_alloc_mutex);
    g_allocs[(uintptr_t)p] = Alloc{ n, m, total, kind };
    if (kind == 2) g_device_bytes += n;
    return p;
}

int guarded_free(void *p)
{
    if (!p) return 0;
    std::lock_guard<std::mutex> lock(g_alloc_mutex);
    auto it = g_allocs.find((uintptr_t)p);
    if (it == g_allocs.end()) { fprintf(stderr, "simt: free of an unknown pointer %p\n", p); abort(); }
    if (it->second.kind == 2) g_device_bytes -= it->second.bytes;
    munmap(it->second.map, it->second.map_bytes);
    g_allocs.erase(it);
    return 0;
}

int kind_of(const void *p)
{
    std::lock_guard<std::mutex> lock(g_alloc_mutex);
    auto it = g_allocs.upper_bound((uintptr_t)p);
    if (it == g_allocs.begin()) return 0;
    --it;
    return (uintptr_t)p < it->first + it->second.bytes ? it->second.kind : 0;
}

struct simt_dummy { int x; };

}  // namespace

extern "C" {

// test hooks: "device" and "pinned host" buffers for inputs and outputs the tests own
__attribute__((visibility("default"))) void *simt_device_alloc(size_t n) { return guarded_alloc(n ? n : 1, 2); }
__attribute__((visibility("default"))) void *simt_pinned_alloc(size_t n) { return guarded_alloc(n ? n : 1, 1); }
__attribute__((visibility("default"))) void simt_free(void *p) { guarded_free(p); }
__attribute__((visibility("default"))) size_t simt_device_bytes_in_use(void) { return g_device_bytes; }
// event counters the kernels bump through VR_TEST_COUNT (vr_internal.h): tests assert that a code path really ran
__attribute__((visibility("default"))) unsigned long long simt_counter(int i) { return i >= 0 && i < 16 ? simt::g_counters[i] : 0; }
__attribute__((visibility("default"))) void simt_reset_counters(void) { for (auto &c : simt::g_counters) c = 0; }
__attribute__((visibility("default"))) void simt_trace(int on) { simt::g_trace = on; for (auto &c : simt::g_trace_stats) c = 0; }
__attribute__((visibility("default"))) unsigned long long simt_trace_stat(int i) { return i >= 0 && i < 8 ? simt::g_trace_stats[i] : 0; }
__attribute__((visibility("default"))) void simt_set_device_capacity(size_t n) { g_device_capacity = n; }

cudaError_t cudaMalloc(void **p, size_t n)
{
    if (g_device_bytes + n > g_device_capacity) { *p = nullptr; return cudaErrorMemoryAllocation; }
    *p = guarded_alloc(n ? n : 1, 2);
    return *p ? cudaSuccess : cudaErrorMemoryAllocation;
}
cudaError_t cudaFree(void *p) { guarded_free(p); return cudaSuccess; }
cudaError_t cudaMallocHost(void **p, size_t n) { *p = guarded_alloc(n ? n : 1, 1); return *p ? cudaSuccess : cudaErrorMemoryAllocation; }
cudaError_t cudaHostAlloc(void **p, size_t n, unsigned int) { return cudaMallocHost(p, n); }
cudaError_t cudaFreeHost(void *p) { guarded_free(p); return cudaSuccess; }
cudaError_t cudaHostGetDevicePointer(void **d, void *h, unsigned int) { *d = h; return cudaSuccess; }
cudaError_t cudaMemcpy(void *d, const void *s, size_t n, cudaMemcpyKind) { memmove(d, s, n); return cudaSuccess; }
cudaError_t cudaMemcpyAsync(void *d, const void *s, size_t n, cudaMemcpyKind, cudaStream_t) { memmove(d, s, n); return cudaSuccess; }
cudaError_t cudaMemcpy2DAsync(void *d, size_t dp, const void *s, size_t sp, size_t w, size_t h, cudaMemcpyKind, cudaStream_t)
{
    for (size_t r = 0; r < h; ++r) memmove((char *)d + r * dp, (const char *)s + r * sp, w);
    return cudaSuccess;
}
cudaError_t cudaMemsetAsync(void *d, int v, size_t n, cudaStream_t) { memset(d, v, n); return cudaSuccess; }
cudaError_t cudaStreamCreateWithFlags(cudaStream_t *s, unsigned int) { *s = (cudaStream_t) new simt_dummy(); return cudaSuccess; }
cudaError_t cudaStreamDestroy(cudaStream_t s) { delete (simt_dummy *)s; return cudaSuccess; }
cudaError_t cudaStreamSynchronize(cudaStream_t) { return cudaSuccess; }
cudaError_t cudaStreamWaitEvent(cudaStream_t, cudaEvent_t, unsigned int) { return cudaSuccess; }
cudaError_t cudaEventCreateWithFlags(cudaEvent_t *e, unsigned int) { *e = (cudaEvent_t) new simt_dummy(); return cudaSuccess; }
cudaError_t cudaEventDestroy(cudaEvent_t e) { delete (simt_dummy *)e; return cudaSuccess; }
cudaError_t cudaEventRecord(cudaEvent_t, cudaStream_t) { return cudaSuccess; }
cudaError_t cudaEventSynchronize(cudaEvent_t) { return cudaSuccess; }
cudaError_t cudaEventQuery(cudaEvent_t) { return cudaSuccess; }
cudaError_t cudaGetDevice(int *d) { *d = 0; return cudaSuccess; }
cudaError_t cudaSetDevice(int) { return cudaSuccess; }
cudaError_t cudaDeviceGetAttribute(int *v, cudaDeviceAttr, int) { *v = 3; return cudaSuccess; }    // "3 SMs": small persistent grids
cudaError_t cudaPointerGetAttributes(cudaPointerAttributes *a, const void *p)
{
    const int k = kind_of(p);
    a->type = k == 2 ? cudaMemoryTypeDevice : k == 1 ? cudaMemoryTypeHost : cudaMemoryTypeUnregistered;
    a->device = 0; a->devicePointer = (void *)p; a->hostPointer = (void *)p;
    return cudaSuccess;
}
cudaError_t cudaMemGetInfo(size_t *free_b, size_t *total_b)
{
    *total_b = g_device_capacity;
    *free_b = g_device_capacity > g_device_bytes ? g_device_capacity - g_device_bytes : 0;
    return cudaSuccess;
}
cudaError_t cudaGetLastError(void) { return cudaSuccess; }
const char *cudaGetErrorString(cudaError_t e) { return e == cudaSuccess ? "no error" : e == cudaErrorMemoryAllocation ? "out of memory" : "error"; }

}  // extern "C"
