// simt_host.h — TEST INFRASTRUCTURE: a small "CUDA on the CPU" layer that lets the library's own .cu sources
// (kernels AND host runtime) be compiled by g++ and executed on the host cores, thread by thread, so that
// tests/test_simt_parity.py can run the real kernel code against the oracle on a box without a GPU.
//
// What it is: every CUDA thread of a CTA is a fiber (own stack, cooperative switches); CTAs run one after
// another; __syncthreads and the warp collectives (*_sync votes, shuffles, reductions) block a fiber until the
// other non-exited threads of the CTA / warp named by the mask have arrived, exactly the rendezvous the
// hardware performs.  Shared memory is one buffer per CTA; global memory is host memory; the runtime API is
// a synchronous stand-in (every stream operation completes before the call returns — a legal schedule of any
// correctly ordered stream program).  Device allocations sit between guard pages, so an out-of-range global
// access of a kernel is a SIGSEGV here instead of an Xid on a GPU.
//
// What it is NOT: a product path.  Nothing under paper_1111_6661_b200/ loads, links or falls back to it; the
// shipped libvr.so is built by nvcc for sm_100a only.  It says nothing about timing, memory-ordering races
// between streams, or instruction selection.  Float arithmetic: the canonical sequences use explicit
// round-to-nearest intrinsics, mapped here to the same IEEE-754 binary32 operations (g++ -mfma
// -ffp-contract=off), so results are expected to be bit-identical to the GPU's and to the oracle's.
#pragma once
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <string.h>

#include <algorithm>
#include <type_traits>

// ------------------------------------------------------------------ qualifiers
#define __global__
#define __device__
#define __host__
#define __forceinline__ inline __attribute__((always_inline))
#define __restrict__
#define __launch_bounds__(...)
#define __shared__ static
#define __constant__ static
#define VR_SIMT_HOST 1

// ------------------------------------------------------------------ vector types
struct float2 { float x, y; };
struct alignas(16) float4 { float x, y, z, w; };
struct int2 { int x, y; };
struct alignas(16) int4 { int x, y, z, w; };
struct uint2 { unsigned int x, y; };
struct alignas(16) uint4 { unsigned int x, y, z, w; };
struct uint3 { unsigned int x, y, z; };
struct dim3 {
    unsigned int x, y, z;
    dim3(unsigned int x_ = 1, unsigned int y_ = 1, unsigned int z_ = 1) : x(x_), y(y_), z(z_) {}
};
inline float2 make_float2(float x, float y) { return float2{ x, y }; }
inline float4 make_float4(float x, float y, float z, float w) { return float4{ x, y, z, w }; }
inline int2 make_int2(int x, int y) { return int2{ x, y }; }
inline uint2 make_uint2(unsigned int x, unsigned int y) { return uint2{ x, y }; }
inline uint4 make_uint4(unsigned int x, unsigned int y, unsigned int z, unsigned int w) { return uint4{ x, y, z, w }; }

#define CUDART_INF_F (__builtin_inff())
#define CUDART_NAN_F (__builtin_nanf(""))

// ------------------------------------------------------------------ runtime API stand-in (simt_runtime.cpp)
typedef int cudaError_t;
enum { cudaSuccess = 0, cudaErrorMemoryAllocation = 2, cudaErrorInvalidValue = 1 };
typedef struct simt_stream_s *cudaStream_t;
typedef struct simt_event_s *cudaEvent_t;
enum cudaMemcpyKind { cudaMemcpyHostToHost = 0, cudaMemcpyHostToDevice = 1, cudaMemcpyDeviceToHost = 2, cudaMemcpyDeviceToDevice = 3, cudaMemcpyDefault = 4 };
enum cudaMemoryType { cudaMemoryTypeUnregistered = 0, cudaMemoryTypeHost = 1, cudaMemoryTypeDevice = 2, cudaMemoryTypeManaged = 3 };
struct cudaPointerAttributes { cudaMemoryType type; int device; void *devicePointer; void *hostPointer; };
enum { cudaStreamNonBlocking = 1, cudaEventDisableTiming = 2, cudaHostAllocMapped = 2, cudaHostAllocDefault = 0 };
enum cudaDeviceAttr { cudaDevAttrMultiProcessorCount = 16 };

extern "C" {
cudaError_t cudaMalloc(void **p, size_t n);
cudaError_t cudaFree(void *p);
cudaError_t cudaMallocHost(void **p, size_t n);
cudaError_t cudaHostAlloc(void **p, size_t n, unsigned int flags);
cudaError_t cudaFreeHost(void *p);
cudaError_t cudaHostGetDevicePointer(void **d, void *h, unsigned int flags);
cudaError_t cudaMemcpy(void *d, const void *s, size_t n, cudaMemcpyKind k);
cudaError_t cudaMemcpyAsync(void *d, const void *s, size_t n, cudaMemcpyKind k, cudaStream_t st);
cudaError_t cudaMemcpy2DAsync(void *d, size_t dp, const void *s, size_t sp, size_t w, size_t h, cudaMemcpyKind k, cudaStream_t st);
cudaError_t cudaMemsetAsync(void *d, int v, size_t n, cudaStream_t st);
cudaError_t cudaStreamCreateWithFlags(cudaStream_t *s, unsigned int flags);
cudaError_t cudaStreamDestroy(cudaStream_t s);
cudaError_t cudaStreamSynchronize(cudaStream_t s);
cudaError_t cudaStreamWaitEvent(cudaStream_t s, cudaEvent_t e, unsigned int flags);
cudaError_t cudaEventCreateWithFlags(cudaEvent_t *e, unsigned int flags);
cudaError_t cudaEventDestroy(cudaEvent_t e);
cudaError_t cudaEventRecord(cudaEvent_t e, cudaStream_t s);
cudaError_t cudaEventSynchronize(cudaEvent_t e);
cudaError_t cudaEventQuery(cudaEvent_t e);
cudaError_t cudaGetDevice(int *d);
cudaError_t cudaSetDevice(int d);
cudaError_t cudaDeviceGetAttribute(int *v, cudaDeviceAttr a, int dev);
cudaError_t cudaPointerGetAttributes(cudaPointerAttributes *a, const void *p);
cudaError_t cudaMemGetInfo(size_t *free_b, size_t *total_b);
cudaError_t cudaGetLastError(void);
const char *cudaGetErrorString(cudaError_t e);
}
template <typename T> inline cudaError_t cudaMalloc(T **p, size_t n) { return cudaMalloc((void **)p, n); }
template <typename T> inline cudaError_t cudaMallocHost(T **p, size_t n) { return cudaMallocHost((void **)p, n); }
template <typename T> inline cudaError_t cudaHostAlloc(T **p, size_t n, unsigned int f) { return cudaHostAlloc((void **)p, n, f); }
template <typename T> inline cudaError_t cudaHostGetDevicePointer(T **d, void *h, unsigned int f) { return cudaHostGetDevicePointer((void **)d, h, f); }

// ------------------------------------------------------------------ execution model (simt_runtime.cpp)
namespace simt {

struct Builtins { uint3 tid, bid; dim3 bdim, gdim; };
extern Builtins g_cur;                     // built-in variables of the running fiber
extern unsigned char *g_dyn_smem;          // dynamic shared memory of the running CTA
extern unsigned long long g_counters[16];  // VR_TEST_COUNT(i) of vr_internal.h
// memory-traffic model of a warp's corner loads (VR_TRACE_CORNER_LOADS of vr_internal.h): when g_trace is set, every
// lane of the warp deposits the addresses of its four row pointers; per load instruction the distinct 128-byte lines
// and 32-byte sectors (relative to `base`, which is 256-byte aligned on hardware) of the active lanes are counted
extern int g_trace;
extern unsigned long long g_trace_stats[8];  // warp iterations, sampling lanes, load instructions, lines, sectors, (quad what-if) loads, lines, loading lanes
void trace_corner_loads(bool sampled, bool loads, const void *base, const void *p0, const void *p1, const void *p2, const void *p3);

struct KernelBody { void (*fn)(void *); void *ctx; };
void launch_cta_grid(dim3 grid, dim3 block, size_t dyn_smem, KernelBody body);

template <typename F>
inline void launch(dim3 grid, dim3 block, size_t dyn_smem, F &&f)
{
    using Fn = typename std::remove_reference<F>::type;
    KernelBody b{ [](void *c) { (*static_cast<Fn *>(c))(); }, (void *)&f };
    launch_cta_grid(grid, block, dyn_smem, b);
}

// rendezvous primitives: every non-exited thread named by `mask` (warp) / every non-exited thread (CTA)
// deposits a 64-bit value; all get the table of deposits back
struct WarpTable { uint64_t v[32]; uint32_t present; };
const WarpTable &warp_exchange(uint32_t mask, uint64_t value);
int cta_barrier(int pred, int mode);       // mode 0 plain, 1 or, 2 and, 3 count
inline int lane_id() { return (int)((g_cur.tid.x + g_cur.bdim.x * (g_cur.tid.y + g_cur.bdim.y * g_cur.tid.z)) & 31u); }

}  // namespace simt

#define threadIdx (::simt::g_cur.tid)
#define blockIdx (::simt::g_cur.bid)
#define blockDim (::simt::g_cur.bdim)
#define gridDim (::simt::g_cur.gdim)

// ------------------------------------------------------------------ synchronisation and warp collectives
inline void __syncthreads() { ::simt::cta_barrier(0, 0); }
inline int __syncthreads_or(int p) { return ::simt::cta_barrier(p, 1); }
inline int __syncthreads_and(int p) { return ::simt::cta_barrier(p, 2); }
inline int __syncthreads_count(int p) { return ::simt::cta_barrier(p, 3); }
inline void __syncwarp(unsigned int mask = 0xffffffffu) { ::simt::warp_exchange(mask, 0); }
inline void __threadfence() {}
inline void __threadfence_block() {}

inline unsigned int __ballot_sync(unsigned int mask, int pred)
{
    const ::simt::WarpTable &t = ::simt::warp_exchange(mask, pred ? 1u : 0u);
    unsigned int r = 0;
    for (int l = 0; l < 32; ++l) if ((t.present >> l & 1u) && t.v[l]) r |= 1u << l;
    return r;
}
inline int __any_sync(unsigned int mask, int pred) { return __ballot_sync(mask, pred) != 0u; }
inline int __all_sync(unsigned int mask, int pred)
{
    const ::simt::WarpTable &t = ::simt::warp_exchange(mask, pred ? 1u : 0u);
    for (int l = 0; l < 32; ++l) if ((t.present >> l & 1u) && !t.v[l]) return 0;
    return 1;
}
inline unsigned int __activemask() { return ::simt::warp_exchange(0u, 0).present; }   // mask 0: whoever is alive

namespace simt {
template <typename T> inline uint64_t to_bits(T v) { uint64_t b = 0; static_assert(sizeof(T) <= 8, ""); memcpy(&b, &v, sizeof(T)); return b; }
template <typename T> inline T from_bits(uint64_t b) { T v; memcpy(&v, &b, sizeof(T)); return v; }
template <typename T> inline T shfl_from(unsigned int mask, T v, int src, int width)
{
    const int lane = lane_id();
    const WarpTable &t = warp_exchange(mask, to_bits(v));
    (void)width;
    if (src < 0 || src > 31 || !(t.present >> src & 1u)) return v;      // undefined on hardware; keep own value
    (void)lane;
    return from_bits<T>(t.v[src]);
}
}  // namespace simt
template <typename T> inline T __shfl_sync(unsigned int mask, T v, int src, int width = 32)
{
    const int lane = ::simt::lane_id();
    return ::simt::shfl_from(mask, v, (lane & ~(width - 1)) | (src & (width - 1)), width);
}
template <typename T> inline T __shfl_xor_sync(unsigned int mask, T v, int lanemask, int width = 32)
{
    const int lane = ::simt::lane_id();
    const int src = lane ^ lanemask;
    return ::simt::shfl_from(mask, v, (src & ~(width - 1)) == (lane & ~(width - 1)) ? src : lane, width);
}
template <typename T> inline T __shfl_down_sync(unsigned int mask, T v, unsigned int delta, int width = 32)
{
    const int lane = ::simt::lane_id();
    const int src = lane + (int)delta;
    return ::simt::shfl_from(mask, v, (src & ~(width - 1)) == (lane & ~(width - 1)) ? src : lane, width);
}
template <typename T> inline T __shfl_up_sync(unsigned int mask, T v, unsigned int delta, int width = 32)
{
    const int lane = ::simt::lane_id();
    const int src = lane - (int)delta;
    return ::simt::shfl_from(mask, v, src >= (lane & ~(width - 1)) ? src : lane, width);
}
#define SIMT_REDUCE(NAME, T, INIT, OP)                                              \
    inline T NAME(unsigned int mask, T v)                                           \
    {                                                                               \
        const ::simt::WarpTable &t = ::simt::warp_exchange(mask, ::simt::to_bits(v)); \
        T r = INIT;                                                                 \
        for (int l = 0; l < 32; ++l)                                                \
            if (t.present >> l & 1u) { const T x = ::simt::from_bits<T>(t.v[l]); r = OP; } \
        return r;                                                                   \
    }
SIMT_REDUCE(__reduce_min_sync, int, 0x7fffffff, (x < r ? x : r))
SIMT_REDUCE(__reduce_max_sync, int, (-0x7fffffff - 1), (x > r ? x : r))
SIMT_REDUCE(__reduce_add_sync, int, 0, (r + x))
SIMT_REDUCE(__reduce_min_sync, unsigned int, 0xffffffffu, (x < r ? x : r))
SIMT_REDUCE(__reduce_max_sync, unsigned int, 0u, (x > r ? x : r))
SIMT_REDUCE(__reduce_add_sync, unsigned int, 0u, (r + x))
SIMT_REDUCE(__reduce_or_sync, unsigned int, 0u, (r | x))
SIMT_REDUCE(__reduce_and_sync, unsigned int, 0xffffffffu, (r & x))
#undef SIMT_REDUCE
template <typename T> inline unsigned int __match_any_sync(unsigned int mask, T v)
{
    const int lane = ::simt::lane_id();
    const ::simt::WarpTable &t = ::simt::warp_exchange(mask, ::simt::to_bits(v));
    unsigned int r = 0;
    for (int l = 0; l < 32; ++l) if ((t.present >> l & 1u) && t.v[l] == t.v[lane]) r |= 1u << l;
    return r;
}

// ------------------------------------------------------------------ atomics (one fiber runs at a time)
template <typename T> inline T atomicAdd(T *p, T v) { const T o = *p; *p = o + v; return o; }
template <typename T> inline T atomicMin(T *p, T v) { const T o = *p; *p = v < o ? v : o; return o; }
template <typename T> inline T atomicMax(T *p, T v) { const T o = *p; *p = v > o ? v : o; return o; }
template <typename T> inline T atomicOr(T *p, T v) { const T o = *p; *p = o | v; return o; }
template <typename T> inline T atomicAnd(T *p, T v) { const T o = *p; *p = o & v; return o; }
template <typename T> inline T atomicExch(T *p, T v) { const T o = *p; *p = v; return o; }
template <typename T> inline T atomicCAS(T *p, T c, T v) { const T o = *p; if (o == c) *p = v; return o; }

// ------------------------------------------------------------------ arithmetic intrinsics (IEEE-754 binary32)
inline float __fmaf_rn(float a, float b, float c) { return fmaf(a, b, c); }
inline float __fadd_rn(float a, float b) { return a + b; }
inline float __fsub_rn(float a, float b) { return a - b; }
inline float __fmul_rn(float a, float b) { return a * b; }
inline float __fdiv_rn(float a, float b) { return a / b; }
inline float __fsqrt_rn(float a) { return sqrtf(a); }
inline float __fdividef(float a, float b) { return a / b; }      // approximate on hardware; only used for estimates
inline float __saturatef(float a) { return a != a ? 0.0f : fminf(fmaxf(a, 0.0f), 1.0f); }
// cvt.r?i.s32.f32 saturates and turns NaN into 0 (a C cast is undefined there)
inline int simt_cvt_s32(float r) { return r != r ? 0 : r >= 2147483648.0f ? 2147483647 : r <= -2147483648.0f ? (-2147483647 - 1) : (int)r; }
inline int __float2int_rd(float a) { return simt_cvt_s32(floorf(a)); }
inline int __float2int_rz(float a) { return simt_cvt_s32(truncf(a)); }
inline int __float2int_rn(float a) { return simt_cvt_s32(nearbyintf(a)); }
inline int __float2int_ru(float a) { return simt_cvt_s32(ceilf(a)); }
inline unsigned int __float_as_uint(float f) { unsigned int u; memcpy(&u, &f, 4); return u; }
inline float __uint_as_float(unsigned int u) { float f; memcpy(&f, &u, 4); return f; }
inline int __float_as_int(float f) { int u; memcpy(&u, &f, 4); return u; }
inline float __int_as_float(int u) { float f; memcpy(&f, &u, 4); return f; }
inline int __popc(unsigned int x) { return __builtin_popcount(x); }
inline int __popcll(unsigned long long x) { return __builtin_popcountll(x); }
inline int __ffs(int x) { return __builtin_ffs(x); }
inline int __clz(int x) { return x ? __builtin_clz((unsigned int)x) : 32; }
inline unsigned int __brev(unsigned int x)
{
    unsigned int r = 0;
    for (int i = 0; i < 32; ++i) r |= (x >> i & 1u) << (31 - i);
    return r;
}
template <typename T> inline T __ldg(const T *p) { return *p; }
template <typename T> inline T __ldcs(const T *p) { return *p; }
template <typename T> inline void __stcs(T *p, T v) { *p = v; }
using std::max;
using std::min;
inline unsigned int min(unsigned int a, int b) { return a < (unsigned int)b ? a : (unsigned int)b; }
inline long long min(long long a, int b) { return a < b ? a : (long long)b; }
inline long long max(long long a, int b) { return a > b ? a : (long long)b; }
