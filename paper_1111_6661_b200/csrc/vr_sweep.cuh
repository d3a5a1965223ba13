// vr_sweep.cuh — the two ways a reduction kernel walks voxels: a flat,
// 16-byte aligned array (VR_LINEAR) and a box inside a strided array (one brick of VR_BRICKED_HALO1 without
// its halo).  HBM-bound streams: persistent grid, grid-stride 16-byte loads that bypass L1
// (ld.global.nc.L1::no_allocate), four loads in flight per thread.  `visit(v)` is called once per voxel.
#pragma once
#include "vr_internal.h"

namespace vr {

constexpr int kSweepThreads = 512;

// order-preserving uint encoding of a float (IEEE totalOrder: -0 before +0): a < b <=> enc(a) < enc(b)
__device__ __forceinline__ unsigned int enc_f(float f)
{
    const unsigned int b = __float_as_uint(f);
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float dec_f(unsigned int u)
{
    return __uint_as_float((u & 0x80000000u) ? (u & 0x7fffffffu) : ~u);
}

__device__ __forceinline__ float4 ld_stream4(const float4 *p)
{
#ifdef VR_SIMT_HOST
    return *p;
#else
    float4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p));
    return r;
#endif
}

template <typename Visit>
__device__ __forceinline__ void sweep_flat(const float *__restrict__ v, unsigned long long n, Visit &&visit)
{
    const unsigned long long n4 = n >> 2;
    const float4 *v4 = reinterpret_cast<const float4 *>(v);
    const unsigned long long stride = (unsigned long long)gridDim.x * kSweepThreads;
    unsigned long long i = (unsigned long long)blockIdx.x * kSweepThreads + threadIdx.x;
    for (; i + 3 * stride < n4; i += 4 * stride) {
        const float4 x0 = ld_stream4(v4 + i), x1 = ld_stream4(v4 + i + stride);
        const float4 x2 = ld_stream4(v4 + i + 2 * stride), x3 = ld_stream4(v4 + i + 3 * stride);
        visit(x0.x); visit(x0.y); visit(x0.z); visit(x0.w);
        visit(x1.x); visit(x1.y); visit(x1.z); visit(x1.w);
        visit(x2.x); visit(x2.y); visit(x2.z); visit(x2.w);
        visit(x3.x); visit(x3.y); visit(x3.z); visit(x3.w);
    }
    for (; i < n4; i += stride) {
        const float4 x = ld_stream4(v4 + i);
        visit(x.x); visit(x.y); visit(x.z); visit(x.w);
    }
    if (blockIdx.x == 0 && threadIdx.x < (unsigned)(n & 3)) visit(v[(n4 << 2) + threadIdx.x]);
}

// one warp per row of the box, lanes along x
template <typename Visit>
__device__ __forceinline__ void sweep_box(const BoxK &b, Visit &&visit)
{
    const int lane = threadIdx.x & 31;
    const long long rows = (long long)b.ey * b.ez;
    const long long wstride = (long long)gridDim.x * (kSweepThreads / 32);
    for (long long r = (long long)blockIdx.x * (kSweepThreads / 32) + (threadIdx.x >> 5); r < rows; r += wstride) {
        const float *row = b.base + (r % b.ey) * b.sy + (r / b.ey) * b.sz;
        for (int x = lane; x < b.ex; x += 32) visit(__ldg(row + x));
    }
}

}  // namespace vr
