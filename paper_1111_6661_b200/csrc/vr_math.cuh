// vr_math.cuh — the canonical float32 operation sequences of DESIGN.md §3 (SURVEY.md §8(c)
// C.1-C.6) as device functions.  Every operation is an explicit round-to-nearest intrinsic, so
// nothing can be contracted or reassociated by the compiler: __fmaf_rn is one fused multiply-add,
// everything else is a separately rounded IEEE-754 binary32 operation, denormals kept.
#pragma once
#ifndef VR_SIMT_HOST               // tests/simt/simt_host.h (force-included by the host emulation build) stands in
#include <cuda_runtime.h>
#include <math_constants.h>
#endif
#include <stdint.h>

namespace vr {

// exact-ends lerp (C.0): a at f = 0, b at f = 1, bit for bit
__device__ __forceinline__ float lerp_ee(float a, float b, float f)
{
    return __fmaf_rn(f, b, __fmaf_rn(-f, a, a));
}

// Two independent correctly rounded float32 fused multiply-adds in one instruction (sm_100 FFMA2):
// (a.x*b.x + c.x, a.y*b.y + c.y).  Same results as two __fmaf_rn; halves the issue slots of the lerps.
__device__ __forceinline__ float2 fma2_rn(float2 a, float2 b, float2 c)
{
#ifdef VR_SIMT_HOST
    return make_float2(__fmaf_rn(a.x, b.x, c.x), __fmaf_rn(a.y, b.y, c.y));
#else
    unsigned long long ua, ub, uc, ud;
    asm("mov.b64 %0, {%1, %2};" : "=l"(ua) : "f"(a.x), "f"(a.y));
    asm("mov.b64 %0, {%1, %2};" : "=l"(ub) : "f"(b.x), "f"(b.y));
    asm("mov.b64 %0, {%1, %2};" : "=l"(uc) : "f"(c.x), "f"(c.y));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(ud) : "l"(ua), "l"(ub), "l"(uc));
    float2 d;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(d.x), "=f"(d.y) : "l"(ud));
    return d;
#endif
}

// exact-ends lerp of two pairs with one fraction: (L(a.x,b.x,f), L(a.y,b.y,f))
__device__ __forceinline__ float2 lerp_ee2(float2 a, float2 b, float f)
{
    return fma2_rn(make_float2(f, f), b, fma2_rn(make_float2(-f, -f), a, a));
}

struct CamK {                       // kernel-side copy of vr_camera (C.1)
    float o0[3], ou[3], ov[3], d0[3], du[3], dv[3];
    float step;
    float t_min;                    // 1 - ert_alpha, rounded once (C.5)
    int width, height;              // the pixels this render produces: the whole image, or the lattice of a progressive pass
    int sub, sx, sy;                // progressive pass (VR_SUBSAMPLE): lattice pixel (i', j') is image pixel (sub i' + sx, sub j' + sy)
};

struct VolK {                       // the voxel box and how to address it
    const float *base;              // voxel (ox,oy,oz) of this view of the data
    long long sy, sz;               // element strides of y and z (x stride = 1)
    int nx, ny, nz;                 // full volume dims (for C.2 slabs and C.3 clamps)
    int ox, oy, oz;                 // index origin of `base` (0 for a linear volume; B*b for a pool slot)
};

struct Ray {
    float d[3], oc[3];              // unit direction; origin - 0.5 (C.3)
    float t_first, t_exit;
};

// C.1 + C.2.  Returns false for a miss.
__device__ __forceinline__ bool make_ray(const CamK &c, int nx, int ny, int nz, int i, int j, Ray &r)
{
    const float px = __fadd_rn((float)i, 0.5f), py = __fadd_rn((float)j, 0.5f);
    float o[3], g[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        o[a] = __fmaf_rn(py, c.ov[a], __fmaf_rn(px, c.ou[a], c.o0[a]));
        g[a] = __fmaf_rn(py, c.dv[a], __fmaf_rn(px, c.du[a], c.d0[a]));
    }
    const float len = __fsqrt_rn(__fmaf_rn(g[2], g[2], __fmaf_rn(g[1], g[1], __fmul_rn(g[0], g[0]))));
    const float n[3] = { (float)nx, (float)ny, (float)nz };
    float t_enter = 0.0f, t_exit = CUDART_INF_F;
    bool hit = true;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        r.d[a] = __fdiv_rn(g[a], len);
        float lo, hi;
        if (r.d[a] != 0.0f) {
            const float inv = __fdiv_rn(1.0f, r.d[a]);
            const float ta = __fmul_rn(__fsub_rn(0.0f, o[a]), inv);
            const float tb = __fmul_rn(__fsub_rn(n[a], o[a]), inv);
            lo = fminf(ta, tb); hi = fmaxf(ta, tb);
        } else {
            if (o[a] < 0.0f || o[a] > n[a]) hit = false;
            lo = -CUDART_INF_F; hi = CUDART_INF_F;
        }
        t_enter = fmaxf(t_enter, lo);
        t_exit = fminf(t_exit, hi);
        r.oc[a] = __fsub_rn(o[a], 0.5f);
    }
    if (!(t_exit > t_enter)) hit = false;
    r.t_first = __fmaf_rn(0.5f, c.step, t_enter);
    // C.2 defines samples for k < 2^24 only ((float)k must be exact): the march loops end at that k at the
    // latest, whatever the step, and a direction that is not finite (g = 0: t_exit = +inf or NaN) is a miss
    if (!(t_exit < CUDART_INF_F)) hit = false;
    r.t_exit = fminf(t_exit, __fmaf_rn(16777216.0f, c.step, r.t_first));
    return hit;
}

// C.3 index/fraction of one axis
__device__ __forceinline__ void axis_cell(float t, float d, float oc, int n, int &i0, float &f)
{
    float q = __fmaf_rn(t, d, oc);
    q = fminf(fmaxf(q, 0.0f), (float)(n - 1));
    i0 = min(__float2int_rd(q), n - 2);
    f = __fsub_rn(q, (float)i0);
}

// C.3 value from the 8 corner voxels
__device__ __forceinline__ float trilerp(float v000, float v100, float v010, float v110, float v001, float v101,
                                         float v011, float v111, float fx, float fy, float fz)
{
    const float c00 = lerp_ee(v000, v100, fx);
    const float c10 = lerp_ee(v010, v110, fx);
    const float c01 = lerp_ee(v001, v101, fx);
    const float c11 = lerp_ee(v011, v111, fx);
    const float c0 = lerp_ee(c00, c10, fy);
    const float c1 = lerp_ee(c01, c11, fy);
    return lerp_ee(c0, c1, fz);
}

// C.3 with the x and y lerps paired over z (same operations and operands as trilerp, 8 instructions)
__device__ __forceinline__ float trilerp_packed(float v000, float v100, float v010, float v110, float v001, float v101,
                                                float v011, float v111, float fx, float fy, float fz)
{
    const float2 c0x = lerp_ee2(make_float2(v000, v001), make_float2(v100, v101), fx);      // (c00, c01)
    const float2 c1x = lerp_ee2(make_float2(v010, v011), make_float2(v110, v111), fx);      // (c10, c11)
    const float2 cy = lerp_ee2(c0x, c1x, fy);                                               // (c0, c1)
    return lerp_ee(cy.x, cy.y, fz);
}

// C.4: post-interpolative classification from a 257-entry shared-memory table (entry 256 is a
// pad copy of entry 255 so that i+1 is always readable; i is clamped to 254 as in C.4 anyway)
__device__ __forceinline__ float4 classify(const float4 *tf, float scale, float bias, float s)
{
    const float u = __saturatef(__fmaf_rn(s, scale, bias));       // NaN -> 0, like fmin(fmax(.,0),1)
    const float x = __fmul_rn(u, 255.0f);
    const int i = min(__float2int_rz(x), 254);
    const float f = __fsub_rn(x, (float)i);
    const float4 a = tf[i], b = tf[i + 1];
    return make_float4(lerp_ee(a.x, b.x, f), lerp_ee(a.y, b.y, f), lerp_ee(a.z, b.z, f), lerp_ee(a.w, b.w, f));
}

// C.5: one front-to-back compositing step
__device__ __forceinline__ void composite(float4 rgba, float &Cr, float &Cg, float &Cb, float &T)
{
    const float w = __fmul_rn(T, rgba.w);
    Cr = __fmaf_rn(w, rgba.x, Cr);
    Cg = __fmaf_rn(w, rgba.y, Cg);
    Cb = __fmaf_rn(w, rgba.z, Cb);
    T = __fsub_rn(T, w);
}

}  // namespace vr
