// vr_range.cuh — which samples of a ray belong to a box of base indices (bricks, staging tiles).
// Reading C.7: sample k is owned by the box iff its clamped base index i0 lies in
// [lo, hi] on every axis.  i0_a(k) is monotone in k, so the owned samples form ONE contiguous
// k-range.  It is estimated from the slab interval of the ownership cell and then FIXED UP by
// evaluating the exact predicate at the ends, so every sample has exactly one owner whatever the
// rounding of the estimate.
#pragma once
#include "vr_math.cuh"

namespace vr {

__device__ __forceinline__ bool owned(int nx, int ny, int nz, const Ray &r, float step, const int *lo, const int *hi,
                                      int k)
{
    if (k < 0) return false;
    const float t = __fmaf_rn((float)k, step, r.t_first);
    if (!(t < r.t_exit)) return false;
    int i; float f;
    axis_cell(t, r.d[0], r.oc[0], nx, i, f);
    if (i < lo[0] || i > hi[0]) return false;
    axis_cell(t, r.d[1], r.oc[1], ny, i, f);
    if (i < lo[1] || i > hi[1]) return false;
    axis_cell(t, r.d[2], r.oc[2], nz, i, f);
    return i >= lo[2] && i <= hi[2];
}

__device__ __forceinline__ bool box_range(int nx, int ny, int nz, const Ray &r, float step, const int *lo,
                                          const int *hi, int &k_lo, int &k_hi)
{
    const int n[3] = { nx, ny, nz };
    float t_lo = r.t_first, t_hi = r.t_exit;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const float qlo = lo[a] == 0 ? -CUDART_INF_F : (float)lo[a];
        const float qhi = hi[a] == n[a] - 2 ? CUDART_INF_F : (float)(hi[a] + 1);
        if (r.d[a] != 0.0f) {
            const float inv = __fdividef(1.0f, r.d[a]);
            const float t0 = (qlo - r.oc[a]) * inv, t1 = (qhi - r.oc[a]) * inv;
            t_lo = fmaxf(t_lo, fminf(t0, t1));
            t_hi = fminf(t_hi, fmaxf(t0, t1));
        } else {
            int i; float f;
            axis_cell(0.0f, 0.0f, r.oc[a], n[a], i, f);          // q == oc for every sample
            if (i < lo[a] || i > hi[a]) return false;
        }
    }
    const float inv_step = __fdividef(1.0f, step);
    const float pad_f = fminf(2.0f + 8e-6f * fabsf(r.t_exit) * inv_step, 64.0f);   // rounding slack of the estimate
    const float a_f = (t_lo - r.t_first) * inv_step, b_f = (t_hi - r.t_first) * inv_step;
    if (!(b_f + pad_f >= a_f - pad_f)) return false;
    const int pad = (int)pad_f;
    int kl = (int)fminf(fmaxf(ceilf(a_f), 0.0f), 16777216.0f) - pad;
    int kh = (int)fminf(fmaxf(floorf(b_f), -1.0f), 16777216.0f) + pad;
    kl = max(kl, 0);
    while (kl <= kh && !owned(nx, ny, nz, r, step, lo, hi, kl)) ++kl;
    if (kl > kh) return false;
    while (owned(nx, ny, nz, r, step, lo, hi, kl - 1)) --kl;
    while (kh > kl && !owned(nx, ny, nz, r, step, lo, hi, kh)) --kh;
    while (owned(nx, ny, nz, r, step, lo, hi, kh + 1)) ++kh;
    k_lo = kl; k_hi = kh;
    return true;
}

}  // namespace vr
