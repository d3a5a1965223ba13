// vr_plan.h — host-only geometry of the per-frame brick plan (reading C.7): the position-space
// cell a brick owns, its visibility key and its conservative screen rectangle.  Plain C++ (no CUDA), so that
// tests/plan_check.cpp can brute-force it on the host.
#pragma once
#include <algorithm>
#include <cmath>

#include "../../include/vr.h"

namespace vr {

inline bool zero3(const float *a) { return a[0] == 0.0f && a[1] == 0.0f && a[2] == 0.0f; }

inline double det3(const double a[3], const double b[3], const double c[3])
{
    return a[0] * (b[1] * c[2] - b[2] * c[1]) - b[0] * (a[1] * c[2] - a[2] * c[1]) + c[0] * (a[1] * b[2] - a[2] * b[1]);
}

// ownership cell, in sample-position space, of the base indices [ilo, ihi] of one axis of length n (C.7: base
// index i0 = floor(p - 1/2) owns p in [i0 + 1/2, i0 + 3/2); the outer base indices reach the volume faces);
// 0.01 voxel of slack for the float32 ray arithmetic
inline void brick_cell(int ilo, int ihi, int n, double &lo, double &hi)
{
    lo = (ilo == 0 ? 0.0 : ilo + 0.5) - 0.01;
    hi = (ihi == n - 2 ? (double)n : ihi + 1.5) + 0.01;
}

// one axis' term of the visibility key of brick index b (edge B): squared distance of the eye to the
// ownership-lattice centre B (b + 1/2) + 1/2 (perspective), or centre . d0 (orthographic)
inline double brick_key_term(bool perspective, double B, unsigned int b, double o0, double d0)
{
    const double centre = B * (b + 0.5) + 0.5;
    if (perspective) { const double e = o0 - centre; return e * e; }
    return centre * d0;
}

// conservative screen rectangle [x0,x1) x [y0,y1) of an axis-aligned box of sample positions
inline void box_rect(const vr_camera *c, bool perspective, const double lo[3], const double hi[3], int &x0, int &y0,
                     int &x1, int &y1)
{
    const int W = (int)c->width, H = (int)c->height;
    double mnx = 1e300, mny = 1e300, mxx = -1e300, mxy = -1e300;
    bool full = false;
    for (int corner = 0; corner < 8 && !full; ++corner) {
        double P[3];
        for (int a = 0; a < 3; ++a) P[a] = (corner >> a & 1) ? hi[a] : lo[a];
        double x, y;
        if (perspective) {            // d0 + x du + y dv = lambda (P - o0)
            double m0[3], m1[3], m2[3], rhs[3];
            for (int a = 0; a < 3; ++a) { m0[a] = c->du[a]; m1[a] = c->dv[a]; m2[a] = -(P[a] - (double)c->o0[a]); rhs[a] = -(double)c->d0[a]; }
            const double D = det3(m0, m1, m2);
            if (std::fabs(D) < 1e-300) { full = true; break; }
            x = det3(rhs, m1, m2) / D; y = det3(m0, rhs, m2) / D;
            const double lambda = det3(m0, m1, rhs) / D;
            if (!(lambda > 1e-9)) { full = true; break; }       // corner at or behind the eye
        } else {                      // o0 + x ou + y ov + t d0 = P
            double m0[3], m1[3], m2[3], rhs[3];
            for (int a = 0; a < 3; ++a) { m0[a] = c->ou[a]; m1[a] = c->ov[a]; m2[a] = c->d0[a]; rhs[a] = P[a] - (double)c->o0[a]; }
            const double D = det3(m0, m1, m2);
            if (std::fabs(D) < 1e-300) { full = true; break; }
            x = det3(rhs, m1, m2) / D; y = det3(m0, rhs, m2) / D;
        }
        if (!std::isfinite(x) || !std::isfinite(y)) { full = true; break; }
        mnx = std::min(mnx, x); mxx = std::max(mxx, x); mny = std::min(mny, y); mxy = std::max(mxy, y);
    }
    if (full) { x0 = 0; y0 = 0; x1 = W; y1 = H; return; }
    // pixel i has x = i + 0.5; one extra pixel of slack for float32 ray arithmetic
    const double fx0 = std::floor(mnx - 0.5) - 1.0, fy0 = std::floor(mny - 0.5) - 1.0;
    const double fx1 = std::ceil(mxx - 0.5) + 2.0, fy1 = std::ceil(mxy - 0.5) + 2.0;
    x0 = (int)std::min(std::max(fx0, 0.0), (double)W); x1 = (int)std::min(std::max(fx1, 0.0), (double)W);
    y0 = (int)std::min(std::max(fy0, 0.0), (double)H); y1 = (int)std::min(std::max(fy1, 0.0), (double)H);
}

}  // namespace vr
