// vr_beamgeom.cuh — geometry of a BEAM (the rays of one 16x16 pixel tile) shared by the host plans
// and the kernels of the two beam paths (vr_beam.cu: TMA slab boxes; vr_shear.cu: sheared planes).
// Nothing here takes part in the canonical arithmetic of a sample (vr_math.cuh): these functions
// only bound WHERE the samples of a beam can fall, conservatively (kMargin >> float32 error).
#pragma once
#include <cuda_runtime.h>
#include <math.h>

#include "vr_math.cuh"

namespace vr {

constexpr int kBW = 16, kBH = 16;                    // beam = 16 x 16 pixels, 8 warps of 8 x 4
constexpr int kStrip = 16;                           // beams per strip row (scheduling order)
constexpr float kMargin = 0.05f;                     // voxels; >> float32 error of any position (< 2e-3 at 2^14)

struct BeamLine { float Au, Ru, Av, Rv; };           // transverse position on the plane p_a = c:  p_u = Au + c Ru

__host__ __device__ inline void beam_axes(int a, int &u, int &v) { u = a == 0 ? 1 : 0; v = a == 2 ? 1 : 2; }

__host__ __device__ inline void cam_ray_at(const CamK &c, float px, float py, float o[3], float g[3])
{
    for (int a = 0; a < 3; ++a) {
        o[a] = fmaf(py, c.ov[a], fmaf(px, c.ou[a], c.o0[a]));
        g[a] = fmaf(py, c.dv[a], fmaf(px, c.du[a], c.d0[a]));
    }
}

// z before y before x on ties: the longer the contiguous rows of a staged plane, the better
__host__ __device__ inline int principal_axis(const float g[3])
{
    const float ax = fabsf(g[0]), ay = fabsf(g[1]), az = fabsf(g[2]);
    return (az >= ax && az >= ay) ? 2 : (ay >= ax ? 1 : 0);
}

// the line of the ray through pixel-space point (px,py), parameterised by the principal coordinate.
// false: the ray does not travel along `sgn` of axis a, or is more oblique than |d_a| = 0.3.
__host__ __device__ inline bool beam_line(const CamK &c, float px, float py, int a, int sgn, BeamLine &L)
{
    float o[3], g[3];
    cam_ray_at(c, px, py, o, g);
    int u, v;
    beam_axes(a, u, v);
    const float ga = g[a], len2 = g[0] * g[0] + g[1] * g[1] + g[2] * g[2];
    if (!(ga * (float)sgn > 0.0f) || !(ga * ga >= 0.09f * len2)) return false;
    L.Ru = g[u] / ga; L.Rv = g[v] / ga;
    L.Au = o[u] - o[a] * L.Ru; L.Av = o[v] - o[a] * L.Rv;
    return true;
}

// the two planes that bound the sample positions a slab of base indices [lo, hi] can own (C.7:
// ownership cell [lo + 1/2, hi + 3/2), outer cells reach the volume faces)
__host__ __device__ inline void slab_planes(int lo, int hi, int na, float &cA, float &cB)
{
    cA = lo <= 0 ? 0.0f : (float)lo + 0.5f;
    cB = hi >= na - 2 ? (float)na : (float)hi + 1.5f;
}

__host__ __device__ inline int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

__host__ __device__ inline int floor_clamped(float q)
{
    q = fminf(fmaxf(q, -1.0e6f), 1.0e6f);
    return (int)floorf(q);
}

// Voxels of DATA plane P (index along the principal axis) that samples of the beam bounded by the four
// corner lines L[0..3] can read.  Plane P is read by samples whose base index is P - 1 or P, i.e. whose
// principal coordinate lies in [P - 1/2, P + 3/2] (to the volume face for the outer base indices, which
// also own the outer half voxel); between two planes the beam is
// the convex hull of its corner lines, so the extremes are taken at the corners on the two end planes.
// A sample at transverse coordinate p reads base index floor(p - 1/2) (clamped to [0, n-2]) and its +1
// neighbour.  raw: widths before the clamp to the volume (a convex function of P: checking both ends of a
// beam bounds every plane in between).
__host__ __device__ inline void plane_rect(const BeamLine L[4], int P, int na, int nu, int nv, bool raw, int &u0,
                                           int &v0, int &w, int &h)
{
    // plane P serves base indices P - 1 and P; the outer base indices also own the outer half voxel (clamp to edge)
    const float c0 = P <= 1 ? 0.0f : (float)P - 0.5f, c1 = P >= na - 2 ? (float)na : (float)P + 1.5f;
    float umin = 3.0e38f, umax = -3.0e38f, vmin = 3.0e38f, vmax = -3.0e38f;
    for (int k = 0; k < 4; ++k) {
        const float ua = fmaf(c0, L[k].Ru, L[k].Au), ub = fmaf(c1, L[k].Ru, L[k].Au);
        const float va = fmaf(c0, L[k].Rv, L[k].Av), vb = fmaf(c1, L[k].Rv, L[k].Av);
        umin = fminf(umin, fminf(ua, ub)); umax = fmaxf(umax, fmaxf(ua, ub));
        vmin = fminf(vmin, fminf(va, vb)); vmax = fmaxf(vmax, fmaxf(va, vb));
    }
    int iu0 = floor_clamped(umin - 0.5f - kMargin), iu1 = floor_clamped(umax - 0.5f + kMargin);
    int iv0 = floor_clamped(vmin - 0.5f - kMargin), iv1 = floor_clamped(vmax - 0.5f + kMargin);
    if (!raw) {
        iu0 = clampi(iu0, 0, nu - 2); iu1 = clampi(iu1, 0, nu - 2);
        iv0 = clampi(iv0, 0, nv - 2); iv1 = clampi(iv1, 0, nv - 2);
    }
    u0 = iu0; v0 = iv0;
    w = iu1 - iu0 + 2; h = iv1 - iv0 + 2;
}

// Largest raw plane rectangle over the planes [Pa, Pb] of a beam, up to one voxel: the raw size is convex in the
// plane index over the interior planes (all serve a 2-voxel range) but not across the two outer planes at
// either volume face (they serve the outer half voxel too), so the three planes at each end are evaluated
// (tests/geom_check.cu checks the bound by brute force).
__host__ __device__ inline void beam_rect_bound(const BeamLine L[4], int Pa, int Pb, int na, int nu, int nv, int &w, int &h)
{
    w = 0; h = 0;
    for (int e = 0; e < 6; ++e) {
        const int P = e < 3 ? Pa + e : Pb - (e - 3);
        if (P < Pa || P > Pb) continue;
        int u0, v0, wp, hp;
        plane_rect(L, P, na, nu, nv, true, u0, v0, wp, hp);
        w = wp > w ? wp : w; h = hp > h ? hp : h;
    }
}

// Range [c_lo, c_hi] of the principal coordinate over which the cross-section of the beam (the quadrilateral of
// its four corner lines) can overlap the volume: [0, na] minus the c-intervals on which all four corner points
// lie beyond the same face of the (u,v) rectangle (by more than a voxel).  Conservative on purpose — a beam that
// straddles a volume edge or contains the whole volume has rays inside the volume although none of its corner
// lines is.  false: no overlap at all.
__host__ __device__ inline bool beam_c_range(const BeamLine L[4], int na, int nu, int nv, float &c_lo, float &c_hi)
{
    // E[i] = open interval of c on which  s * (p_k(c) - bound) > 0  for all four corners k
    float e_lo[4], e_hi[4];
    for (int i = 0; i < 4; ++i) {
        const bool on_u = i < 2, high = (i & 1) != 0;
        const float bound = high ? (float)(on_u ? nu : nv) + 1.0f : -1.0f, sg = high ? 1.0f : -1.0f;
        float lo = -3.0e38f, hi = 3.0e38f;
        for (int k = 0; k < 4; ++k) {
            const float A = sg * ((on_u ? L[k].Au : L[k].Av) - bound), R = sg * (on_u ? L[k].Ru : L[k].Rv);   // A + R c > 0
            if (R > 0.0f) lo = fmaxf(lo, -A / R);
            else if (R < 0.0f) hi = fminf(hi, -A / R);
            else if (!(A > 0.0f)) { lo = 3.0e38f; hi = -3.0e38f; }
        }
        e_lo[i] = lo; e_hi[i] = hi;
    }
    c_lo = 0.0f; c_hi = (float)na;
    for (int pass = 0; pass < 4; ++pass)
        for (int i = 0; i < 4; ++i) {
            if (e_lo[i] < e_hi[i] && e_lo[i] <= c_lo && c_lo < e_hi[i]) c_lo = e_hi[i];
            if (e_lo[i] < e_hi[i] && e_lo[i] < c_hi && c_hi <= e_hi[i]) c_hi = e_lo[i];
        }
    return c_hi >= c_lo;
}

// ---------------------------------------------------------------- step schedule of the sheared-plane path
// (vr_shear.cu; also executed on the host by the schedule model of tests/geom_check.cu).  The data planes of a
// beam, iw_min .. iw_max + 1, are numbered by their ordinal j along the direction of travel; base plane ordinal
// jb needs data ordinals jb and jb + 1.  Step 0 loads G + 1 planes, every later step G; after the planes up to
// ordinal m have landed the base ordinals below m can be marched.  Plane ordinal j lives in ring slot j mod NS.
struct StepPlan { int nload, wlo, wn; };       // planes to load before the step; base planes [wlo, wlo + wn) it marches

__host__ __device__ inline int plane_of_ordinal(int sgn, int iw_min, int iw_max, int j)
{
    return sgn > 0 ? iw_min + j : iw_max + 1 - j;
}
__host__ __device__ inline int ring_slot(int j, int NS) { return j % NS; }

// next step of the schedule; next_ord = first plane ordinal not yet planned, wstart = first base ordinal not yet marched
__host__ __device__ inline StepPlan plan_window(bool first, int G, int sgn, int iw_min, int iw_max, int &next_ord, int &wstart)
{
    const int n_planes = iw_max - iw_min + 2;
    int nload = first ? G + 1 : G;
    if (nload > n_planes - next_ord) nload = n_planes - next_ord;
    if (nload < 0) nload = 0;
    next_ord += nload;
    const int wend = next_ord - 1 > wstart ? next_ord - 1 : wstart;
    StepPlan S;
    S.nload = nload;
    S.wlo = sgn > 0 ? iw_min + wstart : iw_max - wend + 1;
    S.wn = wend - wstart;
    wstart = wend;
    return S;
}

}  // namespace vr
