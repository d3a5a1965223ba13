// vr_shear.cu — sheared-plane beam ray casting: the in-HBM fast path of vr_render for VR_LINEAR
// volumes ("the GPU part" of the case study;
// PAPER.md:L66 sub-cube partitioning, applied here per beam and per frame instead of per GPU).
//
// Design.  As in vr_beam.cu a CTA owns a BEAM — the rays of one 16x16 pixel tile, one
// thread per ray, ray state (C, T) / m in registers from the first sample to the last, so the
// recurrence of C.5 runs in k order and early termination is exact — and the beam is traversed along
// its PRINCIPAL axis a, its samples marched out of shared memory.  What differs is how the voxels
// are staged, because profiles/r1a_beam_tma_ncu.md showed the TMA slab boxes bound by the
// shared-memory data pipe (7.2 wavefronts per LDS) and staging 6.5 x the voxels the samples touch:
//   * each DATA plane (one index q along a) is staged as its own rectangle — the bounding rectangle
//     of the beam's cross-section on that plane, + the trilinear halo — at its own origin, so the
//     staged volume follows the beam (a sheared prism) instead of bounding it with one box;
//   * planes are copied with 4-byte cp.async (LDGSTS), which can write ANY layout: rows have a
//     pitch PU and planes a pitch PP chosen (host plan, residue tables below) so that the 32 lanes
//     of a warp — which at equal k sit on a surface parallel to the volume face they entered
//     through, i.e. vary in two of the three indices — spread over the 32 banks.  TMA writes 16-byte
//     granules, so all its y/z pitches are multiples of 4 words and an x-face pattern has 8 banks.
//   * the planes live in a RING of NS fixed-size slots (plane ordinal mod NS).  A step marches the
//     base planes of a window of G + 1 resident data planes while the next G planes are in flight
//     (NS >= 2G + 1), so no plane is loaded twice; one __syncthreads per step; warp 0 plans two
//     steps ahead (triple-buffered step records).  A table indexed by (q mod 64) holds, per
//     resident plane, the shared-memory address of its voxel (0,0): a corner address is
//     table[q] + 4 (iu + PU iv).
//
// Arithmetic.  Identical to k_march_full: positions, indices and fractions come from the canonical
// GLOBAL position (vr_math.cuh); the shared-memory address is formed by integer arithmetic on the
// base indices.  Results are bit-identical to the ray-major kernel.
#include <algorithm>
#include <climits>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "vr_beamgeom.cuh"
#include "vr_internal.h"

namespace vr {

namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kMaxLoad = 17;                         // planes per load list: G + 1 <= 17
constexpr unsigned kSmemMax = 232448;                // 227 KB per CTA (B200)
constexpr unsigned kSmemSM = 233472;                 // 228 KB per SM, 1 KB reserved per resident CTA

// shared-memory map (bytes)
constexpr unsigned kTfOff = 0;                       // float2 rg[257] at + 0, float2 ba[257] at + kTfBA (entry i = T[i])
constexpr unsigned kTfBA = 2064;
constexpr unsigned kTfBytes = 2 * kTfBA;
constexpr unsigned kCtlOff = kTfOff + kTfBytes;      // int ctl[8]
constexpr unsigned kLineOff = kCtlOff + 32;          // BeamLine line[4]
constexpr unsigned kStepOff = kLineOff + 64;         // StepRec step[3]
constexpr unsigned kTabOff = kStepOff + 3 * 32;      // unsigned tab[128]: entry (q & 63) and its mirror at + 64
constexpr unsigned kLoadOff = kTabOff + 128 * 4;     // LoadRec load[3][20]
constexpr unsigned kBufOff = (kLoadOff + 3 * 20 * 32 + 127) & ~127u;

struct StepRec {               // one step: march base planes [wlo, wlo + wn) after load[.][0 .. nload) have landed
    int wlo, wn, nload, wmax, hmax, pad0, pad1, pad2;
};
struct LoadRec {               // one plane to stage
    int q, u0, v0, w, h;       // plane index along a; rectangle origin and size (u, v)
    unsigned int sdst;         // shared-memory byte address of voxel (u0, v0) of the plane
    const float *g0;           // global address of voxel (u0, v0) of the plane
};

static_assert(sizeof(LoadRec) == 32 && sizeof(StepRec) == 32, "plan records are addressed with fixed byte offsets");
enum { kCtlMin = 0, kCtlMax = 1, kCtlDirect = 2 };

struct ShearPlanK {
    int tiles_x, tiles_y;
    int G[3];                  // planes per step per principal-axis class
    int NS[3];                 // ring slots per class (>= 2 G + 1)
    int PU[3], PV[3], PP[3];   // row pitch, rows, plane pitch (words) per class
    int sparse[3];             // 1: beams of this class sample so sparsely that staging whole planes costs more than
                               //    it saves; they march through global memory (host plan, see launch_shear)
    unsigned int *overflow;    // mapped host words: [0] set to 1 if a plane ever exceeded its slot (never expected),
                               // [1] counts the beams marched from global memory
};

// Best plane-pitch residue (mod 32) for each row-pitch residue, per class, and the row-pitch residues
// to avoid: minimum mean conflict degree of one corner LDS over 2280 warp patterns of 76 views
// (random eyes, the six axis views, the cfg2 orbit), bank model of DESIGN.md §7.  All "good" pairs
// give 2.3-2.6 wavefronts per LDS (measured 2.34, profiles/r1b_shear_ncu.md); 16-byte-granular
// layouts give 3.7-8 (measured 7.2).
constexpr unsigned char kBestPP[3][32] = {
    { 22, 18, 27, 2, 9, 4, 25, 26, 9, 6, 9, 6, 9, 14, 5, 14, 9, 20, 5, 12, 23, 14, 23, 26, 25, 6, 25, 9, 9, 27, 27, 14 },
    { 17, 13, 19, 21, 25, 28, 27, 19, 25, 28, 13, 13, 19, 27, 19, 9, 25, 26, 13, 14, 25, 19, 9, 20, 25, 10, 25, 6, 19, 11, 19, 13 },
    { 15, 14, 3, 4, 27, 4, 7, 28, 7, 20, 23, 12, 25, 20, 19, 21, 15, 19, 19, 21, 25, 20, 25, 19, 7, 20, 7, 4, 19, 20, 21, 20 } };
constexpr unsigned int kBadPU[3] = {
    (1u << 0) | (1u << 1) | (1u << 2) | (1u << 11) | (1u << 15) | (1u << 16) | (1u << 17) | (1u << 21) | (1u << 22) | (1u << 30) | (1u << 31),
    (1u << 0) | (1u << 1) | (1u << 2) | (1u << 16) | (1u << 17) | (1u << 30) | (1u << 31),
    (1u << 0) | (1u << 1) | (1u << 2) | (1u << 3) | (1u << 15) | (1u << 16) | (1u << 29) | (1u << 30) | (1u << 31) };

// ------------------------------------------------------------------ PTX helpers (explicit shared-space addressing)
__device__ __forceinline__ unsigned int smem_u32(const void *p) { return (unsigned int)__cvta_generic_to_shared(p); }

template <int OFF>
__device__ __forceinline__ float lds_f32(unsigned int a)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1+%2];" : "=f"(v) : "r"(a), "n"(OFF));
    return v;
}
template <int OFF>
__device__ __forceinline__ unsigned int lds_u32(unsigned int a)
{
    unsigned int v;
    asm volatile("ld.shared.u32 %0, [%1+%2];" : "=r"(v) : "r"(a), "n"(OFF));
    return v;
}
template <int OFF>
__device__ __forceinline__ unsigned long long lds_u64(unsigned int a)
{
    unsigned long long v;
    asm volatile("ld.shared.u64 %0, [%1+%2];" : "=l"(v) : "r"(a), "n"(OFF));
    return v;
}
template <int OFF>
__device__ __forceinline__ float2 lds_f32x2(unsigned int a)
{
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2+%3];" : "=f"(v.x), "=f"(v.y) : "r"(a), "n"(OFF));
    return v;
}
template <int OFF>
__device__ __forceinline__ void cp_async4(unsigned int dst_smem, const float *src_global)
{
    asm volatile("cp.async.ca.shared.global [%0+%2], [%1+%2], 4;" ::"r"(dst_smem), "l"(src_global), "n"(OFF) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

struct Acc { float cr, cg, cb, T, m; };

// C.3 straight from global memory: the per-beam fallback when a beam is too wide for its plane slots
__device__ __forceinline__ float sample_global(const VolK &V, const Ray &r, float t)
{
    int ix, iy, iz;
    float fx, fy, fz;
    axis_cell(t, r.d[0], r.oc[0], V.nx, ix, fx);
    axis_cell(t, r.d[1], r.oc[1], V.ny, iy, fy);
    axis_cell(t, r.d[2], r.oc[2], V.nz, iz, fz);
    const float *p = V.base + ((long long)iz * V.sz + (long long)iy * V.sy + ix);
    const float *pz = p + V.sz;
    return trilerp(__ldg(p), __ldg(p + 1), __ldg(p + V.sy), __ldg(p + V.sy + 1), __ldg(pz), __ldg(pz + 1),
                   __ldg(pz + V.sy), __ldg(pz + V.sy + 1), fx, fy, fz);
}

// C.4 from the two half tables at shared address tfa ((r,g) of entry i at tfa + 8 i, (b,a) at + kTfBA); same
// arithmetic as classify() of vr_math.cuh with the four channel lerps paired
__device__ __forceinline__ float4 classify_pairs(unsigned int tfa, float scale, float bias, float s)
{
    const float u = __saturatef(__fmaf_rn(s, scale, bias));
    const float x = __fmul_rn(u, 255.0f);
    const int i = min(__float2int_rz(x), 254);
    const float f = __fsub_rn(x, (float)i);
    const unsigned int e = tfa + 8u * (unsigned int)i;
    const float2 rg = lerp_ee2(lds_f32x2<0>(e), lds_f32x2<8>(e), f);
    const float2 ba = lerp_ee2(lds_f32x2<kTfBA>(e), lds_f32x2<kTfBA + 8>(e), f);
    return make_float4(rg.x, rg.y, ba.x, ba.y);
}

// C.5 with the r and g accumulations paired
__device__ __forceinline__ void composite_packed(float4 rgba, float &Cr, float &Cg, float &Cb, float &T)
{
    const float w = __fmul_rn(T, rgba.w);
    const float2 c = fma2_rn(make_float2(w, w), make_float2(rgba.x, rgba.y), make_float2(Cr, Cg));
    Cr = c.x; Cg = c.y;
    Cb = __fmaf_rn(w, rgba.z, Cb);
    T = __fsub_rn(T, w);
}

// ------------------------------------------------------------------ per-beam state shared by the helpers
struct BeamCtx {
    // uniform over the CTA
    int sgn, na, nu, nv;
    int G, NS, PU, PV, PP;
    int iw_min, iw_max;
    const float *vbase;        // volume base and the element strides of the plane index, u and v
    long long sq, su, sv;
    unsigned int *overflow;
    // shared memory: generic views (warp 0 writes the plan through these) and shared-space addresses (reads)
    BeamLine *lines;
    StepRec *steps;
    unsigned int *tab;
    LoadRec *loads;
    unsigned int tf_a, step_a, tab_a, load_a, buf_a;
};

// warp 0: the next step in travel order -> step record `rec` (wn = 0 marks the end).  Data planes are
// numbered by their ordinal j along the direction of travel (q = iw_min + j, or iw_max + 1 - j when
// travelling towards smaller indices); base plane ordinal jb needs data ordinals jb and jb + 1.  One lane
// per plane of the load list computes that plane's rectangle from the four corner lines.
__device__ __forceinline__ void plan_step(const BeamCtx &B, int rec, bool first, int &next_ord, int &wstart)
{
    const int lane = threadIdx.x & 31;
    const int ord0 = next_ord;
    const StepPlan S = plan_window(first, B.G, B.sgn, B.iw_min, B.iw_max, next_ord, wstart);
    BeamLine L[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) L[k] = B.lines[k];
    int w = 0, h = 0;
    if (lane < S.nload) {
        const int j = ord0 + lane;
        const int q = plane_of_ordinal(B.sgn, B.iw_min, B.iw_max, j);
        int u0, v0;
        plane_rect(L, q, B.na, B.nu, B.nv, false, u0, v0, w, h);
        if (w > B.PU || h > B.PV) {                                   // never expected (fit test over the beam's planes)
            *reinterpret_cast<volatile unsigned int *>(B.overflow) = 1u;
            w = min(w, B.PU); h = min(h, B.PV);
        }
        const unsigned int sdst = B.buf_a + 4u * (unsigned int)(ring_slot(j, B.NS) * B.PP);
        const unsigned int tv = sdst - 4u * (unsigned int)(u0 + v0 * B.PU);
        B.tab[q & 63] = tv; B.tab[(q & 63) + 64] = tv;
        LoadRec &R = B.loads[rec * 20 + lane];
        R.q = q; R.u0 = u0; R.v0 = v0; R.w = w; R.h = h; R.sdst = sdst;
        R.g0 = B.vbase + ((long long)q * B.sq + (long long)u0 * B.su + (long long)v0 * B.sv);
    }
    const int wmax = __reduce_max_sync(0xffffffffu, w), hmax = __reduce_max_sync(0xffffffffu, h);
    if (lane == 0) {
        StepRec &R = B.steps[rec];
        R.wlo = S.wlo; R.wn = S.wn; R.nload = S.nload; R.wmax = wmax; R.hmax = hmax;
    }
}

// all warps: enqueue the cp.async copies of the load list of step record `rec`.
// A != 0: planes contain x (u = x): a warp copies one row of a plane per instruction, lanes along x.
// A == 0: planes are x = const (u = y, v = z): lanes run along x ACROSS the planes of the list (coalesced
//         global reads of consecutive voxels per cell), 32 / Gp cells per instruction.
template <int A>
__device__ __forceinline__ void load_planes(const BeamCtx &B, const VolK &V, int rec)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned int sa_rec = B.step_a + 32u * (unsigned int)rec;
    const int nload = (int)lds_u32<8>(sa_rec);
    if (nload == 0) return;
    const unsigned int PU4 = 4u * (unsigned int)B.PU;
    if (A != 0) {
        const long long sv = A == 2 ? V.sy : V.sz;
        const long long goff = (long long)warp * sv + lane;                  // this thread's first element of a plane
        const unsigned int soff = PU4 * (unsigned int)warp + 4u * (unsigned int)lane;
        for (int k = 0; k < nload; ++k) {
            const unsigned int la = B.load_a + 32u * (unsigned int)(rec * 20 + k);
            const int w = (int)lds_u32<12>(la), h = (int)lds_u32<16>(la);
            const float *g = reinterpret_cast<const float *>(lds_u64<24>(la)) + goff;
            unsigned int s = lds_u32<20>(la) + soff;
            for (int x0 = 0; x0 < w; x0 += 64) {                       // one pass unless a plane is wider than 64
                const bool p0 = lane + x0 < w, p1 = lane + x0 + 32 < w;
                const float *gr = g + x0;
                unsigned int sr = s + 4u * (unsigned int)x0;
                if (x0 + 32 < w) {
                    for (int r = warp; r < h; r += kWarps) {
                        if (p0) cp_async4<0>(sr, gr);
                        if (p1) cp_async4<128>(sr, gr);
                        gr += kWarps * sv; sr += kWarps * PU4;
                    }
                } else {
                    for (int r = warp; r < h; r += kWarps) {
                        if (p0) cp_async4<0>(sr, gr);
                        gr += kWarps * sv; sr += kWarps * PU4;
                    }
                }
            }
        }
    } else {
        const int sh = nload <= 2 ? 1 : nload <= 4 ? 2 : nload <= 8 ? 3 : nload <= 16 ? 4 : 5;    // lanes per cell = 2^sh
        const int pl = lane & ((1 << sh) - 1), sub = lane >> sh, per = 32 >> sh;
        const bool act = pl < nload;
        const unsigned int la = B.load_a + 32u * (unsigned int)(rec * 20 + (act ? pl : 0));
        const int w = act ? (int)lds_u32<12>(la) : 0, h = act ? (int)lds_u32<16>(la) : 0;
        const int wmax = (int)lds_u32<12>(sa_rec), hmax = (int)lds_u32<16>(sa_rec);
        const float *g = reinterpret_cast<const float *>(lds_u64<24>(la)) + ((long long)warp * V.sz + (long long)sub * V.sy);
        unsigned int s = lds_u32<20>(la) + PU4 * (unsigned int)warp + 4u * (unsigned int)sub;
        const long long gstep = (long long)per * V.sy;
        const unsigned int sstep = 4u * (unsigned int)per;
        for (int r = warp; r < hmax; r += kWarps) {
            const int wr = r < h ? w : 0;
            const float *gr = g;
            unsigned int sr = s;
            for (int uc = sub; uc < wmax; uc += 2 * per) {
                if (uc < wr) cp_async4<0>(sr, gr);
                if (uc + per < wr) cp_async4<0>(sr + sstep, gr + gstep);
                gr += 2 * gstep; sr += 2 * sstep;
            }
            g += kWarps * V.sz; s += kWarps * PU4;
        }
    }
}

// every thread: the samples of its ray owned by base planes [wlo, wlo + wn) (C.7 at plane granularity), in
// k order, corners from the staged planes.
template <int MODE, bool ERT, int A>
__device__ __forceinline__ void march_step(const BeamCtx &B, const VolK &V, const CamK &cam, const Ray &r, float scale,
                                           float bias, int wlo, int wn, float &kf, bool &alive, Acc &acc)
{
    const int PU = B.PU;
    const unsigned int PU4 = 4u * (unsigned int)PU;
    for (;;) {
        const float t = __fmaf_rn(kf, cam.step, r.t_first);
        if (!(t < r.t_exit)) { alive = false; break; }                       // C.2: sample k exists iff t_k < t_exit
        int ix, iy, iz;
        float fx, fy, fz;
        axis_cell(t, r.d[0], r.oc[0], V.nx, ix, fx);
        axis_cell(t, r.d[1], r.oc[1], V.ny, iy, fy);
        axis_cell(t, r.d[2], r.oc[2], V.nz, iz, fz);
        const int ia = A == 0 ? ix : A == 1 ? iy : iz;
        if ((unsigned int)(ia - wlo) >= (unsigned int)wn) break;             // owned by a later step (C.7)
        const int iu = A == 0 ? iy : ix, iv = A == 2 ? iy : iz;
        const unsigned int ta = B.tab_a + 4u * (unsigned int)(ia & 63);
        const unsigned int e4 = 4u * (unsigned int)(iu + iv * PU);
        const unsigned int a0 = lds_u32<0>(ta) + e4, a1 = lds_u32<4>(ta) + e4;   // planes ia and ia + 1
        const unsigned int a0v = a0 + PU4, a1v = a1 + PU4;
        // a: a0 -> a1; u: + 4 bytes; v: + PU4
        const float q00 = lds_f32<0>(a0), q10 = lds_f32<4>(a0), q01 = lds_f32<0>(a0v), q11 = lds_f32<4>(a0v);
        const float p00 = lds_f32<0>(a1), p10 = lds_f32<4>(a1), p01 = lds_f32<0>(a1v), p11 = lds_f32<4>(a1v);
        float sv;
        if (A == 2)      sv = trilerp_packed(q00, q10, q01, q11, p00, p10, p01, p11, fx, fy, fz);   // a = z, u = x, v = y
        else if (A == 1) sv = trilerp_packed(q00, q10, p00, p10, q01, q11, p01, p11, fx, fy, fz);   // a = y, u = x, v = z
        else             sv = trilerp_packed(q00, p00, q10, p10, q01, p01, q11, p11, fx, fy, fz);   // a = x, u = y, v = z
        if (MODE == VR_MIP) acc.m = fmaxf(acc.m, sv);
        else {
            composite_packed(classify_pairs(B.tf_a, scale, bias, sv), acc.cr, acc.cg, acc.cb, acc.T);
            if (ERT && acc.T <= cam.t_min) { alive = false; break; }         // stop AFTER compositing this sample (C.5)
        }
        kf = __fadd_rn(kf, 1.0f);                                            // exact: k < 2^24
    }
}

// the step loop of one beam of principal-axis class A
template <int MODE, bool ERT, int A>
__device__ __forceinline__ void run_beam(const BeamCtx &B, const VolK &V, const CamK &cam, const Ray &r, float scale,
                                         float bias, bool alive, Acc &acc, int next_ord, int wstart)
{
    const int warp = threadIdx.x >> 5;
    float kf = 0.0f;
    load_planes<A>(B, V, 0);
    cp_async_commit();
    for (int it = 0;; ++it) {
        cp_async_wait_all();                                                 // my copies for step `it` have landed
        const int any = __syncthreads_or(alive ? 1 : 0);                     // everyone's have; step it-1 is finished
        const unsigned int sa_rec = B.step_a + 32u * (unsigned int)(it % 3);
        const int wlo = (int)lds_u32<0>(sa_rec), wn = (int)lds_u32<4>(sa_rec);
        if (!any || wn == 0) break;
        load_planes<A>(B, V, (it + 1) % 3);
        cp_async_commit();
        if (warp == 0) plan_step(B, (it + 2) % 3, false, next_ord, wstart);
        if (alive) march_step<MODE, ERT, A>(B, V, cam, r, scale, bias, wlo, wn, kf, alive, acc);
    }
    cp_async_wait_all();
}

// ------------------------------------------------------------------ the kernel
template <int MODE, bool ERT>
__global__ void __launch_bounds__(kThreads, 3)
k_shear(CamK cam, VolK V, TfK tf, ShearPlanK P, float *__restrict__ image, long long pitch_f)
{
    extern __shared__ __align__(128) unsigned char smem[];
    float2 *tfp = reinterpret_cast<float2 *>(smem + kTfOff);
    volatile int *ctl = reinterpret_cast<volatile int *>(smem + kCtlOff);

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    // which beam: strips of kStrip beams, row-major inside a strip (co-resident CTAs form a compact block)
    int tx, ty;
    {
        const int per_strip = kStrip * P.tiles_y;
        const int b = blockIdx.x;
        const int s = b / per_strip, rem = b - s * per_strip;
        const int w = min(kStrip, P.tiles_x - s * kStrip);
        ty = rem / w; tx = s * kStrip + rem - ty * w;
    }
    const int x0 = tx * kBW, y0 = ty * kBH;
    const int i = x0 + (warp & 1) * 8 + (lane & 7), j = y0 + (warp >> 1) * 4 + (lane >> 3);

    if (threadIdx.x == 0) { ctl[kCtlMin] = INT_MAX; ctl[kCtlMax] = INT_MIN; ctl[kCtlDirect] = 0; }
    if (MODE == VR_EA)
        for (int e = threadIdx.x; e < 257; e += kThreads) {                      // entry 256 is the pad copy of 255
            const float4 t = __ldg(tf.table + e);
            tfp[e] = make_float2(t.x, t.y);
            *reinterpret_cast<float2 *>(smem + kTfOff + kTfBA + 8 * e) = make_float2(t.z, t.w);
        }

    // principal axis and direction of travel of this beam (uniform: from the beam centre)
    int a, sgn;
    {
        float oc[3], gc[3];
        cam_ray_at(cam, (float)x0 + 0.5f * kBW, (float)y0 + 0.5f * kBH, oc, gc);
        a = principal_axis(gc);
        sgn = (a == 0 ? gc[0] : a == 1 ? gc[1] : gc[2]) > 0.0f ? 1 : -1;
    }
    int au, av;
    beam_axes(a, au, av);

    BeamCtx B;
    B.sgn = sgn;
    B.na = a == 0 ? V.nx : a == 1 ? V.ny : V.nz;
    B.nu = au == 0 ? V.nx : V.ny;
    B.nv = av == 1 ? V.ny : V.nz;
    B.G = a == 0 ? P.G[0] : a == 1 ? P.G[1] : P.G[2];
    B.NS = a == 0 ? P.NS[0] : a == 1 ? P.NS[1] : P.NS[2];
    B.PU = a == 0 ? P.PU[0] : a == 1 ? P.PU[1] : P.PU[2];
    B.PV = a == 0 ? P.PV[0] : a == 1 ? P.PV[1] : P.PV[2];
    B.PP = a == 0 ? P.PP[0] : a == 1 ? P.PP[1] : P.PP[2];
    B.overflow = P.overflow;
    B.vbase = V.base;
    B.sq = a == 0 ? 1 : a == 1 ? V.sy : V.sz;
    B.su = a == 0 ? V.sy : 1;
    B.sv = a == 2 ? V.sy : V.sz;
    B.lines = reinterpret_cast<BeamLine *>(smem + kLineOff);
    B.steps = reinterpret_cast<StepRec *>(smem + kStepOff);
    B.tab = reinterpret_cast<unsigned int *>(smem + kTabOff);
    B.loads = reinterpret_cast<LoadRec *>(smem + kLoadOff);
    const unsigned int smem_a = smem_u32(smem);
    B.tf_a = smem_a + kTfOff; B.step_a = smem_a + kStepOff; B.tab_a = smem_a + kTabOff;
    B.load_a = smem_a + kLoadOff; B.buf_a = smem_a + kBufOff;

    Ray r;
    Acc acc = { 0.0f, 0.0f, 0.0f, 1.0f, -CUDART_INF_F };
    const bool in_image = i < cam.width && j < cam.height;
    bool alive = in_image && make_ray(cam, V.nx, V.ny, V.nz, i, j, r);
    if (alive && !(r.t_first < r.t_exit)) alive = false;                         // no sample at all (C.2)
    {
        const float da = a == 0 ? r.d[0] : a == 1 ? r.d[1] : r.d[2];
        const float oca = a == 0 ? r.oc[0] : a == 1 ? r.oc[1] : r.oc[2];
        int lo_i = INT_MAX, hi_i = INT_MIN;
        if (alive) {
            int ia, ib; float f;
            axis_cell(r.t_first, da, oca, B.na, ia, f);
            axis_cell(r.t_exit, da, oca, B.na, ib, f);
            lo_i = min(ia, ib); hi_i = max(ia, ib);
        }
        lo_i = __reduce_min_sync(0xffffffffu, lo_i);
        hi_i = __reduce_max_sync(0xffffffffu, hi_i);
        __syncthreads();                                                         // ctl initialised
        if (lane == 0 && lo_i <= hi_i) { atomicMin(const_cast<int *>(&ctl[kCtlMin]), lo_i); atomicMax(const_cast<int *>(&ctl[kCtlMax]), hi_i); }
        __syncthreads();
    }
    float *px_out = image + (long long)j * pitch_f + (MODE == VR_MIP ? i : 4 * i);
    B.iw_min = ctl[kCtlMin]; B.iw_max = ctl[kCtlMax];
    if (B.iw_min > B.iw_max) {                                                   // the whole beam misses
        if (in_image) {
            if (MODE == VR_MIP) *px_out = -CUDART_INF_F;
            else *reinterpret_cast<float4 *>(px_out) = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        }
        return;
    }

    // ---- warp 0: the four corner lines of the beam, the fit test, the plans of the first two steps
    int next_ord = 0, wstart = 0;
    const bool sparse_class = (a == 0 ? P.sparse[0] : a == 1 ? P.sparse[1] : P.sparse[2]) != 0;
    if (warp == 0 && sparse_class) { if (lane == 0) ctl[kCtlDirect] = 1; }
    if (warp == 0 && !sparse_class) {
        BeamLine Lm = { 0.0f, 0.0f, 0.0f, 0.0f };
        const float cx = (float)((lane & 1) ? min(x0 + kBW, cam.width) : x0);
        const float cy = (float)((lane & 2) ? min(y0 + kBH, cam.height) : y0);
        bool ok = beam_line(cam, cx, cy, a, sgn, Lm);
        ok = __all_sync(0xffffffffu, ok);
        if (ok) {
            if (lane < 4) B.lines[lane] = Lm;
            __syncwarp();
            BeamLine L[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) L[k] = B.lines[k];
            // every plane of the beam must fit a slot: beam_rect_bound() is their largest raw size up to one voxel
            int wb, hb;
            beam_rect_bound(L, B.iw_min, B.iw_max + 1, B.na, B.nu, B.nv, wb, hb);
            ok = min(wb + 1, B.nu) <= B.PU && min(hb + 1, B.nv) <= B.PV;
        }
        if (!ok) { if (lane == 0) { ctl[kCtlDirect] = 1; atomicAdd(P.overflow + 1, 1u); } }
        else { plan_step(B, 0, true, next_ord, wstart); plan_step(B, 1, false, next_ord, wstart); }
    }
    __syncthreads();

    if (ctl[kCtlDirect]) {
        // this beam is wider than a plane slot (extreme wide angle / grazing rays): march through global memory
        if (alive) {
            float kf = 0.0f;
            for (;;) {
                const float t = __fmaf_rn(kf, cam.step, r.t_first);
                if (!(t < r.t_exit)) break;
                const float sv = sample_global(V, r, t);
                if (MODE == VR_MIP) acc.m = fmaxf(acc.m, sv);
                else {
                    composite(classify_pairs(B.tf_a, tf.scale, tf.bias, sv), acc.cr, acc.cg, acc.cb, acc.T);
                    if (ERT && acc.T <= cam.t_min) break;
                }
                kf = __fadd_rn(kf, 1.0f);
            }
        }
    } else if (a == 2) run_beam<MODE, ERT, 2>(B, V, cam, r, tf.scale, tf.bias, alive, acc, next_ord, wstart);
    else if (a == 1) run_beam<MODE, ERT, 1>(B, V, cam, r, tf.scale, tf.bias, alive, acc, next_ord, wstart);
    else run_beam<MODE, ERT, 0>(B, V, cam, r, tf.scale, tf.bias, alive, acc, next_ord, wstart);

    if (in_image) {
        if (MODE == VR_MIP) *px_out = acc.m;
        else *reinterpret_cast<float4 *>(px_out) = make_float4(acc.cr, acc.cg, acc.cb, __fsub_rn(1.0f, acc.T));
    }
}

// ------------------------------------------------------------------ host: per-frame plan
// Largest plane rectangle per principal-axis class over the frame's beams (every beam up to 65536 beams — all of
// the five configs —, a regular sub-grid plus the image border beyond).  The raw rectangle size is convex in the plane
// index, so per beam it is evaluated at the two ends of the part of the beam inside the volume.  A sizing
// heuristic, not a guarantee: the kernel marches a beam whose planes do not fit from global memory, so an
// under-estimate costs time, never correctness.  cap[a][0] == 0: no sampled beam of class a.
void plan_caps(const CamK &cam, const int n[3], int tiles_x, int tiles_y, int cap[3][2])
{
    for (int a = 0; a < 3; ++a) cap[a][0] = cap[a][1] = 0;
    const int W = cam.width, H = cam.height;
    const int stride = std::max(1, (int)std::ceil(std::sqrt((double)tiles_x * tiles_y / 65536.0)));
    for (int ty = 0; ty < tiles_y; ++ty)
        for (int tx = 0; tx < tiles_x; ++tx) {
            const bool border = tx == 0 || ty == 0 || tx == tiles_x - 1 || ty == tiles_y - 1;
            if (!border && ((tx % stride) || (ty % stride))) continue;
            const int x0 = tx * kBW, y0 = ty * kBH;
            float oc[3], gc[3];
            cam_ray_at(cam, (float)x0 + 0.5f * kBW, (float)y0 + 0.5f * kBH, oc, gc);
            const int a = principal_axis(gc);
            const int sgn = gc[a] > 0.0f ? 1 : -1;
            int u, v;
            beam_axes(a, u, v);
            BeamLine L[4];
            bool valid = true;
            for (int c = 0; c < 4 && valid; ++c) {
                const float cx = (float)((c & 1) ? std::min(x0 + kBW, W) : x0), cy = (float)((c & 2) ? std::min(y0 + kBH, H) : y0);
                valid = beam_line(cam, cx, cy, a, sgn, L[c]);
            }
            float c_lo, c_hi;
            if (!valid || !beam_c_range(L, n[a], n[u], n[v], c_lo, c_hi)) continue;   // marched from global memory / misses the volume
            const int P0 = std::max(0, (int)std::floor(c_lo) - 1), P1 = std::min(n[a] - 1, (int)std::ceil(c_hi) + 1);
            int wb, hb;
            beam_rect_bound(L, P0, P1, n[a], n[u], n[v], wb, hb);
            // + 2: the kernel tests the planes at the ends of the beam's own sample range (the floors let the
            // size differ by one between neighbouring planes) and asks for one voxel to spare
            cap[a][0] = std::max(cap[a][0], std::min(wb + 2, n[u]));
            cap[a][1] = std::max(cap[a][1], std::min(hb + 2, n[v]));
        }
}

// The per-frame plan of k_shear: slot size per principal-axis class, planes per step, ring slots, shared memory.
// Pure host arithmetic on the camera and the volume dims (tests/shear_plan_check.cu runs it without a GPU).
// false: not even three plane slots fit shared memory.
bool make_shear_plan(bool sparse_direct, const CamK &cam, const int n[3], unsigned int *overflow_dev, ShearPlanK &P,
                     unsigned int &smem_bytes)
{
    const int W = cam.width, H = cam.height;
    const int tiles_x = (W + kBW - 1) / kBW, tiles_y = (H + kBH - 1) / kBH;
    memset(&P, 0, sizeof(P));
    P.tiles_x = tiles_x; P.tiles_y = tiles_y; P.overflow = overflow_dev;
    int cap[3][2];
    plan_caps(cam, n, tiles_x, tiles_y, cap);
    // Per class: the ring of 2 G + 1 plane slots with the largest G that leaves room for three CTAs per SM
    // (if G >= 3), else for two (G >= 2), else for one; else shrink the slots (beams that then do not fit
    // march from global memory).  (Class 0 loads with 2^ceil(log2(planes)) lanes per cell; any G works, G + 1 or G
    // a power of two wastes no lanes.)
    // VR_OPT_SPARSE_DIRECT (experimental, off by default; not yet measured end to end).  Sparse sampling (cfg4:
    // 1.7-3.3 voxels per pixel, step 1): neighbouring rays share no voxel, so staging a whole plane rectangle
    // moves cap_w * cap_h / 256 words per ray and plane for the 8 a ray reads.  Measured on cfg4 with the
    // separate kernels (BENCH_NOTES.md): views whose planes contain x march faster straight through L1 (lanes
    // along x share sectors: 19 ms against 38 ms for a z-class view); x-principal views do not (169 ms against
    // 88 ms: through L1 every lane touches its own line).  With the option set, beams of classes 1 and 2 that
    // would stage more than ~6 words per sample march through global memory.
    for (int a = 1; a < 3 && sparse_direct; ++a) {
        if (cap[a][0] == 0) continue;
        float oc[3], gc[3];
        cam_ray_at(cam, 0.5f * (float)W, 0.5f * (float)H, oc, gc);
        const float len = std::sqrt(gc[0] * gc[0] + gc[1] * gc[1] + gc[2] * gc[2]);
        const float per_plane = std::max(1.0f / (cam.step * std::max(std::fabs(gc[a]) / len, 0.3f)), 1.0f);   // samples per plane
        const float words = (float)cap[a][0] * (float)cap[a][1] / (float)(kBW * kBH);
        if (words / per_plane > 6.0f) { P.sparse[a] = 1; cap[a][0] = cap[a][1] = 0; }
    }
    bool fits = false;
    unsigned int ring_words = 0;
    for (int shrink = 0; shrink < 24 && !fits; ++shrink) {
        for (int a = 0; a < 3; ++a) {
            int pu = std::max(cap[a][0], 4), pv = std::max(cap[a][1], 4);
            while (kBadPU[a] >> (pu & 31) & 1u) ++pu;
            int pp = pu * pv;
            while ((pp & 31) != kBestPP[a][pu & 31]) ++pp;
            P.PU[a] = pu; P.PV[a] = pv; P.PP[a] = pp;
        }
        for (int ctas = 3; ctas >= 1 && !fits; --ctas) {
            const unsigned int budget = (kSmemSM / (unsigned int)ctas - 1024u - kBufOff) / 4u;      // ring words
            const int g_min = ctas == 3 ? 3 : ctas == 2 ? 2 : 1;
            fits = true;
            ring_words = 0;
            for (int a = 0; a < 3; ++a) {
                if (cap[a][0] == 0) { P.G[a] = 1; P.NS[a] = 3; continue; }         // class not in this frame
                const int ns = (int)std::min<unsigned int>(budget / (unsigned int)P.PP[a], 2u * (kMaxLoad - 1) + 1u);
                const int g = (ns - 1) / 2;
                if (g < g_min) { fits = false; break; }
                P.G[a] = g; P.NS[a] = 2 * g + 1;
                ring_words = std::max(ring_words, (unsigned int)P.NS[a] * (unsigned int)P.PP[a]);
            }
        }
        if (!fits)
            for (int a = 0; a < 3; ++a)
                for (int e = 0; e < 2; ++e) cap[a][e] = cap[a][e] ? std::max(4, cap[a][e] * 4 / 5) : 0;
    }
#ifdef VR_BEAM_DEBUG
    for (int a = 0; a < 3; ++a)
        fprintf(stderr, "shear: class %d G %d NS %d PU %d PV %d PP %d\n", a, P.G[a], P.NS[a], P.PU[a], P.PV[a], P.PP[a]);
    fprintf(stderr, "fits %d ring_words %u\n", (int)fits, ring_words);
#endif
    if (!fits) return false;
    for (int a = 0; a < 3; ++a)                                                      // unused classes: still addressable
        ring_words = std::max(ring_words, (unsigned int)P.NS[a] * (unsigned int)P.PP[a]);
    smem_bytes = kBufOff + 4u * ring_words;
    return smem_bytes <= kSmemMax;
}

}  // namespace

// The plan depends only on the camera, the volume dims and the option: a handle keeps the last plans, so an orbit
// that is rendered again (or a still camera) pays the host arithmetic (cfg2: ~2 ms, cfg4: ~12 ms) once.
struct ShearPlanCache {
    struct Entry { CamK cam; int n[3]; int sparse; ShearPlanK P; unsigned int smem_bytes; int fits; unsigned long long stamp; };
    std::vector<Entry> e;
    unsigned long long clock = 0;
};
ShearPlanCache *shear_cache_create() { return new (std::nothrow) ShearPlanCache(); }
void shear_cache_destroy(ShearPlanCache *c) { delete c; }

// Enqueues one frame.  *applied = false (and VR_OK) if nothing was enqueued because not even three plane slots
// fit shared memory (the caller then uses another path).
vr_status launch_shear(int mode, bool ert, bool sparse_direct, const CamK &cam, const VolK &V, const TfK &tf,
                       unsigned int *overflow_dev, ShearPlanCache *cache, float *image, long long pitch_f,
                       cudaStream_t st, bool *applied)
{
    *applied = false;
    const int n[3] = { V.nx, V.ny, V.nz };
    const int tiles_x = (cam.width + kBW - 1) / kBW, tiles_y = (cam.height + kBH - 1) / kBH;
    if ((long long)tiles_x * tiles_y > 0x7fffffffll) return VR_OK;
    ShearPlanK P;
    unsigned int smem_bytes = 0;
    bool fits = false, found = false;
    if (cache) {
        for (auto &en : cache->e)
            if (memcmp(&en.cam, &cam, sizeof(CamK)) == 0 && memcmp(en.n, n, sizeof(n)) == 0 && en.sparse == (int)sparse_direct &&
                en.P.overflow == overflow_dev) {
                P = en.P; smem_bytes = en.smem_bytes; fits = en.fits != 0; en.stamp = ++cache->clock; found = true;
                break;
            }
    }
    if (!found) {
        fits = make_shear_plan(sparse_direct, cam, n, overflow_dev, P, smem_bytes);
        if (cache) {
            ShearPlanCache::Entry en;
            memset(&en, 0, sizeof(en));
            en.cam = cam; memcpy(en.n, n, sizeof(n)); en.sparse = (int)sparse_direct; en.P = P; en.smem_bytes = smem_bytes;
            en.fits = fits ? 1 : 0; en.stamp = ++cache->clock;
            if (cache->e.size() < 256) cache->e.push_back(en);
            else *std::min_element(cache->e.begin(), cache->e.end(), [](const ShearPlanCache::Entry &a, const ShearPlanCache::Entry &b) { return a.stamp < b.stamp; }) = en;
        }
    }
    if (!fits) return VR_OK;

    const int grid = tiles_x * tiles_y;
#define VR_SHEAR_LAUNCH(M, E)                                                                                         \
    do {                                                                                                              \
        auto kern = k_shear<M, E>;                                                                                    \
        static bool attr_set = false;                                                                                 \
        if (!attr_set) {                                                                                              \
            VR_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemMax));          \
            attr_set = true;                                                                                          \
        }                                                                                                             \
        kern<<<grid, kThreads, smem_bytes, st>>>(cam, V, tf, P, image, pitch_f);                                      \
    } while (0)
    if (mode == VR_MIP) VR_SHEAR_LAUNCH(VR_MIP, false);
    else if (ert) VR_SHEAR_LAUNCH(VR_EA, true);
    else VR_SHEAR_LAUNCH(VR_EA, false);
#undef VR_SHEAR_LAUNCH
    *applied = true;
    return VR_OK;
}

}  // namespace vr
