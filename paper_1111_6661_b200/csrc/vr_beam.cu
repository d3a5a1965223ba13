// vr_beam.cu — beam-slab ray casting: the in-HBM fast path of vr_render for VR_LINEAR volumes
// ("the GPU part" of the case study; PAPER.md:L66
// sub-cube partitioning, here applied per beam and per frame instead of per GPU).
//
// Design (kept as the ablation path 3, superseded by vr_shear.cu).  A CTA owns a BEAM: the rays of one 16x16 pixel tile, one thread per ray,
// ray state (C, T) / m in registers from the first sample to the last — so the recurrence of C.5
// runs in k order, early termination is exact, and nothing is exchanged between CTAs.  The beam
// is cut along its PRINCIPAL axis a (largest |d_a| of the centre ray) into slabs of D base-index
// planes.  For every slab the voxel box that the beam can touch (the bounding box of the four
// corner rays of the beam between the two slab planes, + the one-voxel trilinear halo) is copied
// into shared memory by ONE TMA instruction (cp.async.bulk.tensor.3d, SASS UTMALDG) issued by an
// elected thread, double buffered on two mbarriers, and every thread marches the samples of its
// ray that the slab OWNS (C.7 at slab granularity: sample k belongs to the slab iff its clamped
// base index i0_a lies in [lo, hi]; i0_a is monotone in k, so ownership is one compare per
// sample) out of shared memory: 8 LDS per sample instead of 8 global loads that each touch
// ~10-25 L1 sectors (ray-major path: 7.08 ms per cfg2 frame, BENCH_NOTES.md).  All 32 lanes of a warp work on every slab
// (every ray of a beam crosses every slab of the beam), which is what the tile-wave path
// (vr_tiles.cu) lacked: there ~60 % of the issue slots went to rays that missed the tile and to
// per-segment set-up (an ncu capture of an earlier session, not kept).
//
// Arithmetic.  Identical to k_march_full: positions, indices and fractions come from the
// canonical GLOBAL position (vr_math.cuh); the shared-memory address is formed by integer
// subtraction of the box origin.  Results are bit-identical to the ray-major kernel.
//
// HBM traffic.  Beams are scheduled in 16-beam-wide strips so that co-resident CTAs form a
// compact block of the image; neighbouring beams overlap only in the halo and in the slack of
// the bounding box, which L2 (126 MB) serves.  Every voxel inside the view is read from HBM about
// once per frame; the box slack is re-read from L2 (profiles/r1a_beam_tma_ncu.md: 1.2-1.4 GB of DRAM reads per 1.07 GB frame, 7 GB staged).
#include <cuda.h>

#include <algorithm>
#include <climits>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <vector>

#include "vr_beamgeom.cuh"
#include "vr_internal.h"

namespace vr {

namespace {

constexpr int kThreads = 256;
constexpr unsigned kTfBytes = 257 * 16;              // transfer function
constexpr unsigned kCtlOff = kTfBytes;               // 2 mbarriers (16 B) + control words
constexpr unsigned kBufOff = 4352;                   // first stage buffer (multiple of 128)
constexpr unsigned kSmemMax = 232448;                // 227 KB per CTA (B200)

// beam geometry (BeamLine, beam_line, slab_planes, ...): vr_beamgeom.cuh

struct BeamPlanK {
    int tiles_x, tiles_y;
    int D[3];                  // slab depth (base-index planes) per principal-axis class
    int box[3][3];             // TMA box extent per class, [class][x,y,z] voxels
    unsigned int box_bytes[3];
    unsigned int stage_bytes;  // distance between the two stage buffers (multiple of 128)
    unsigned int *overflow;    // mapped host word, set to 1 if a slab box ever exceeded its capacity
};

// ------------------------------------------------------------------ PTX helpers
__device__ __forceinline__ unsigned int smem_u32(const void *p) { return (unsigned int)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned int bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned int parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *tm, int x, int y, int z, unsigned long long *bar)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
        ::"r"(smem_u32(dst)), "l"(reinterpret_cast<unsigned long long>(tm)), "r"(x), "r"(y), "r"(z), "r"(smem_u32(bar))
        : "memory");
}

struct Acc { float cr, cg, cb, T, m; };

// control words in shared memory (ints after the two mbarriers)
enum { kCtlMin = 0, kCtlMax = 1, kCtlDirect = 2, kCtlStage = 4 /* + 4*stage: org, lo, d, - */, kCtlBox = 12 /* ox, oy, oz */ };

// C.3 straight from global memory: the per-beam fallback when a beam is too wide for its slab box
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

// ------------------------------------------------------------------ the kernel
template <int MODE, bool ERT, bool TMA>
__global__ void __launch_bounds__(kThreads, 2)
k_beam(const __grid_constant__ CUtensorMap tm_x, const __grid_constant__ CUtensorMap tm_y,
       const __grid_constant__ CUtensorMap tm_z, CamK cam, VolK V, TfK tf, BeamPlanK P, float *__restrict__ image,
       long long pitch_f)
{
    extern __shared__ __align__(128) unsigned char smem[];
    float4 *tf_s = reinterpret_cast<float4 *>(smem);
    unsigned long long *bar = reinterpret_cast<unsigned long long *>(smem + kCtlOff);
    volatile int *ctl = reinterpret_cast<volatile int *>(smem + kCtlOff + 16);
    unsigned char *buf0 = smem + kBufOff;

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

    if (threadIdx.x == 0) {
        mbar_init(&bar[0], 1); mbar_init(&bar[1], 1);
        ctl[kCtlMin] = INT_MAX; ctl[kCtlMax] = INT_MIN; ctl[kCtlDirect] = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (MODE == VR_EA) for (int e = threadIdx.x; e < 257; e += kThreads) tf_s[e] = __ldg(tf.table + e);

    // principal axis and direction of travel of this beam (uniform: from the beam centre)
    int a, sgn;
    {
        float oc[3], gc[3];
        cam_ray_at(cam, (float)x0 + 0.5f * kBW, (float)y0 + 0.5f * kBH, oc, gc);
        a = principal_axis(gc);
        sgn = (a == 0 ? gc[0] : a == 1 ? gc[1] : gc[2]) > 0.0f ? 1 : -1;
    }
    const int na = a == 0 ? V.nx : a == 1 ? V.ny : V.nz;
    const int D = a == 0 ? P.D[0] : a == 1 ? P.D[1] : P.D[2];
    const int SY = a == 0 ? P.box[0][0] : a == 1 ? P.box[1][0] : P.box[2][0];
    const int BY = a == 0 ? P.box[0][1] : a == 1 ? P.box[1][1] : P.box[2][1];
    const int BZ = a == 0 ? P.box[0][2] : a == 1 ? P.box[1][2] : P.box[2][2];
    const int SZ = SY * BY;

    Ray r;
    Acc A = { 0.0f, 0.0f, 0.0f, 1.0f, -CUDART_INF_F };
    const bool in_image = i < cam.width && j < cam.height;
    bool alive = in_image && make_ray(cam, V.nx, V.ny, V.nz, i, j, r);
    if (alive && !(r.t_first < r.t_exit)) alive = false;                         // no sample at all (C.2)
    {
        const float da = a == 0 ? r.d[0] : a == 1 ? r.d[1] : r.d[2];
        const float oca = a == 0 ? r.oc[0] : a == 1 ? r.oc[1] : r.oc[2];
        int lo_i = INT_MAX, hi_i = INT_MIN;
        if (alive) {
            int ia, ib; float f;
            axis_cell(r.t_first, da, oca, na, ia, f);
            axis_cell(r.t_exit, da, oca, na, ib, f);
            lo_i = min(ia, ib); hi_i = max(ia, ib);
        }
        lo_i = __reduce_min_sync(0xffffffffu, lo_i);
        hi_i = __reduce_max_sync(0xffffffffu, hi_i);
        __syncthreads();                                                         // ctl initialised
        if (lane == 0 && lo_i <= hi_i) { atomicMin(const_cast<int *>(&ctl[kCtlMin]), lo_i); atomicMax(const_cast<int *>(&ctl[kCtlMax]), hi_i); }
        __syncthreads();
    }
    float *px_out = image + (long long)j * pitch_f + (MODE == VR_MIP ? i : 4 * i);
    const int iw_min = ctl[kCtlMin], iw_max = ctl[kCtlMax];
    if (iw_min > iw_max) {                                                       // the whole beam misses
        if (in_image) {
            if (MODE == VR_MIP) *px_out = -CUDART_INF_F;
            else *reinterpret_cast<float4 *>(px_out) = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        }
        return;
    }

    // ---- warp 0: the four corner lines of the beam (lane & 3), slab boxes, loads
    BeamLine L = { 0.0f, 0.0f, 0.0f, 0.0f };
    int au, av;
    beam_axes(a, au, av);
    const int nu = au == 0 ? V.nx : V.ny, nv = av == 1 ? V.ny : V.nz;
    const int cap_u = a == 0 ? BY : SY, cap_v = a == 2 ? BY : BZ;
    const CUtensorMap *tm = a == 0 ? &tm_x : a == 1 ? &tm_y : &tm_z;
    const unsigned int box_bytes = a == 0 ? P.box_bytes[0] : a == 1 ? P.box_bytes[1] : P.box_bytes[2];

    // voxel box of the slab of base indices [lo, hi]: origin, and whether it fits the staged box.  RAW: judge the
    // box before it is clipped to the volume and with the worst row alignment — that need is a convex function of
    // the slab position, so a beam that passes at both of its ends passes everywhere in between.
    auto slab_box = [&](int lo, int hi, bool raw, int &ox, int &oy, int &oz) -> bool {
        float cA, cB;
        slab_planes(lo, hi, na, cA, cB);
        const float c = (lane & 4) ? cB : cA;
        const float qu = fmaf(c, L.Ru, L.Au) - 0.5f, qv = fmaf(c, L.Rv, L.Av) - 0.5f;
        const int umin_r = __reduce_min_sync(0xffffffffu, floor_clamped(qu - kMargin));
        const int umax_r = __reduce_max_sync(0xffffffffu, floor_clamped(qu + kMargin));
        const int vmin_r = __reduce_min_sync(0xffffffffu, floor_clamped(qv - kMargin));
        const int vmax_r = __reduce_max_sync(0xffffffffu, floor_clamped(qv + kMargin));
        const int umin = clampi(umin_r, 0, nu - 2), umax = clampi(umax_r, 0, nu - 2);
        const int vmin = clampi(vmin_r, 0, nv - 2), vmax = clampi(vmax_r, 0, nv - 2);
        ox = (a == 0 ? lo : umin) & ~3;                      // TMA: the box rows start on a 16-byte boundary
        oy = a == 0 ? umin : (a == 1 ? lo : vmin);
        oz = a == 2 ? lo : vmin;
        int need_u, need_v;
        if (raw) { need_u = umax_r - umin_r + 3 + (a == 0 ? 0 : 3); need_v = vmax_r - vmin_r + 3; }   // one voxel to spare
        else { need_u = umax - (a == 0 ? umin : ox) + 2; need_v = vmax - vmin + 2; }
        const int need_a = hi - (a == 0 ? ox : lo) + 2;
        const int cap_a = a == 0 ? SY : a == 1 ? BY : BZ;
        return need_u <= cap_u && need_v <= cap_v && need_a <= cap_a;
    };

    int cursor = sgn > 0 ? iw_min : iw_max;          // warp 0: next unprocessed base-index plane in travel order
    // next slab in travel order -> control words of stage `st` (+ the TMA load).  d = 0 marks the end.
    auto produce = [&](int st) {
        const int remaining = sgn > 0 ? iw_max - cursor + 1 : cursor - iw_min + 1;
        int d = min(D, remaining), lo = 0, ox = 0, oy = 0, oz = 0;
        if (d > 0) {
            for (;;) {
                lo = sgn > 0 ? cursor : cursor - d + 1;
                if (slab_box(lo, lo + d - 1, false, ox, oy, oz)) break;
                if (d == 1) { if (lane == 0) *reinterpret_cast<volatile unsigned int *>(P.overflow) = 1u; break; }
                d >>= 1;
            }
            cursor += sgn > 0 ? d : -d;
        } else d = 0;
        if (lane == 0) {
            ctl[kCtlStage + 4 * st + 0] = ox + oy * SY + oz * SZ;
            ctl[kCtlStage + 4 * st + 1] = lo;
            ctl[kCtlStage + 4 * st + 2] = d;
            if (!TMA) { ctl[kCtlBox + 0] = ox; ctl[kCtlBox + 1] = oy; ctl[kCtlBox + 2] = oz; }
            if (TMA && d > 0) {
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                mbar_expect_tx(&bar[st], box_bytes);
                tma_load_3d(buf0 + (size_t)st * P.stage_bytes, tm, ox, oy, oz, &bar[st]);
            }
        }
    };

    if (warp == 0) {
        const float cx = (float)((lane & 1) ? min(x0 + kBW, cam.width) : x0);
        const float cy = (float)((lane & 2) ? min(y0 + kBH, cam.height) : y0);
        bool ok = beam_line(cam, cx, cy, a, sgn, L);
        ok = __all_sync(0xffffffffu, ok);
        // a one-plane slab must fit at both ends of the beam (then it fits everywhere in between)
        int ox, oy, oz;
        if (ok) ok = slab_box(iw_min, iw_min, true, ox, oy, oz);
        if (ok) ok = slab_box(iw_max, iw_max, true, ox, oy, oz);
        if (!ok) { if (lane == 0) ctl[kCtlDirect] = 1; }
        else { produce(0); if (TMA) produce(1); }
    }
    __syncthreads();

    float kf = 0.0f;
    if (ctl[kCtlDirect]) {
        // this beam is wider than the staged box (extreme wide angle / grazing rays): march through global memory
        if (alive) {
            for (;;) {
                const float t = __fmaf_rn(kf, cam.step, r.t_first);
                if (!(t < r.t_exit)) break;
                const float sv = sample_global(V, r, t);
                if (MODE == VR_MIP) A.m = fmaxf(A.m, sv);
                else {
                    composite(classify(tf_s, tf.scale, tf.bias, sv), A.cr, A.cg, A.cb, A.T);
                    if (ERT && A.T <= cam.t_min) break;
                }
                kf = __fadd_rn(kf, 1.0f);
            }
        }
    } else {
        for (int it = 0;; ++it) {
            const int st = TMA ? (it & 1) : 0;
            const int d = ctl[kCtlStage + 4 * st + 2];
            if (d == 0) break;
            const int org = ctl[kCtlStage + 4 * st + 0], lo = ctl[kCtlStage + 4 * st + 1];
            float *tb = reinterpret_cast<float *>(buf0 + (size_t)st * P.stage_bytes);
            if (TMA) mbar_wait(&bar[st], (unsigned)(it >> 1) & 1u);
            else {
                // fallback loader (row pitch not a multiple of 16 bytes, or unaligned base): plain loads
                const int ox = ctl[kCtlBox + 0], oy = ctl[kCtlBox + 1], oz = ctl[kCtlBox + 2];
                const int ex = min(SY, V.nx - ox), ey = min(BY, V.ny - oy), ez = min(BZ, V.nz - oz);
                const float *g0 = V.base + ((long long)oz * V.sz + (long long)oy * V.sy + ox);
                for (int row = warp; row < ey * ez; row += kThreads / 32) {
                    const int y = row % ey, z = row / ey;
                    const float *g = g0 + ((long long)z * V.sz + (long long)y * V.sy);
                    float *s = tb + (y * SY + z * SZ);
                    for (int x = lane; x < ex; x += 32) s[x] = __ldg(g + x);
                }
                __syncthreads();
            }
            if (alive) {
                for (;;) {
                    const float t = __fmaf_rn(kf, cam.step, r.t_first);
                    if (!(t < r.t_exit)) { alive = false; break; }               // C.2: sample k exists iff t_k < t_exit
                    int ix, iy, iz;
                    float fx, fy, fz;
                    axis_cell(t, r.d[0], r.oc[0], V.nx, ix, fx);
                    axis_cell(t, r.d[1], r.oc[1], V.ny, iy, fy);
                    axis_cell(t, r.d[2], r.oc[2], V.nz, iz, fz);
                    const int iw = a == 0 ? ix : a == 1 ? iy : iz;
                    if ((unsigned int)(iw - lo) >= (unsigned int)d) break;       // owned by a later slab (C.7)
                    const float *p = tb + (ix + iy * SY + iz * SZ - org);
                    const float v000 = p[0], v100 = p[1], v010 = p[SY], v110 = p[SY + 1];
                    const float v001 = p[SZ], v101 = p[SZ + 1], v011 = p[SZ + SY], v111 = p[SZ + SY + 1];
                    const float sv = trilerp(v000, v100, v010, v110, v001, v101, v011, v111, fx, fy, fz);
                    if (MODE == VR_MIP) A.m = fmaxf(A.m, sv);
                    else {
                        composite(classify(tf_s, tf.scale, tf.bias, sv), A.cr, A.cg, A.cb, A.T);
                        if (ERT && A.T <= cam.t_min) { alive = false; break; }   // stop AFTER compositing this sample (C.5)
                    }
                    kf = __fadd_rn(kf, 1.0f);                                    // exact: k < 2^24
                }
            }
            const int any = __syncthreads_or(alive ? 1 : 0);                     // also: everyone is done with buffer st
            if (!any) {                                                          // every ray finished: drain the prefetch
                if (TMA && ctl[kCtlStage + 4 * (st ^ 1) + 2] != 0) mbar_wait(&bar[st ^ 1], (unsigned)((it + 1) >> 1) & 1u);
                break;
            }
            if (warp == 0) produce(st);
            if (!TMA) __syncthreads();
        }
    }
    if (in_image) {
        if (MODE == VR_MIP) *px_out = A.m;
        else *reinterpret_cast<float4 *>(px_out) = make_float4(A.cr, A.cg, A.cb, __fsub_rn(1.0f, A.T));
    }
}

// ------------------------------------------------------------------ host: per-frame plan
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled_fn()
{
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
        cudaGetLastError();
    }
    return fn;
}

constexpr int kNumDepth = 6;
constexpr int kDepth[kNumDepth] = { 16, 12, 8, 4, 2, 1 };       // slab depth candidates (base-index planes)

// What the transverse axes of a slab box should hold, per principal-axis class and slab-depth candidate: the
// largest need over a sample of the frame's beams (every beam when there are few, a regular sub-grid plus the
// image border otherwise).  For one beam the bounding box of its four corner rays between the planes c and
// c + D' is at most  spread(c) + D' * (max(0, Rmax) - min(0, Rmin))  wide, and spread(c) is convex in c, so over
// the part of the beam inside the volume it is largest at one of the two ends.  This is a sizing heuristic, not
// a guarantee: the kernel shortens a slab whose box would not fit and marches a beam that never fits from
// global memory, so an under-estimate costs time, never correctness.
void plan_capacity(const CamK &cam, const int n[3], int tiles_x, int tiles_y, const std::vector<float> &grid_o,
                   const std::vector<float> &grid_g, int cap[3][kNumDepth][2])
{
    float need[3][kNumDepth][2];
    for (int a = 0; a < 3; ++a)
        for (int k = 0; k < kNumDepth; ++k) need[a][k][0] = need[a][k][1] = 0.0f;
    const int gx = tiles_x + 1;
    const int stride = std::max(1, (int)std::ceil(std::sqrt((double)tiles_x * tiles_y / 4096.0)));
    for (int ty = 0; ty < tiles_y; ++ty)
        for (int tx = 0; tx < tiles_x; ++tx) {
            const bool border = tx == 0 || ty == 0 || tx == tiles_x - 1 || ty == tiles_y - 1;
            if (!border && ((tx % stride) || (ty % stride))) continue;
            float oc[3], gc[3];
            cam_ray_at(cam, (float)(tx * kBW) + 0.5f * kBW, (float)(ty * kBH) + 0.5f * kBH, oc, gc);
            const int a = principal_axis(gc);
            const int sgn = gc[a] > 0.0f ? 1 : -1;
            int u, v;
            beam_axes(a, u, v);
            const int ax[2] = { u, v };
            float R[4][2], Aq[4][2];
            float c_lo = 1e30f, c_hi = -1e30f;
            bool valid = true;
            for (int c = 0; c < 4 && valid; ++c) {
                const size_t gi = (size_t)(ty + (c >> 1)) * gx + (tx + (c & 1));
                const float *o = &grid_o[3 * gi], *g = &grid_g[3 * gi];
                const float ga = g[a], len2 = g[0] * g[0] + g[1] * g[1] + g[2] * g[2];
                if (!(ga * (float)sgn > 0.0f) || !(ga * ga >= 0.09f * len2)) { valid = false; break; }
                // the part of this corner line inside the volume, as an interval of the principal coordinate
                float lo = 0.0f, hi = (float)n[a];
                for (int e = 0; e < 2; ++e) {
                    R[c][e] = g[ax[e]] / ga;
                    Aq[c][e] = o[ax[e]] - o[a] * R[c][e];
                    if (R[c][e] != 0.0f) {
                        const float c0 = (0.0f - Aq[c][e]) / R[c][e], c1 = ((float)n[ax[e]] - Aq[c][e]) / R[c][e];
                        lo = std::max(lo, std::min(c0, c1)); hi = std::min(hi, std::max(c0, c1));
                    } else if (Aq[c][e] < 0.0f || Aq[c][e] > (float)n[ax[e]]) hi = -1e30f;
                }
                if (hi >= lo) { c_lo = std::min(c_lo, lo); c_hi = std::max(c_hi, hi); }
            }
            if (!valid || c_hi < c_lo) continue;            // marched from global memory / misses the volume
            for (int e = 0; e < 2; ++e) {
                float s0[2] = { 1e30f, -1e30f }, s1[2] = { 1e30f, -1e30f }, rr[2] = { 0.0f, 0.0f };
                for (int c = 0; c < 4; ++c) {
                    const float q0 = fmaf(c_lo, R[c][e], Aq[c][e]), q1 = fmaf(c_hi, R[c][e], Aq[c][e]);
                    s0[0] = std::min(s0[0], q0); s0[1] = std::max(s0[1], q0);
                    s1[0] = std::min(s1[0], q1); s1[1] = std::max(s1[1], q1);
                    rr[0] = std::min(rr[0], R[c][e]); rr[1] = std::max(rr[1], R[c][e]);
                }
                const float S = std::max(s0[1] - s0[0], s1[1] - s1[0]), G = rr[1] - rr[0];
                for (int k = 0; k < kNumDepth; ++k) need[a][k][e] = std::max(need[a][k][e], S + (float)(kDepth[k] + 1) * G);
            }
        }
    for (int a = 0; a < 3; ++a) {
        int u, v;
        beam_axes(a, u, v);
        const int nt[2] = { n[u], n[v] };
        for (int k = 0; k < kNumDepth; ++k)
            for (int e = 0; e < 2; ++e) {
                // floor(b) - floor(a) <= ceil(b - a); + 1 inclusive count, + 1 trilinear halo
                const float w = need[a][k][e] + 2.0f * kMargin;
                cap[a][k][e] = std::max(4, (int)std::min((float)nt[e], std::ceil(std::min(w, 1.0e6f)) + 2.0f));
            }
    }
}

inline int round_up(int v, int m) { return (v + m - 1) / m * m; }

// box extents of class a at depth candidate k
void class_box(int a, int k, const int cap[3][kNumDepth][2], int ext[3])
{
    int u, v;
    beam_axes(a, u, v);
    const int D = kDepth[k];
    ext[a] = D + 1; ext[u] = cap[a][k][0]; ext[v] = cap[a][k][1];
    // TMA: the box must start on a 16-byte boundary of a row (x origin rounded down to a multiple of 4 voxels:
    // up to 3 extra voxels in front) and its rows are multiples of 16 bytes
    ext[0] = round_up(ext[0] + 3, 4);
    if (a != 0) {
        if (ext[0] % 8 == 0) ext[0] += 4;                               // row pitch 4 (mod 8) banks
        if (ext[1] % 2 == 0) ext[1] += 1;                               // plane pitch 4 (mod 8) banks
    }
}

}  // namespace

// Enqueues one frame.  *applied = false (and VR_OK) if nothing was enqueued because even the smallest slab box
// does not fit shared memory (the caller then uses the ray-major kernel).
vr_status launch_beam(int mode, bool ert, const CamK &cam, const VolK &V, const TfK &tf, unsigned int *overflow_dev,
                      float *image, long long pitch_f, cudaStream_t st, bool *applied)
{
    *applied = false;
    const int n[3] = { V.nx, V.ny, V.nz };
    const int W = cam.width, H = cam.height;
    const int tiles_x = (W + kBW - 1) / kBW, tiles_y = (H + kBH - 1) / kBH;
    if ((long long)tiles_x * tiles_y > 0x7fffffffll) return VR_OK;

    // rays through the corners of the beam grid (shared by neighbouring beams)
    const int gx = tiles_x + 1, gy = tiles_y + 1;
    std::vector<float> grid_o((size_t)gx * gy * 3), grid_g((size_t)gx * gy * 3);
    for (int y = 0; y < gy; ++y)
        for (int x = 0; x < gx; ++x) {
            const size_t gi = (size_t)y * gx + x;
            cam_ray_at(cam, (float)std::min(x * kBW, W), (float)std::min(y * kBH, H), &grid_o[3 * gi], &grid_g[3 * gi]);
        }

    const bool tma_ok = encode_tiled_fn() != nullptr && (V.nx % 4) == 0 && ((uintptr_t)V.base & 15u) == 0 &&
                        V.sy == V.nx && V.sz == (long long)V.nx * V.ny;
    BeamPlanK P;
    memset(&P, 0, sizeof(P));
    P.tiles_x = tiles_x; P.tiles_y = tiles_y; P.overflow = overflow_dev;
    int cap[3][kNumDepth][2];
    plan_capacity(cam, n, tiles_x, tiles_y, grid_o, grid_g, cap);
    const int stages = tma_ok ? 2 : 1;
    // per class the deepest slab whose stages leave room for two CTAs per SM; else for one; else shrink the boxes
    // (beams that then do not fit use shorter slabs or march from global memory)
    bool fits = false;
    for (int shrink = 0; shrink < 24 && !fits; ++shrink) {
        for (int pass = 0; pass < 2 && !fits; ++pass) {
            const unsigned int budget = ((pass == 0 ? kSmemMax / 2 - 1024u : kSmemMax) - kBufOff) / (unsigned int)stages;
            fits = true;
            P.stage_bytes = 0;
            for (int a = 0; a < 3; ++a) {
                int pick = -1, ext[3] = { 4, 1, 1 };
                for (int k = 0; k < kNumDepth && pick < 0; ++k) {
                    if (a == 0 && kDepth[k] < 4) break;                 // x class: rows hold >= 8 voxels anyway (alignment)
                    class_box(a, k, cap, ext);
                    const unsigned long long bytes = 4ull * ext[0] * ext[1] * ext[2];
                    if (ext[0] <= 256 && ext[1] <= 256 && ext[2] <= 256 && ((bytes + 127u) & ~127ull) <= budget) pick = k;
                }
                if (pick < 0) { fits = false; break; }
                P.D[a] = kDepth[pick];
                for (int e = 0; e < 3; ++e) P.box[a][e] = ext[e];
                P.box_bytes[a] = 4u * (unsigned int)ext[0] * (unsigned int)ext[1] * (unsigned int)ext[2];
                P.stage_bytes = std::max(P.stage_bytes, (P.box_bytes[a] + 127u) & ~127u);
            }
        }
        if (!fits)
            for (int a = 0; a < 3; ++a)
                for (int k = 0; k < kNumDepth; ++k)
                    for (int e = 0; e < 2; ++e) cap[a][k][e] = std::max(4, cap[a][k][e] * 4 / 5);
    }
#ifdef VR_BEAM_DEBUG
    for (int a = 0; a < 3; ++a)
        fprintf(stderr, "beam: class %d D %d box %d x %d x %d (%u B)\n", a, P.D[a], P.box[a][0], P.box[a][1], P.box[a][2], P.box_bytes[a]);
    fprintf(stderr, "fits %d stage %u tma %d\n", (int)fits, P.stage_bytes, (int)tma_ok);
#endif
    if (!fits) return VR_OK;
    const unsigned int smem_bytes = kBufOff + (unsigned int)stages * P.stage_bytes;

    CUtensorMap tmap[3];
    memset(tmap, 0, sizeof(tmap));
    if (tma_ok) {
        const cuuint64_t gdim[3] = { (cuuint64_t)V.nx, (cuuint64_t)V.ny, (cuuint64_t)V.nz };
        const cuuint64_t gstr[2] = { (cuuint64_t)V.nx * 4u, (cuuint64_t)V.nx * (cuuint64_t)V.ny * 4u };
        const cuuint32_t estr[3] = { 1, 1, 1 };
        for (int a = 0; a < 3; ++a) {
            const cuuint32_t box[3] = { (cuuint32_t)P.box[a][0], (cuuint32_t)P.box[a][1], (cuuint32_t)P.box[a][2] };
            const CUresult rc = encode_tiled_fn()(&tmap[a], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float *>(V.base),
                                                  gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                                  CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                                                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            if (rc != CUDA_SUCCESS) { set_error("cuTensorMapEncodeTiled failed (%d)", (int)rc); return VR_ERR_CUDA; }
        }
    }

    const int grid = tiles_x * tiles_y;
#define VR_BEAM_LAUNCH(M, E, T)                                                                                       \
    do {                                                                                                              \
        auto kern = k_beam<M, E, T>;                                                                                  \
        static bool attr_set = false;                                                                                 \
        if (!attr_set) {                                                                                              \
            VR_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemMax));          \
            attr_set = true;                                                                                          \
        }                                                                                                             \
        kern<<<grid, kThreads, smem_bytes, st>>>(tmap[0], tmap[1], tmap[2], cam, V, tf, P, image, pitch_f);           \
    } while (0)
    if (tma_ok) {
        if (mode == VR_MIP) VR_BEAM_LAUNCH(VR_MIP, false, true);
        else if (ert) VR_BEAM_LAUNCH(VR_EA, true, true);
        else VR_BEAM_LAUNCH(VR_EA, false, true);
    } else {
        if (mode == VR_MIP) VR_BEAM_LAUNCH(VR_MIP, false, false);
        else if (ert) VR_BEAM_LAUNCH(VR_EA, true, false);
        else VR_BEAM_LAUNCH(VR_EA, false, false);
    }
#undef VR_BEAM_LAUNCH
    *applied = true;
    return VR_OK;
}

}  // namespace vr
