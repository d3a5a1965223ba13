// vr_raycast.cu — sm_100a ray-casting kernels: single-march (ray-major), per-brick partial
// images, the sort-last compositor and the brick-by-brick chained march used when streaming.
// SURVEY.md §8(a) rows A6-A10; arithmetic = readings C.1-C.7, all through the
// explicit-rounding device functions of vr_math.cuh.  PAPER.md:L34, L48 (the volume-rendering
// kernel), L32, L50 (gather of partial images).
//
// Thread mapping: one thread per ray; a CTA is a 16x8 pixel tile of four warps, each warp an
// 8x4 pixel patch, so the 32 rays of a warp stay within a few voxels of each other at every
// depth and their 8 corner loads fall into a handful of 128-byte lines (served by L1; L2 holds
// the slab of the volume the active tiles are crossing).  The 256-entry RGBA transfer function
// lives in shared memory (4 KiB + one pad entry).
#include "vr_internal.h"
#include "vr_range.cuh"

namespace vr {

namespace {

constexpr int kTileW = 16, kTileH = 8, kThreads = kTileW * kTileH;

__device__ __forceinline__ void thread_pixel(int tile_x, int tile_y, int &i, int &j)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    i = tile_x * kTileW + (warp & 1) * 8 + (lane & 7);
    j = tile_y * kTileH + (warp >> 1) * 4 + (lane >> 3);
}

__device__ __forceinline__ void stage_tf(float4 *tf_s, const TfK &tf)
{
    for (int e = threadIdx.x; e < 257; e += kThreads) tf_s[e] = __ldg(tf.table + e);
    __syncthreads();
}

// C.3: reconstruct the scalar at parameter t.  WIDE: 64-bit element offsets (volumes > 2^32-1
// voxels); ORG: subtract the index origin of `base` (pool slots / sub-boxes).
template <bool WIDE, bool ORG>
__device__ __forceinline__ float sample_at(const VolK &V, const Ray &r, float t)
{
    int ix, iy, iz;
    float fx, fy, fz;
    axis_cell(t, r.d[0], r.oc[0], V.nx, ix, fx);
    axis_cell(t, r.d[1], r.oc[1], V.ny, iy, fy);
    axis_cell(t, r.d[2], r.oc[2], V.nz, iz, fz);
    if (ORG) { ix -= V.ox; iy -= V.oy; iz -= V.oz; }
    const float *p;
    if (WIDE) p = V.base + ((long long)iz * V.sz + (long long)iy * V.sy + ix);
    else p = V.base + ((unsigned int)iz * (unsigned int)V.sz + (unsigned int)iy * (unsigned int)V.sy + (unsigned int)ix);
    const float *pz = p + V.sz;
    VR_TRACE_CORNER_LOADS(true, true, V.base, p, p + V.sy, pz, pz + V.sy);
    const float v000 = __ldg(p), v100 = __ldg(p + 1);
    const float v010 = __ldg(p + V.sy), v110 = __ldg(p + V.sy + 1);
    const float v001 = __ldg(pz), v101 = __ldg(pz + 1);
    const float v011 = __ldg(pz + V.sy), v111 = __ldg(pz + V.sy + 1);
    return trilerp(v000, v100, v010, v110, v001, v101, v011, v111, fx, fy, fz);
}

struct Accum { float cr, cg, cb, T, m; };

// samples k_lo .. (k_hi inclusive | until t_k >= t_exit when k_hi < 0), in k order (C.5 / C.6)
template <int MODE, bool ERT, bool WIDE, bool ORG>
__device__ __forceinline__ void march(const VolK &V, const Ray &r, const CamK &cam, const float4 *tf_s, float scale,
                                      float bias, int k_lo, int k_hi, Accum &A)
{
    float kf = (float)k_lo;
    const bool bounded = k_hi >= 0;
    int remaining = bounded ? (k_hi - k_lo + 1) : 0x7fffffff;
    for (; remaining > 0; --remaining) {
        const float t = __fmaf_rn(kf, cam.step, r.t_first);
        if (!bounded && !(t < r.t_exit)) break;                 // C.2: sample k exists iff t_k < t_exit
        const float s = sample_at<WIDE, ORG>(V, r, t);
        if (MODE == VR_MIP) A.m = fmaxf(A.m, s);
        else {
            composite(classify(tf_s, scale, bias, s), A.cr, A.cg, A.cb, A.T);
            if (ERT && A.T <= cam.t_min) break;                 // stop AFTER compositing this sample
        }
        kf = __fadd_rn(kf, 1.0f);                               // exact: k < 2^24
    }
}

// ---------------------------------------------------------------- single march, ray-major
template <int MODE, bool ERT, bool WIDE>
__global__ void __launch_bounds__(kThreads)
k_march_full(CamK cam, VolK V, TfK tf, float *__restrict__ image, long long pitch_f)
{
    __shared__ float4 tf_s[257];
    if (MODE == VR_EA) stage_tf(tf_s, tf);
    int i, j;
    thread_pixel(blockIdx.x, blockIdx.y, i, j);
    if (i >= cam.width || j >= cam.height) return;
    i = i * cam.sub + cam.sx; j = j * cam.sub + cam.sy;          // progressive pass: lattice pixel -> image pixel
    Ray r;
    Accum A = { 0.0f, 0.0f, 0.0f, 1.0f, -CUDART_INF_F };
    if (make_ray(cam, V.nx, V.ny, V.nz, i, j, r)) march<MODE, ERT, WIDE, false>(V, r, cam, tf_s, tf.scale, tf.bias, 0, -1, A);
    if (MODE == VR_MIP) image[(long long)j * pitch_f + i] = A.m;
    else
        *reinterpret_cast<float4 *>(image + (long long)j * pitch_f + 4 * i) =
            make_float4(A.cr, A.cg, A.cb, __fsub_rn(1.0f, A.T));
}

// per-(ray, brick) sample range: box_range() of vr_range.cuh
__device__ __forceinline__ bool brick_range(const VolK &V, const Ray &r, float step, const BrickK &b, int &k_lo,
                                            int &k_hi)
{
    return box_range(V.nx, V.ny, V.nz, r, step, b.lo, b.hi, k_lo, k_hi);
}

// ---------------------------------------------------------------- per-brick partial images
// One CTA = one 16x8 pixel tile of one brick's screen rectangle (work table built per frame on
// the host in visibility order).  Writes the fragment (C_b, T_b) / m_b of every pixel of the
// rectangle; pixels whose ray owns no sample in the brick get the identity (0,0,0,1) / -inf.
template <int MODE, bool WIDE>
__global__ void __launch_bounds__(kThreads)
k_march_bricks(CamK cam, VolK Vdims, TfK tf, const BrickK *__restrict__ bricks, const WorkK *__restrict__ work,
               float *__restrict__ arena)
{
    __shared__ float4 tf_s[257];
    __shared__ BrickK bk;
    const WorkK w = work[blockIdx.x];
    if (threadIdx.x == 0) bk = bricks[w.brick];
    if (MODE == VR_EA) stage_tf(tf_s, tf); else __syncthreads();
    int i, j;
    thread_pixel(w.tx, w.ty, i, j);
    i += bk.x0; j += bk.y0;
    if (i >= bk.x1 || j >= bk.y1) return;
    VolK V = Vdims;
    V.base = bk.base; V.sy = bk.sy; V.sz = bk.sz; V.ox = bk.ox; V.oy = bk.oy; V.oz = bk.oz;
    Ray r;
    Accum A = { 0.0f, 0.0f, 0.0f, 1.0f, -CUDART_INF_F };
    int k_lo, k_hi;
    if (make_ray(cam, V.nx, V.ny, V.nz, i, j, r) && brick_range(V, r, cam.step, bk, k_lo, k_hi))
        march<MODE, false, WIDE, true>(V, r, cam, tf_s, tf.scale, tf.bias, k_lo, k_hi, A);
    const unsigned long long f = bk.frag_off + (unsigned long long)(j - bk.y0) * (unsigned)(bk.x1 - bk.x0) + (i - bk.x0);
    if (MODE == VR_MIP) arena[f] = A.m;
    else reinterpret_cast<float4 *>(arena)[f] = make_float4(A.cr, A.cg, A.cb, A.T);
}

// ---------------------------------------------------------------- sort-last compositor (C.7)
// One thread per pixel; a CTA is one 16x16 screen bin whose brick list (visibility order) was
// built on the host.  Fold: C = fma(T, C_b, C); T = T * T_b (EA), m = max(m, m_b) (MIP).
// Folding an identity fragment is exact, so a superset of the contributing bricks is harmless.
template <int MODE>
__global__ void __launch_bounds__(256)
k_composite(int W, int H, const BrickK *__restrict__ bricks, BinsK bins, const float *__restrict__ arena,
            float *__restrict__ image, long long pitch_f)
{
    const int i = blockIdx.x * 16 + (threadIdx.x & 15), j = blockIdx.y * 16 + (threadIdx.x >> 4);
    const unsigned int beg = bins.offs[blockIdx.y * bins.tiles_x + blockIdx.x];
    const unsigned int end = bins.offs[blockIdx.y * bins.tiles_x + blockIdx.x + 1];
    if (i >= W || j >= H) return;
    float cr = 0.0f, cg = 0.0f, cb = 0.0f, T = 1.0f, m = -CUDART_INF_F;
    for (unsigned int e = beg; e < end; ++e) {
        const BrickK *b = bricks + bins.list[e];
        const int x0 = __ldg(&b->x0), y0 = __ldg(&b->y0), x1 = __ldg(&b->x1), y1 = __ldg(&b->y1);
        if (i < x0 || i >= x1 || j < y0 || j >= y1) continue;
        const unsigned long long f = __ldg(&b->frag_off) + (unsigned long long)(j - y0) * (unsigned)(x1 - x0) + (i - x0);
        if (MODE == VR_MIP) m = fmaxf(m, __ldg(arena + f));
        else {
            const float4 p = __ldg(reinterpret_cast<const float4 *>(arena) + f);
            cr = __fmaf_rn(T, p.x, cr); cg = __fmaf_rn(T, p.y, cg); cb = __fmaf_rn(T, p.z, cb);
            T = __fmul_rn(T, p.w);
        }
    }
    if (MODE == VR_MIP) image[(long long)j * pitch_f + i] = m;
    else *reinterpret_cast<float4 *>(image + (long long)j * pitch_f + 4 * i) = make_float4(cr, cg, cb, __fsub_rn(1.0f, T));
}

// ---------------------------------------------------------------- chained march (streaming)
// Bricks arrive front to back; the ray state (C, T) / m lives in the image between bricks, so
// the recurrence of C.5 runs in the same k order as a single march and ERT stays exact.
template <int MODE>
__global__ void k_chain_init(int W, int H, float *__restrict__ image, long long pitch_f)
{
    const int i = blockIdx.x * 32 + (threadIdx.x & 31), j = blockIdx.y * 8 + (threadIdx.x >> 5);
    if (i >= W || j >= H) return;
    if (MODE == VR_MIP) image[(long long)j * pitch_f + i] = -CUDART_INF_F;
    else *reinterpret_cast<float4 *>(image + (long long)j * pitch_f + 4 * i) = make_float4(0.0f, 0.0f, 0.0f, 1.0f);
}

template <int MODE, bool ERT, bool WIDE>
__global__ void __launch_bounds__(kThreads)
k_chain_brick(CamK cam, VolK V, TfK tf, BrickK bk, float *__restrict__ image, long long pitch_f)
{
    __shared__ float4 tf_s[257];
    if (MODE == VR_EA) stage_tf(tf_s, tf);
    int i, j;
    thread_pixel(blockIdx.x, blockIdx.y, i, j);
    i += bk.x0; j += bk.y0;
    if (i >= bk.x1 || j >= bk.y1) return;
    Ray r;
    int k_lo, k_hi;
    if (!make_ray(cam, V.nx, V.ny, V.nz, i, j, r)) return;
    Accum A = { 0.0f, 0.0f, 0.0f, 1.0f, -CUDART_INF_F };
    float *px = image + (long long)j * pitch_f + (MODE == VR_MIP ? i : 4 * i);
    if (MODE == VR_MIP) A.m = *px;
    else {
        const float4 s = *reinterpret_cast<const float4 *>(px);
        A.cr = s.x; A.cg = s.y; A.cb = s.z; A.T = s.w;
        if (ERT && A.T <= cam.t_min) return;                    // this ray already terminated
    }
    if (!brick_range(V, r, cam.step, bk, k_lo, k_hi)) return;
    march<MODE, ERT, WIDE, true>(V, r, cam, tf_s, tf.scale, tf.bias, k_lo, k_hi, A);
    if (MODE == VR_MIP) *px = A.m;
    else *reinterpret_cast<float4 *>(px) = make_float4(A.cr, A.cg, A.cb, A.T);
}

__global__ void k_chain_finish(int W, int H, float *__restrict__ image, long long pitch_f)
{
    const int i = blockIdx.x * 32 + (threadIdx.x & 31), j = blockIdx.y * 8 + (threadIdx.x >> 5);
    if (i >= W || j >= H) return;
    float *a = image + (long long)j * pitch_f + 4 * i + 3;
    *a = __fsub_rn(1.0f, *a);                                   // T -> opacity
}

inline dim3 tiles(int w, int h) { return dim3((w + kTileW - 1) / kTileW, (h + kTileH - 1) / kTileH); }

inline bool needs_wide(const VolK &V)
{
    // largest element offset any corner load can form from base
    const unsigned long long span = (unsigned long long)(V.nz - 1) * (unsigned long long)V.sz +
                                    (unsigned long long)(V.ny - 1) * (unsigned long long)V.sy + V.nx;
    return span > 0xffffffffull || (unsigned long long)V.sz > 0xffffffffull;
}

}  // namespace

void launch_march_full(int mode, bool ert, bool force_wide, const CamK &cam, const VolK &vol, const TfK &tf, float *image,
                       long long pitch_f, cudaStream_t st)
{
    const dim3 g = tiles(cam.width, cam.height);
    const bool wide = force_wide || needs_wide(vol);
#define VR_LAUNCH(M, E, Wd) vr_launch(k_march_full<M, E, Wd>, g, kThreads, 0, st, cam, vol, tf, image, pitch_f)
    if (mode == VR_MIP) { if (wide) VR_LAUNCH(VR_MIP, false, true); else VR_LAUNCH(VR_MIP, false, false); }
    else if (ert) { if (wide) VR_LAUNCH(VR_EA, true, true); else VR_LAUNCH(VR_EA, true, false); }
    else { if (wide) VR_LAUNCH(VR_EA, false, true); else VR_LAUNCH(VR_EA, false, false); }
#undef VR_LAUNCH
}

void launch_march_bricks(int mode, bool wide, const CamK &cam, const VolK &vol, const TfK &tf, const BrickK *bricks,
                         const WorkK *work, int n_work, float *arena, cudaStream_t st)
{
    if (n_work <= 0) return;
#define VR_LAUNCH(M, Wd) vr_launch(k_march_bricks<M, Wd>, n_work, kThreads, 0, st, cam, vol, tf, bricks, work, arena)
    if (mode == VR_MIP) { if (wide) VR_LAUNCH(VR_MIP, true); else VR_LAUNCH(VR_MIP, false); }
    else { if (wide) VR_LAUNCH(VR_EA, true); else VR_LAUNCH(VR_EA, false); }
#undef VR_LAUNCH
}

void launch_composite(int mode, const CamK &cam, const BrickK *bricks, BinsK bins, const float *arena, float *image,
                      long long pitch_f, cudaStream_t st)
{
    const dim3 g((cam.width + 15) / 16, (cam.height + 15) / 16);
    if (mode == VR_MIP) vr_launch(k_composite<VR_MIP>, g, 256, 0, st, cam.width, cam.height, bricks, bins, arena, image, pitch_f);
    else vr_launch(k_composite<VR_EA>, g, 256, 0, st, cam.width, cam.height, bricks, bins, arena, image, pitch_f);
}

void launch_chain_init(int mode, int W, int H, float *image, long long pitch_f, cudaStream_t st)
{
    const dim3 g((W + 31) / 32, (H + 7) / 8);
    if (mode == VR_MIP) vr_launch(k_chain_init<VR_MIP>, g, 256, 0, st, W, H, image, pitch_f);
    else vr_launch(k_chain_init<VR_EA>, g, 256, 0, st, W, H, image, pitch_f);
}

void launch_chain_brick(int mode, bool ert, bool force_wide, const CamK &cam, const VolK &vol, const TfK &tf,
                        const BrickK &brick, float *image, long long pitch_f, cudaStream_t st)
{
    const dim3 g = tiles(brick.x1 - brick.x0, brick.y1 - brick.y0);
    if (g.x == 0 || g.y == 0) return;
    VolK V = vol;
    V.base = brick.base; V.sy = brick.sy; V.sz = brick.sz; V.ox = brick.ox; V.oy = brick.oy; V.oz = brick.oz;
    const bool wide = force_wide || (unsigned long long)V.sz * (unsigned long long)(V.sz / (V.sy ? V.sy : 1) + 2) > 0xffffffffull;   // slot of E^3 elements
#define VR_LAUNCH(M, E, Wd) vr_launch(k_chain_brick<M, E, Wd>, g, kThreads, 0, st, cam, V, tf, brick, image, pitch_f)
    if (mode == VR_MIP) { if (wide) VR_LAUNCH(VR_MIP, false, true); else VR_LAUNCH(VR_MIP, false, false); }
    else if (ert) { if (wide) VR_LAUNCH(VR_EA, true, true); else VR_LAUNCH(VR_EA, true, false); }
    else { if (wide) VR_LAUNCH(VR_EA, false, true); else VR_LAUNCH(VR_EA, false, false); }
#undef VR_LAUNCH
}

void launch_chain_finish(int W, int H, float *image, long long pitch_f, cudaStream_t st)
{
    const dim3 g((W + 31) / 32, (H + 7) / 8);
    vr_launch(k_chain_finish, g, 256, 0, st, W, H, image, pitch_f);
}

}  // namespace vr
