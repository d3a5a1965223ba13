// vr_tiles.cu — tile-wave ray casting: the in-HBM fast path of vr_render (SURVEY.md §8(a) rows
// A6-A9; "the GPU part" of the case study, L66 sub-cube partitioning).
//
// Why.  One thread per ray marching through global memory is bound by the L1 tag stage: the 32
// rays of a warp touch ~25 different 32-byte sectors per corner load, eight loads per sample
// (an ncu capture of an earlier session, not kept; BENCH_NOTES.md has the timings).  Shared memory has no sector granularity: 32 lanes reading 32
// different words cost ~2 wavefronts with the padded strides below.  So the volume is cut into
// staging tiles of TX x TY x TZ ownership cells (C.7 applied at tile granularity), a CTA copies
// one tile (+1 high-side halo) into shared memory with cp.async and marches every ray segment
// that crosses it from there.
//
// Order.  Emission-absorption needs a ray's samples in k order (C.5), and early termination needs
// the running transmittance.  The ray state (C, T) / m lives in the output image between tiles.
// Tiles are listed level-major, level = sum over axes of the tile distance from the eye tile
// (perspective) or along sign(d) (orthographic).  Along a ray every per-axis tile index moves
// monotonically away from the eye tile (fmaf is monotone in t and t_k is monotone in k), so a
// ray visits tiles in strictly increasing level and every tile of the dependence cone of tile b
// is reachable through face neighbours "towards the eye".  A persistent grid pops tiles from
// the list; a tile is processed once its <= 3 face predecessors have published completion, and
// EVERY tile (also one without pixels) waits for them before it publishes, so completion is
// transitive over the whole cone.  The pop order is a topological order and a CTA only waits
// for tiles popped earlier (by CTAs that are running), so the scheme cannot deadlock.
//
// Arithmetic.  Identical to the ray-major kernel: positions, indices and fractions come from the
// canonical GLOBAL position (vr_math.cuh); the shared-memory address is formed by integer
// subtraction of the tile origin.  Results are bit-identical to k_march_full.
#include <cuda_pipeline.h>

#include "vr_internal.h"
#include "vr_range.cuh"

namespace vr {

namespace {

constexpr int kThreads = 256;

constexpr int pad_mod32(int v, int r) { return v + ((r - v % 32) + 32) % 32; }

// shared-memory strides: sy = 5 (mod 32), sz = 7 (mod 32) gave the lowest bank-conflict degree
// (2.1 wavefronts per corner load vs 3.8 for dense 33 x 33) over random views (bank model)
template <int TX_, int TY_, int TZ_>
struct TileCfg {
    static constexpr int TX = TX_, TY = TY_, TZ = TZ_;
    static constexpr int EX = TX + 1, EY = TY + 1, EZ = TZ + 1;
    static constexpr int SY = pad_mod32(EX, 5);
    static constexpr int SZ = pad_mod32(SY * EY, 7);
    static constexpr int WORDS = SZ * EZ;
    static constexpr size_t SMEM = (size_t)WORDS * 4 + 257 * 16 + 64;
};

__device__ __forceinline__ unsigned int ld_acquire(const unsigned int *p)
{
    unsigned int v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release(unsigned int *p, unsigned int v)
{
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// conservative screen rectangle of the box [lo, hi] of sample positions (double precision)
__device__ double det3(const double a[3], const double b[3], const double c[3])
{
    return a[0] * (b[1] * c[2] - b[2] * c[1]) - b[0] * (a[1] * c[2] - a[2] * c[1]) + c[0] * (a[1] * b[2] - a[2] * b[1]);
}

__device__ void box_rect_dev(const CamK &c, bool persp, const double lo[3], const double hi[3], int &x0, int &y0,
                             int &x1, int &y1)
{
    const int W = c.width, H = c.height;
    double mnx = 1e300, mny = 1e300, mxx = -1e300, mxy = -1e300;
    bool full = false;
    for (int corner = 0; corner < 8 && !full; ++corner) {
        double P[3], m0[3], m1[3], m2[3], rhs[3];
        for (int a = 0; a < 3; ++a) P[a] = (corner >> a & 1) ? hi[a] : lo[a];
        double x, y;
        if (persp) {                   // d0 + x du + y dv = lambda (P - o0)
            for (int a = 0; a < 3; ++a) { m0[a] = c.du[a]; m1[a] = c.dv[a]; m2[a] = -(P[a] - (double)c.o0[a]); rhs[a] = -(double)c.d0[a]; }
            const double D = det3(m0, m1, m2);
            if (fabs(D) < 1e-300) { full = true; break; }
            x = det3(rhs, m1, m2) / D; y = det3(m0, rhs, m2) / D;
            const double lambda = det3(m0, m1, rhs) / D;
            if (!(lambda > 1e-9)) { full = true; break; }        // corner at or behind the eye
        } else {                       // o0 + x ou + y ov + t d0 = P
            for (int a = 0; a < 3; ++a) { m0[a] = c.ou[a]; m1[a] = c.ov[a]; m2[a] = c.d0[a]; rhs[a] = P[a] - (double)c.o0[a]; }
            const double D = det3(m0, m1, m2);
            if (fabs(D) < 1e-300) { full = true; break; }
            x = det3(rhs, m1, m2) / D; y = det3(m0, rhs, m2) / D;
        }
        if (!isfinite(x) || !isfinite(y)) { full = true; break; }
        mnx = fmin(mnx, x); mxx = fmax(mxx, x); mny = fmin(mny, y); mxy = fmax(mxy, y);
    }
    if (full) { x0 = 0; y0 = 0; x1 = W; y1 = H; return; }
    // pixel i has x = i + 0.5; one extra pixel of slack for the float32 ray arithmetic
    const double fx0 = floor(mnx - 0.5) - 1.0, fy0 = floor(mny - 0.5) - 1.0;
    const double fx1 = ceil(mxx - 0.5) + 2.0, fy1 = ceil(mxy - 0.5) + 2.0;
    x0 = (int)fmin(fmax(fx0, 0.0), (double)W); x1 = (int)fmin(fmax(fx1, 0.0), (double)W);
    y0 = (int)fmin(fmax(fy0, 0.0), (double)H); y1 = (int)fmin(fmax(fy1, 0.0), (double)H);
}

__device__ __forceinline__ void tile_owned(const TilePlanK &P, int a, int b, int n, int &lo, int &hi)
{
    lo = P.T[a] * b;
    hi = min(lo + P.T[a] - 1, n - 2);
}

// ---------------------------------------------------------------- per-frame work list (A4 at tile level)
__global__ void __launch_bounds__(256)
k_tile_plan(CamK cam, TilePlanK P, int nx, int ny, int nz, const unsigned int *__restrict__ lvl_off,
            unsigned int *__restrict__ ctrl, TileWork *__restrict__ work)
{
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= P.n_tiles) return;
    const int n[3] = { nx, ny, nz };
    int b[3] = { id % P.nt[0], (id / P.nt[0]) % P.nt[1], id / (P.nt[0] * P.nt[1]) };
    int level = 0;
    double lo[3], hi[3];
    bool empty = false;
    for (int a = 0; a < 3; ++a) {
        int l, h;
        tile_owned(P, a, b[a], n[a], l, h);
        if (l > h) empty = true;
        lo[a] = (l == 0 ? 0.0 : l + 0.5) - 0.01;                   // ownership cell in position space (C.7),
        hi[a] = (h == n[a] - 2 ? (double)n[a] : h + 1.5) + 0.01;   // outer cells reach the volume faces
        level += tile_axis_level(P, a, b[a]);
    }
    TileWork w;
    w.x0 = w.y0 = w.x1 = w.y1 = 0;
    if (!empty) box_rect_dev(cam, P.persp != 0, lo, hi, w.x0, w.y0, w.x1, w.y1);
    w.b[0] = (unsigned short)b[0]; w.b[1] = (unsigned short)b[1]; w.b[2] = (unsigned short)b[2];
    w.flags = (w.x1 > w.x0 && w.y1 > w.y0) ? 1 : 0;
    const unsigned int slot = lvl_off[level] + atomicAdd(&ctrl[1 + level], 1u);
    work[slot] = w;
}

// ---------------------------------------------------------------- sampling from the staged tile
// C.3 with the tile in shared memory.  `org` = ox + oy*SY + oz*SZ of the tile origin.
// INTERIOR: the tile owns no base index 0 or n-2 on any axis, so for an owned sample the clamps of
// C.3 are no-ops (its clamped q lies in [1, n-2)) and are skipped; the result is bit-identical.
template <class C, bool INTERIOR>
__device__ __forceinline__ float sample_tile(const float *__restrict__ ts, int org, const Ray &r, float t, int nx,
                                             int ny, int nz)
{
    int ix, iy, iz;
    float fx, fy, fz;
    if (INTERIOR) {
        const float qx = __fmaf_rn(t, r.d[0], r.oc[0]), qy = __fmaf_rn(t, r.d[1], r.oc[1]), qz = __fmaf_rn(t, r.d[2], r.oc[2]);
        ix = __float2int_rd(qx); iy = __float2int_rd(qy); iz = __float2int_rd(qz);
        fx = __fsub_rn(qx, (float)ix); fy = __fsub_rn(qy, (float)iy); fz = __fsub_rn(qz, (float)iz);
    } else {
        axis_cell(t, r.d[0], r.oc[0], nx, ix, fx);
        axis_cell(t, r.d[1], r.oc[1], ny, iy, fy);
        axis_cell(t, r.d[2], r.oc[2], nz, iz, fz);
    }
    const float *p = ts + (ix + iy * C::SY + iz * C::SZ - org);
    const float v000 = p[0], v100 = p[1], v010 = p[C::SY], v110 = p[C::SY + 1];
    const float v001 = p[C::SZ], v101 = p[C::SZ + 1], v011 = p[C::SZ + C::SY], v111 = p[C::SZ + C::SY + 1];
    return trilerp(v000, v100, v010, v110, v001, v101, v011, v111, fx, fy, fz);
}

struct State { float cr, cg, cb, T, m; };

// samples k_lo..k_hi of one ray from the staged tile, in k order, U samples in flight
template <class C, int MODE, bool ERT, bool INTERIOR>
__device__ __forceinline__ void march_tile(const float *__restrict__ ts, int org, const Ray &r, const CamK &cam,
                                           int nx, int ny, int nz, const float4 *tf_s, float scale, float bias,
                                           int k_lo, int k_hi, State &A)
{
    constexpr int U = 4;
    for (int k = k_lo; k <= k_hi; k += U) {
        float s[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int kk = min(k + u, k_hi);                       // tail: a repeat of the last sample, not composited
            const float t = __fmaf_rn((float)kk, cam.step, r.t_first);
            s[u] = sample_tile<C, INTERIOR>(ts, org, r, t, nx, ny, nz);
        }
        if (MODE == VR_MIP) {
#pragma unroll
            for (int u = 0; u < U; ++u) A.m = fmaxf(A.m, s[u]);   // max is idempotent: the repeated tail is harmless
        } else {
            bool stop = false;
#pragma unroll
            for (int u = 0; u < U; ++u) {
                if (k + u <= k_hi && !stop) {
                    composite(classify(tf_s, scale, bias, s[u]), A.cr, A.cg, A.cb, A.T);
                    if (ERT && A.T <= cam.t_min) stop = true;     // stop AFTER compositing this sample (C.5)
                }
            }
            if (stop) break;
        }
    }
}

// ---------------------------------------------------------------- the persistent tile-wave kernel
template <class C, int MODE, bool ERT>
__global__ void __launch_bounds__(kThreads)
k_tile_march(CamK cam, TilePlanK P, VolK V, TfK tf, const TileWork *__restrict__ work, unsigned int *ctrl,
             unsigned int *done, unsigned int serial, float *image, long long pitch_f)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4 *tf_s = reinterpret_cast<float4 *>(smem_raw);
    float *ts = reinterpret_cast<float *>(smem_raw + 257 * 16);
    int *s_ctl = reinterpret_cast<int *>(smem_raw + 257 * 16 + (size_t)C::WORDS * 4);   // [0] item, [1] patch counter

    if (MODE == VR_EA) for (int e = threadIdx.x; e < 257; e += kThreads) tf_s[e] = __ldg(tf.table + e);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int n[3] = { V.nx, V.ny, V.nz };
    int finished = -1;                                            // tile id to publish at the top of the loop

    for (;;) {
        __syncthreads();                                          // everyone is done with the previous tile
        if (threadIdx.x == 0) {
            if (finished >= 0) { __threadfence(); st_release(done + finished, serial); }
            s_ctl[0] = (int)atomicAdd(&ctrl[0], 1u);
            s_ctl[1] = 0;
        }
        __syncthreads();
        const int item = s_ctl[0];
        if (item >= P.n_tiles) break;
        const TileWork w = work[item];
        const int b[3] = { w.b[0], w.b[1], w.b[2] };
        const int tile_id = b[0] + P.nt[0] * (b[1] + P.nt[1] * b[2]);
        int lo[3], hi[3];
        bool interior = true;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            tile_owned(P, a, b[a], n[a], lo[a], hi[a]);
            if (lo[a] < 1 || hi[a] > n[a] - 3) interior = false;
        }
        if (w.flags) {
            // stage voxels [lo, min(lo + T, n - 1)] per axis: one warp per x-row, 4-byte cp.async
            const int ex = min(C::EX, V.nx - lo[0]), ey = min(C::EY, V.ny - lo[1]), ez = min(C::EZ, V.nz - lo[2]);
            const float *g0 = V.base + ((long long)lo[2] * V.sz + (long long)lo[1] * V.sy + lo[0]);
            const int rows = ey * ez;
            for (int rrow = warp; rrow < rows; rrow += kThreads / 32) {
                const int y = rrow % ey, z = rrow / ey;
                const float *g = g0 + ((long long)z * V.sz + (long long)y * V.sy);
                float *s = ts + (y * C::SY + z * C::SZ);
                for (int x = lane; x < ex; x += 32) __pipeline_memcpy_async(s + x, g + x, 4);
            }
            __pipeline_commit();
        }
        if (threadIdx.x < 3) {                                    // wait for the face neighbours towards the eye
            const int a = threadIdx.x;
            const int pb = tile_axis_pred(P, a, b[a]);
            if (pb >= 0) {
                int q[3] = { b[0], b[1], b[2] };
                q[a] = pb;
                const unsigned int *flag = done + (q[0] + P.nt[0] * (q[1] + P.nt[1] * q[2]));
                while (ld_acquire(flag) != serial) __nanosleep(100);
                __threadfence();
            }
        }
        finished = tile_id;
        if (!w.flags) continue;
        __pipeline_wait_prior(0);
        __syncthreads();                                          // tile staged, predecessors complete

        const int org = lo[0] + lo[1] * C::SY + lo[2] * C::SZ;
        const int rw = w.x1 - w.x0, rh = w.y1 - w.y0;
        const int npx = (rw + 7) >> 3, npatch = npx * ((rh + 3) >> 2);
        for (;;) {
            int p = 0;
            if (lane == 0) p = atomicAdd(&s_ctl[1], 1);
            p = __shfl_sync(0xffffffffu, p, 0);
            if (p >= npatch) break;
            const int i = w.x0 + (p % npx) * 8 + (lane & 7), j = w.y0 + (p / npx) * 4 + (lane >> 3);
            if (i >= w.x1 || j >= w.y1) continue;
            Ray r;
            int k_lo, k_hi;
            if (!make_ray(cam, V.nx, V.ny, V.nz, i, j, r)) continue;
            if (!box_range(V.nx, V.ny, V.nz, r, cam.step, lo, hi, k_lo, k_hi)) continue;
            float *px = image + (long long)j * pitch_f + (MODE == VR_MIP ? i : 4 * i);
            State A = { 0.0f, 0.0f, 0.0f, 1.0f, -CUDART_INF_F };
            if (MODE == VR_MIP) A.m = __ldcg(px);
            else {
                const float4 s = __ldcg(reinterpret_cast<const float4 *>(px));
                A.cr = s.x; A.cg = s.y; A.cb = s.z; A.T = s.w;
                if (ERT && A.T <= cam.t_min) continue;            // this ray already terminated
            }
            if (interior) march_tile<C, MODE, ERT, true>(ts, org, r, cam, V.nx, V.ny, V.nz, tf_s, tf.scale, tf.bias, k_lo, k_hi, A);
            else march_tile<C, MODE, ERT, false>(ts, org, r, cam, V.nx, V.ny, V.nz, tf_s, tf.scale, tf.bias, k_lo, k_hi, A);
            if (MODE == VR_MIP) __stcg(px, A.m);
            else __stcg(reinterpret_cast<float4 *>(px), make_float4(A.cr, A.cg, A.cb, A.T));
        }
    }
}

template <class C>
vr_status launch_cfg(int mode, bool ert, const CamK &cam, const TilePlanK &P, const VolK &vol, const TfK &tf,
                     const TileWork *work, unsigned int *ctrl, unsigned int *done, unsigned int serial, float *image,
                     long long pitch_f, int sm_count, cudaStream_t st)
{
#define VR_TILE_LAUNCH(M, E)                                                                                          \
    do {                                                                                                              \
        auto kern = k_tile_march<C, M, E>;                                                                            \
        static int occ = 0;                                                                                           \
        if (occ == 0) {                                                                                               \
            VR_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM));           \
            VR_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, kThreads, C::SMEM));                    \
            if (occ < 1) { occ = 0; set_error("tile kernel does not fit on this device"); return VR_ERR_UNSUPPORTED; } \
        }                                                                                                             \
        const int grid = (int)std::min<long long>((long long)sm_count * occ, P.n_tiles);                              \
        kern<<<grid, kThreads, C::SMEM, st>>>(cam, P, vol, tf, work, ctrl, done, serial, image, pitch_f);             \
    } while (0)
    if (mode == VR_MIP) VR_TILE_LAUNCH(VR_MIP, false);
    else if (ert) VR_TILE_LAUNCH(VR_EA, true);
    else VR_TILE_LAUNCH(VR_EA, false);
#undef VR_TILE_LAUNCH
    return VR_OK;
}

}  // namespace

void tile_dims(int kind, int T[3])
{
    switch (kind) {
    case VR_TILE_32: T[0] = T[1] = T[2] = 32; break;
    case VR_TILE_32x16x16: T[0] = 32; T[1] = T[2] = 16; break;
    case VR_TILE_16: T[0] = T[1] = T[2] = 16; break;
    default: T[0] = T[1] = 32; T[2] = 16; break;
    }
}

void launch_tile_plan(const CamK &cam, const TilePlanK &P, const VolK &vol, const unsigned int *lvl_off,
                      unsigned int *ctrl, TileWork *work, cudaStream_t st)
{
    k_tile_plan<<<(P.n_tiles + 255) / 256, 256, 0, st>>>(cam, P, vol.nx, vol.ny, vol.nz, lvl_off, ctrl, work);
}

vr_status launch_tile_march(int kind, int mode, bool ert, const CamK &cam, const TilePlanK &P, const VolK &vol,
                            const TfK &tf, const TileWork *work, unsigned int *ctrl, unsigned int *done,
                            unsigned int serial, float *image, long long pitch_f, int sm_count, cudaStream_t st)
{
    switch (kind) {
    case VR_TILE_32:
        return launch_cfg<TileCfg<32, 32, 32>>(mode, ert, cam, P, vol, tf, work, ctrl, done, serial, image, pitch_f, sm_count, st);
    case VR_TILE_32x16x16:
        return launch_cfg<TileCfg<32, 16, 16>>(mode, ert, cam, P, vol, tf, work, ctrl, done, serial, image, pitch_f, sm_count, st);
    case VR_TILE_16:
        return launch_cfg<TileCfg<16, 16, 16>>(mode, ert, cam, P, vol, tf, work, ctrl, done, serial, image, pitch_f, sm_count, st);
    default:
        return launch_cfg<TileCfg<32, 32, 16>>(mode, ert, cam, P, vol, tf, work, ctrl, done, serial, image, pitch_f, sm_count, st);
    }
}

}  // namespace vr
