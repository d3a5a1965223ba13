// vr_lanes.cu — the default ray-caster of resident linear volumes: one thread per ray, ray state in
// registers from the first sample to the last (exact C.5 / ERT), the 8 corner voxels of every sample read
// straight from global memory through L1 ("the GPU part").
//
// What decides the speed of such a kernel on B200 is the number of distinct 128-byte lines the 32 lanes of
// a warp touch per corner load: the L1 pipe retires about one line per clock per SM, and the path issues 8
// loads per sample.  The design therefore chooses, per frame, WHICH 32 rays form a warp so that their
// samples at equal k run along the memory-fast axis of the volume:
//   * lanes run along the image axis (u or v) whose footprint on the principal plane of the view moves
//     most along the fast axis, and the image rows are SHEARED by an integer row offset off(p) =
//     floor(sigma p + 1/2) of the lane coordinate p, so that a warp follows one row of voxels instead of
//     drifting across rows (any function off(p) gives a bijection of the pixels: sigma only affects speed);
//   * the sample lattice of C.2 is anchored at the volume entry, so the lanes of a warp start on the same
//     entry face; a lane that gets more than `lag` base planes ahead of the slowest active lane of its warp
//     waits one iteration, which keeps the 32 samples of an iteration on one or two data planes;
//   * rays that travel mostly along x cannot be served from an x-fastest array (every lane would sit on its
//     own line): the library keeps a second, z-fastest copy of the volume (vr_api.cu, made once, lazily)
//     and such pixels are rendered from it by the same kernel with permuted strides.  A pixel belongs to
//     the x-fastest copy iff |d_x| <= |d_z|.
// All arithmetic is the canonical sequence of vr_math.cuh; indices are the clamped base indices of C.3, so
// every address formed here is inside the volume by construction.
#include <climits>

#include "vr_internal.h"

namespace vr {

namespace {

constexpr int kRowsPerCta = kLaneRowsPerCta, kLaneThreads = 32 * kRowsPerCta;

// transfer function in shared memory as two float2 tables ((r,g) and (b,a)); entry 256 = copy of 255
struct TfS { float2 rg[257], ba[257]; };

__device__ __forceinline__ void stage_tf_pairs(TfS &s, const TfK &tf)
{
    for (int e = threadIdx.x; e < 257; e += kLaneThreads) {
        const float4 v = __ldg(tf.table + e);
        s.rg[e] = make_float2(v.x, v.y);
        s.ba[e] = make_float2(v.z, v.w);
    }
    __syncthreads();
}

// C.4 with the four channel lerps paired (same operations and operands as classify() of vr_math.cuh)
__device__ __forceinline__ float4 classify_s(const TfS &s, float scale, float bias, float v)
{
    const float u = __saturatef(__fmaf_rn(v, scale, bias));
    const float x = __fmul_rn(u, 255.0f);
    const int i = min(__float2int_rz(x), 254);
    const float f = __fsub_rn(x, (float)i);
    const float2 rg = lerp_ee2(s.rg[i], s.rg[i + 1], f);
    const float2 ba = lerp_ee2(s.ba[i], s.ba[i + 1], f);
    return make_float4(rg.x, rg.y, ba.x, ba.y);
}

// C.5 with the r and g accumulations paired
__device__ __forceinline__ void composite_p(float4 rgba, float &Cr, float &Cg, float &Cb, float &T)
{
    const float w = __fmul_rn(T, rgba.w);
    const float2 c = fma2_rn(make_float2(w, w), make_float2(rgba.x, rgba.y), make_float2(Cr, Cg));
    Cr = c.x; Cg = c.y;
    Cb = __fmaf_rn(w, rgba.z, Cb);
    T = __fsub_rn(T, w);
}

// the 8 corners of base index (ix,iy,iz): FAST = the axis with element stride 1 (0: x-fastest array,
// 2: z-fastest copy); sa, sb = element strides of the other two axes in ascending axis order
template <bool WIDE, int FAST>
__device__ __forceinline__ const float *cell_pointer(const LaneVolK &V, int ix, int iy, int iz)
{
    // offset = slow index * slow stride + (middle index * middle stride + fast index): the bracket is an offset
    // inside one plane and the slow stride is a plane size, both < 2^32 (checked by launch_rows), so the only
    // 64-bit operation of the WIDE case is one 32 x 32 -> 64-bit multiply-add (indices are >= 0 by C.3)
    const unsigned int in_plane = FAST == 0 ? (unsigned int)iy * (unsigned int)V.sa + (unsigned int)ix
                                            : (unsigned int)iy * (unsigned int)V.sb + (unsigned int)iz;
    const unsigned int slow = FAST == 0 ? (unsigned int)iz : (unsigned int)ix;
    const unsigned int s_slow = FAST == 0 ? (unsigned int)V.sb : (unsigned int)V.sa;
    const float *p;
    if (WIDE) p = V.base + ((unsigned long long)slow * s_slow + in_plane);
    else p = V.base + (slow * s_slow + in_plane);
    return p;
}

// elements u and u + 1 of a row through ONE aligned 16-byte load of the quad that holds u (o = u & 3 is u's place in
// it) plus, only where u ends its quad, a scalar load of u + 1.  Rows start 16-byte aligned and their length is a
// multiple of 4 (checked by launch_rows), so the quad never leaves the row; u + 1 is a voxel by C.3.
__device__ __forceinline__ void load_pair_quad(const float *quad, int o, float &a, float &b)
{
    const float4 q = __ldg(reinterpret_cast<const float4 *>(quad));
    float e = 0.0f;
    if (o == 3) e = __ldg(quad + 4);
    const bool hi = (o & 2) != 0, odd = (o & 1) != 0;
    const float t0 = hi ? q.z : q.x, t1 = hi ? q.w : q.y, t2 = hi ? e : q.z;
    a = odd ? t1 : t0;
    b = odd ? t2 : t1;
}

// the 8 corner voxels of a ray's current cell, kept in registers from one sample to the next
struct Cell {
    int ix, iy, iz;                                          // base index the values belong to (ix < 0: none yet)
    float q00, q01, q10, q11, r00, r01, r10, r11;
};

// REUSE (kernel-uniform): with a step below one voxel consecutive samples of a ray often fall into the same cell
// (all three base indices unchanged: ~40 % of the samples at step 0.5); their 8 voxels are then still in registers
// and nothing is loaded.  Same values, so bit-identical results; fewer cache lines touched per sample.
template <bool WIDE, int FAST, bool QUAD>
__device__ __forceinline__ float sample_cell(const LaneVolK &V, Cell &c, bool reuse, int ix, int iy, int iz, float fx, float fy,
                                             float fz)
{
    if (!reuse || ix != c.ix || iy != c.iy || iz != c.iz) {
        const int o = QUAD ? ((FAST == 0 ? ix : iz) & 3) : 0;
        // QUAD: p addresses the aligned quad of the fast index (the fast index enters the offset rounded down to 4)
        const float *p = FAST == 0 ? cell_pointer<WIDE, FAST>(V, ix - o, iy, iz) : cell_pointer<WIDE, FAST>(V, ix, iy, iz - o);
        const float *pa = p + V.sa, *pb = p + V.sb, *pab = pb + V.sa;
        if (QUAD) {
            load_pair_quad(p, o, c.q00, c.q01); load_pair_quad(pa, o, c.q10, c.q11);
            load_pair_quad(pb, o, c.r00, c.r01); load_pair_quad(pab, o, c.r10, c.r11);
        } else {
            c.q00 = __ldg(p); c.q01 = __ldg(p + 1);          // (a, b) = (0, 0): unit-stride neighbours
            c.q10 = __ldg(pa); c.q11 = __ldg(pa + 1);        // a + 1
            c.r00 = __ldg(pb); c.r01 = __ldg(pb + 1);        // b + 1
            c.r10 = __ldg(pab); c.r11 = __ldg(pab + 1);      // a + 1, b + 1
        }
        c.ix = ix; c.iy = iy; c.iz = iz;
    }
    // trilerp_packed(v000, v100, v010, v110, v001, v101, v011, v111): corner (X,Y,Z)
    if (FAST == 0)      // u = x, a = y, b = z
        return trilerp_packed(c.q00, c.q01, c.q10, c.q11, c.r00, c.r01, c.r10, c.r11, fx, fy, fz);
    else                // u = z, a = x, b = y
        return trilerp_packed(c.q00, c.q10, c.r00, c.r10, c.q01, c.q11, c.r01, c.r11, fx, fy, fz);
}

// Empty-space leap (vr_macro.cu): sample k of the ray, at parameter t with base index (ix,iy,iz), lies in an empty
// cell of 2^lg base indices per axis.  Returns n >= 1 such that samples k .. k+n-1 all lie in that cell (so all
// have opacity exactly 0 and may be skipped).  n is ESTIMATED from the slab exit of the cell and then VERIFIED:
// base indices are monotone in t on every axis, so if the position of sample k+n-1 (or the ray's exit point, if
// that comes first) has the same cell, every sample in between has it too; otherwise n = 1.  The march continues from the canonical t_{k+n} = fma(k+n, step, t_first).
__device__ __forceinline__ float leap_samples(int lg, const Ray &r, const float *inv, float inv_step, float step, float t,
                                              float kf, int ix, int iy, int iz, int nx, int ny, int nz)
{
    const int i[3] = { ix, iy, iz };
    float t_out = CUDART_INF_F;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const int org = (i[a] >> lg) << lg;
        const float bound = (float)(r.d[a] > 0.0f ? org + (1 << lg) : org);
        if (r.d[a] != 0.0f) t_out = fminf(t_out, (bound - r.oc[a]) * inv[a]);
    }
    float nf = fminf(fmaxf(floorf((t_out - t) * inv_step), 1.0f), 65536.0f);      // NaN -> 1
    if (nf > 1.0f) {
        // the last skipped sample, or the exit point of the ray when that comes first (the cell of a position is
        // monotone in t for every real t, so the samples up to the exit are covered as well)
        const float tl = fminf(__fmaf_rn(__fadd_rn(kf, __fsub_rn(nf, 1.0f)), step, r.t_first), r.t_exit);
        int jx, jy, jz;
        float g;
        axis_cell(tl, r.d[0], r.oc[0], nx, jx, g);
        axis_cell(tl, r.d[1], r.oc[1], ny, jy, g);
        axis_cell(tl, r.d[2], r.oc[2], nz, jz, g);
        const bool same = (jx >> lg) == (ix >> lg) && (jy >> lg) == (iy >> lg) && (jz >> lg) == (iz >> lg);
        if (!same) { nf = 1.0f; VR_TEST_COUNT(VR_CNT_LEAP_REJECTED); }
        else VR_TEST_COUNT(lg == 6 ? VR_CNT_LEAP_BLOCK : VR_CNT_LEAP_CELL);
    }
    return nf;
}

// sort-last partials (C.7): writes the fragment (C_b, T_b) / m_b of pixel (i,j) for the brick with plan index `cur`
template <int MODE>
__device__ __forceinline__ void flush_fragment(const PartK &P, int cur, int i, int j, float cr, float cg, float cb, float T,
                                               float m)
{
    const BrickK *b = P.bricks + cur;
    const int x0 = __ldg(&b->x0), y0 = __ldg(&b->y0), x1 = __ldg(&b->x1), y1 = __ldg(&b->y1);
    if (i < x0 || i >= x1 || j < y0 || j >= y1) { VR_TEST_COUNT(VR_CNT_FRAG_OUTSIDE); return; }   // never: the rectangle holds every owning pixel (A4)
    const unsigned long long f = __ldg(&b->frag_off) + (unsigned long long)(j - y0) * (unsigned)(x1 - x0) + (unsigned)(i - x0);
    if (MODE == VR_MIP) P.arena[f] = m;
    else reinterpret_cast<float4 *>(P.arena)[f] = make_float4(cr, cg, cb, T);
}

// PART: instead of one pixel value per ray, one fragment per (ray, owner brick): the ray state is flushed to the
// brick's fragment and reset whenever the owner brick (ix/B, iy/B, iz/B) of the next sample changes — the same
// samples in the same order as the per-brick marches of C.7, so the fragments are bit-identical to theirs.
template <int MODE, bool ERT, bool WIDE, int FAST, bool SKIP, bool PART, bool QUAD>
__global__ void __launch_bounds__(kLaneThreads)
k_rows(CamK cam, LaneVolK V, TfK tf, LaneMapK M, MacroK Mc, PartK P, float *__restrict__ image, long long pitch_f)
{
    __shared__ TfS tf_s;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // pixel of this lane (vr_lanemap.h): tiles of 32 lanes x kLaneTileH rows, each sheared by its own sigma
    int li, lj, rows_of_tile;
    lane_pixel(cam, M, cam.sub, cam.sx, cam.sy, (int)blockIdx.x, (int)blockIdx.y, warp, lane, li, lj, rows_of_tile);
    if (((int)blockIdx.y % M.bpt) * kLaneRowsPerCta >= rows_of_tile) return;    // a CTA beyond the tile's sheared rows (CTA-uniform)
    if (MODE == VR_EA) stage_tf_pairs(tf_s, tf);
    // exact empty-space skipping (vr_macro.cu): used only when enough cells are empty under this transfer function
    const bool skipping = SKIP && __ldg(Mc.n_skip) >= Mc.min_skip;
    const int cxy = Mc.cx * Mc.cy;
    const bool inside = li >= 0 && li < cam.width && lj >= 0 && lj < cam.height;
    const int i = li * cam.sub + cam.sx, j = lj * cam.sub + cam.sy;              // image pixel (C.1 uses these)
    Ray r;
    bool mine = false, alive = false;
    if (inside) {
        const bool hit = make_ray(cam, V.nx, V.ny, V.nz, i, j, r);
        const bool xmajor = fabsf(r.d[0]) > fabsf(r.d[2]);
        mine = M.cls == 0 || (M.cls == 2) == xmajor;
        // a direction that is not finite (d0 + px du + py dv = 0) has no defined samples: treated as a miss
        alive = mine && hit && r.t_exit < CUDART_INF_F;
    }
    if (!__any_sync(0xffffffffu, mine)) return;
    if (!alive) { r.t_first = 0.0f; r.t_exit = -CUDART_INF_F; r.d[0] = r.d[1] = r.d[2] = 0.0f; r.oc[0] = r.oc[1] = r.oc[2] = 0.0f; }
    float cr = 0.0f, cg = 0.0f, cb = 0.0f, T = 1.0f, m = -CUDART_INF_F;
    float kf = 0.0f;
    const int lag = M.lag;
    Cell cell;
    cell.ix = cell.iy = cell.iz = -1;
    cell.q00 = cell.q01 = cell.q10 = cell.q11 = cell.r00 = cell.r01 = cell.r10 = cell.r11 = 0.0f;
    const bool reuse = M.reuse != 0;
    int cur = -1, blo[3] = { 1, 1, 1 }, bhi[3] = { 0, 0, 0 };      // PART: plan index and base-index box of the owner brick
    float inv[3] = { 0.0f, 0.0f, 0.0f };
    const float inv_step = SKIP ? 1.0f / cam.step : 0.0f;
    if (SKIP) {
#pragma unroll
        for (int a = 0; a < 3; ++a) inv[a] = 1.0f / r.d[a];          // only used by the leap estimate (d_a != 0 checked there)
    }
    // a ray that is not marched (miss, other class, outside the image) or has terminated has t_exit below every t_k
    for (;;) {
        const float t = __fmaf_rn(kf, cam.step, r.t_first);
        alive = t < r.t_exit;                                        // C.2: sample k exists iff t_k < t_exit
        if (!__any_sync(0xffffffffu, alive)) break;
        int ix, iy, iz;
        float fx, fy, fz;
        axis_cell(t, r.d[0], r.oc[0], V.nx, ix, fx);
        axis_cell(t, r.d[1], r.oc[1], V.ny, iy, fy);
        axis_cell(t, r.d[2], r.oc[2], V.nz, iz, fz);
        bool go = alive;
        if (lag > 0) {
            const int prog = ix * M.w[0] + iy * M.w[1] + iz * M.w[2];        // +- the base index along the principal axis
            const int slowest = __reduce_min_sync(0xffffffffu, alive ? prog : INT_MAX);
            go = alive && prog - slowest <= lag;
            if (alive && !go) VR_TEST_COUNT(VR_CNT_LAG_WAIT);
        }
#ifdef VR_SIMT_HOST
        if (!SKIP) {                 // traffic model of the emulation: reached by every lane of the warp, every iteration
            const float *p = cell_pointer<WIDE, FAST>(V, ix, iy, iz);
            const bool loads = go && (!reuse || ix != cell.ix || iy != cell.iy || iz != cell.iz);
            VR_TRACE_CORNER_LOADS(go, loads, V.base, p, p + V.sa, p + V.sb, p + V.sb + V.sa);
        }
#endif
        if (PART && go && (ix < blo[0] || ix > bhi[0] || iy < blo[1] || iy > bhi[1] || iz < blo[2] || iz > bhi[2])) {
            if (cur >= 0) flush_fragment<MODE>(P, cur, i, j, cr, cg, cb, T, m);
            const int bx = ix / P.B, by = iy / P.B, bz = iz / P.B;
            cur = __ldg(P.lut + (bz * P.nby + by) * P.nbx + bx);
            if (cur < 0) VR_TEST_COUNT(VR_CNT_FRAG_NO_BRICK);      // never: a brick that owns a sample is in the plan (A4)
            blo[0] = bx * P.B; blo[1] = by * P.B; blo[2] = bz * P.B;
            bhi[0] = blo[0] + P.B - 1; bhi[1] = blo[1] + P.B - 1; bhi[2] = blo[2] + P.B - 1;
            cr = cg = cb = 0.0f; T = 1.0f; m = -CUDART_INF_F;
        }
        if (go) {
            // a sample based in an empty macrocell has opacity exactly 0: compositing it changes nothing (C.5)
            unsigned int empty = 0u;
            if (SKIP && skipping) empty = __ldg(Mc.flag + ((iz >> 3) * cxy + (iy >> 3) * Mc.cx + (ix >> 3)));
            if (!SKIP || empty == 0u) {
                const float s = sample_cell<WIDE, FAST, QUAD>(V, cell, reuse, ix, iy, iz, fx, fy, fz);
                if (MODE == VR_MIP) m = fmaxf(m, s);
                else {
                    composite_p(classify_s(tf_s, tf.scale, tf.bias, s), cr, cg, cb, T);
                    if (ERT && T <= cam.t_min) r.t_exit = -CUDART_INF_F;      // stop AFTER compositing this sample (C.5)
                }
                kf = __fadd_rn(kf, 1.0f);                            // exact: k < 2^24
            } else                                                   // leap to the end of the empty cell (or block of cells)
                kf = __fadd_rn(kf, leap_samples((empty & 2u) ? 6 : 3, r, inv, inv_step, cam.step, t, kf, ix, iy, iz, V.nx, V.ny, V.nz));
        }
    }
    if (!mine) return;
    if (PART) {
        if (cur >= 0) flush_fragment<MODE>(P, cur, i, j, cr, cg, cb, T, m);
        return;
    }
    if (MODE == VR_MIP) image[(long long)j * pitch_f + i] = m;
    else
        *reinterpret_cast<float4 *>(image + (long long)j * pitch_f + 4 * (long long)i) =
            make_float4(cr, cg, cb, __fsub_rn(1.0f, T));
}

// identity fragments (C.7): a pixel of a brick's rectangle whose ray owns no sample in the brick folds as nothing
template <int MODE>
__global__ void __launch_bounds__(256) k_fragment_init(float *__restrict__ arena, unsigned long long n_frag)
{
    const unsigned long long stride = (unsigned long long)gridDim.x * 256;
    for (unsigned long long f = (unsigned long long)blockIdx.x * 256 + threadIdx.x; f < n_frag; f += stride) {
        if (MODE == VR_MIP) arena[f] = -CUDART_INF_F;
        else reinterpret_cast<float4 *>(arena)[f] = make_float4(0.0f, 0.0f, 0.0f, 1.0f);
    }
}

// z-fastest copy: out[x][y][z] = in[z][y][x]; one CTA transposes a 32 (x) by 32 (z) tile of one y
__global__ void __launch_bounds__(256)
k_transpose_xz(const float *__restrict__ in, float *__restrict__ out, int nx, int ny, int nz)
{
    __shared__ float tile[32][33];
    const int y = blockIdx.z, x0 = blockIdx.x * 32, z0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int r = ty; r < 32; r += 8) {
        const int x = x0 + tx, z = z0 + r;
        if (x < nx && z < nz) tile[r][tx] = __ldg(in + ((long long)z * ny + y) * nx + x);
    }
    __syncthreads();
    for (int r = ty; r < 32; r += 8) {
        const int x = x0 + r, z = z0 + tx;
        if (x < nx && z < nz) out[((long long)x * ny + y) * nz + z] = tile[tx][r];
    }
}

}  // namespace

bool launch_rows(int mode, bool ert, const CamK &cam, const LaneVolK &vol, int fast, const TfK &tf, const LaneMapK &map,
                 const MacroK &macro, const PartK *part, bool force_wide, bool quad_loads, int rows, float *image,
                 long long pitch_f, cudaStream_t st)
{
    const int n_lane = map.lane_axis == 0 ? cam.width : cam.height;
    const dim3 g((unsigned)((n_lane + 31) / 32), (unsigned)((rows + kRowsPerCta - 1) / kRowsPerCta));
    if (g.x == 0 || g.y == 0) return false;
    const unsigned long long span = (unsigned long long)((fast == 0 ? vol.nz : vol.ny) - 1) * (unsigned long long)vol.sb +
                                    (unsigned long long)((fast == 0 ? vol.ny : vol.nx) - 1) * (unsigned long long)vol.sa +
                                    (unsigned long long)(fast == 0 ? vol.nx : vol.nz);
    const bool wide = force_wide || span > 0xffffffffull;
    const bool skip = mode == VR_EA && macro.flag != nullptr && !part;
    // 16-byte row loads need rows that start 16-byte aligned (the base is, vr_create_volume) and hold a multiple of 4
    const bool quad = quad_loads && !skip && ((fast == 0 ? vol.nx : vol.nz) & 3) == 0 &&
                      (((uintptr_t)vol.base) & 15u) == 0;
    PartK P;
    if (part) P = *part;
    else { P.bricks = nullptr; P.lut = nullptr; P.arena = nullptr; P.B = 1; P.nbx = P.nby = 0; }
#define VR_L4(M, E, Wd, F, S) vr_launch(k_rows<M, E, Wd, F, S, false, false>, g, kLaneThreads, 0, st, cam, vol, tf, map, macro, P, image, pitch_f)
#define VR_L3(M, E, Wd, F) do { \
        if (part && quad) vr_launch(k_rows<M, false, Wd, F, false, true, true>, g, kLaneThreads, 0, st, cam, vol, tf, map, macro, P, image, pitch_f); \
        else if (part) vr_launch(k_rows<M, false, Wd, F, false, true, false>, g, kLaneThreads, 0, st, cam, vol, tf, map, macro, P, image, pitch_f); \
        else if (quad) vr_launch(k_rows<M, E, Wd, F, false, false, true>, g, kLaneThreads, 0, st, cam, vol, tf, map, macro, P, image, pitch_f); \
        else if (M == VR_EA && skip) VR_L4(M, E, Wd, F, (M == VR_EA)); else VR_L4(M, E, Wd, F, false); } while (0)
#define VR_L2(M, E, Wd) do { if (fast == 0) VR_L3(M, E, Wd, 0); else VR_L3(M, E, Wd, 2); } while (0)
#define VR_L1(M, E) do { if (wide) VR_L2(M, E, true); else VR_L2(M, E, false); } while (0)
    if (mode == VR_MIP) VR_L1(VR_MIP, false);
    else if (ert) VR_L1(VR_EA, true);
    else VR_L1(VR_EA, false);
#undef VR_L1
#undef VR_L2
#undef VR_L3
#undef VR_L4
    return quad;
}

void launch_fragment_init(int mode, float *arena, unsigned long long n_frag, int grid, cudaStream_t st)
{
    if (n_frag == 0) return;
    if (mode == VR_MIP) vr_launch(k_fragment_init<VR_MIP>, grid, 256, 0, st, arena, n_frag);
    else vr_launch(k_fragment_init<VR_EA>, grid, 256, 0, st, arena, n_frag);
}

void launch_transpose_xz(const float *in, float *out, int nx, int ny, int nz, cudaStream_t st)
{
    // gridDim.y, .z <= 65535: nz <= 2^21 and ny <= 65535 per launch; larger y extents go slab by slab
    for (int y0 = 0; y0 < ny; y0 += 65535) {
        const int yn = ny - y0 < 65535 ? ny - y0 : 65535;
        const dim3 g((unsigned)((nx + 31) / 32), (unsigned)((nz + 31) / 32), (unsigned)yn);
        vr_launch(k_transpose_xz, g, 256, 0, st, in + (long long)y0 * nx, out + (long long)y0 * nz, nx, ny, nz);
    }
}

}  // namespace vr
