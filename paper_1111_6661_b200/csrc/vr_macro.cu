// vr_macro.cu — exact transfer-function-aware empty-space skipping (the "interactive" of
// PAPER.md:L34): a grid of macrocells of 8^3 base indices with the min / max of every voxel a sample based in
// the cell can read, and, per transfer function, one byte per cell that says "every sample based here has
// opacity exactly 0".  Such a sample changes nothing in C.5 (w = T * 0 = 0; fma(0, rgb, C) = C; T - 0 = T), so
// the ray-caster may skip it without reading its 8 voxels: the image stays bit-identical.
//
// Why the byte is exact.  A sample based at (ix,iy,iz) reads voxels [ix, ix+1] x [iy, iy+1] x [iz, iz+1]; cell c
// covers base indices [8c, 8c+7] per axis, hence voxels [8c, 8c+8] (clamped to the volume).  The trilinear value
// is three levels of exact-ends lerps L(a,b,f) = fma(f, b, fma(-f, a, a)), each within 2^-23 max(|a|,|b|) of a
// convex combination of its operands, so s lies in [mn - e, mx + e] with e = 2^-21 max(|mn|,|mx|) + FLT_MIN (four
// times the three-level bound, plus the absolute error of results in the subnormal range).  C.4's u = sat(fma(s, scale, bias)), x = u * 255, i = min((int)x, 254) are monotone
// non-decreasing in s (scale > 0; rounding is monotone), so i lies in [i(mn - e), i(mx + e)], both evaluated by
// the same float32 sequence.  The sample's opacity is L(A[i], A[i+1], f), which is exactly +0 when A[i] = A[i+1]
// = 0.  The cell is skippable iff A[j] = 0 for all j in [i(mn - e), i(mx + e) + 1].  A cell that holds a
// non-finite voxel is never skippable.
#include <float.h>

#include "vr_internal.h"

namespace vr {

namespace {

constexpr int kM = kMacroEdge;

// One CTA = one row of cells along x at cell coordinates (blockIdx.x = cy, blockIdx.y = cz): 9 x 9 voxel rows,
// threads along x (coalesced), per-column min / max in shared memory, then one thread per cell.
__global__ void __launch_bounds__(256) k_macro_minmax(const float *__restrict__ v, int nx, int ny, int nz, int cx,
                                                      float2 *__restrict__ mm)
{
    __shared__ float s_mn[257], s_mx[257];
    const int cy = blockIdx.x, cz = blockIdx.y;
    const long long sy = nx, sz = (long long)nx * ny;
    for (int x0 = 0; x0 < cx * kM; x0 += 256) {
        for (int col = threadIdx.x; col < 257; col += 256) {
            const int x = min(x0 + col, nx - 1);
            float mn = CUDART_INF_F, mx = -CUDART_INF_F;
            bool bad = false;
            for (int dz = 0; dz <= kM; ++dz) {
                const int z = min(cz * kM + dz, nz - 1);
                for (int dy = 0; dy <= kM; ++dy) {
                    const int y = min(cy * kM + dy, ny - 1);
                    const float a = __ldg(v + z * sz + y * sy + x);
                    if (fabsf(a) <= FLT_MAX) { mn = fminf(mn, a); mx = fmaxf(mx, a); } else bad = true;
                }
            }
            s_mn[col] = bad ? -CUDART_INF_F : mn;
            s_mx[col] = bad ? CUDART_INF_F : mx;
        }
        __syncthreads();
        const int c = x0 / kM + threadIdx.x;
        if (threadIdx.x < 32 && c < cx) {
            float mn = CUDART_INF_F, mx = -CUDART_INF_F;
            for (int d = 0; d <= kM; ++d) { mn = fminf(mn, s_mn[threadIdx.x * kM + d]); mx = fmaxf(mx, s_mx[threadIdx.x * kM + d]); }
            mm[((long long)cz * gridDim.x + cy) * cx + c] = make_float2(mn, mx);
        }
        __syncthreads();
    }
}

// C.4 table index of a scalar (the same float32 sequence as classify())
__device__ __forceinline__ int tf_index(float s, float scale, float bias)
{
    const float u = __saturatef(__fmaf_rn(s, scale, bias));
    return min(__float2int_rz(__fmul_rn(u, 255.0f)), 254);
}

__global__ void __launch_bounds__(256) k_macro_flags(const float2 *__restrict__ mm, long long n_cells, TfK tf,
                                                     unsigned char *__restrict__ flag, unsigned long long *n_skip)
{
    __shared__ int s_nz[258];                       // s_nz[j] = number of entries < j with alpha != 0 (entry 256 = pad copy)
    if (threadIdx.x == 0) {
        int acc = 0;
        for (int j = 0; j <= 256; ++j) { s_nz[j] = acc; acc += __ldg(&tf.table[j].w) != 0.0f ? 1 : 0; }
        s_nz[257] = acc;
    }
    __syncthreads();
    unsigned int mine = 0;
    for (long long c = (long long)blockIdx.x * 256 + threadIdx.x; c < n_cells; c += (long long)gridDim.x * 256) {
        const float2 r = mm[c];
        unsigned char f = 0;
        if (r.x >= -FLT_MAX && r.y <= FLT_MAX && r.x <= r.y) {
            const float e = __fmaf_rn(fmaxf(fabsf(r.x), fabsf(r.y)), 4.76837158203125e-7f, FLT_MIN);     // 2^-21 R (+ the subnormal range)
            const int lo = tf_index(__fsub_rn(r.x, e), tf.scale, tf.bias), hi = tf_index(__fadd_rn(r.y, e), tf.scale, tf.bias);
            f = s_nz[hi + 2] - s_nz[lo] == 0 ? 1 : 0;     // entries lo .. hi+1 all have alpha == 0
        }
        flag[c] = f;
        mine += f;
    }
    mine = __reduce_add_sync(0xffffffffu, mine);
    if ((threadIdx.x & 31) == 0 && mine) atomicAdd(n_skip, (unsigned long long)mine);
}

// bit 1 of a cell's byte: every cell of its block of 8 x 8 x 8 cells (64^3 base indices) is empty.  One warp per block.
__global__ void __launch_bounds__(256) k_macro_blocks(unsigned char *__restrict__ flag, int cx, int cy, int cz)
{
    const int bx_n = (cx + 7) / 8, by_n = (cy + 7) / 8, bz_n = (cz + 7) / 8;
    const long long n_blocks = (long long)bx_n * by_n * bz_n;
    const int lane = threadIdx.x & 31;
    for (long long b = (long long)blockIdx.x * 8 + (threadIdx.x >> 5); b < n_blocks; b += (long long)gridDim.x * 8) {
        const int bx = (int)(b % bx_n), by = (int)(b / bx_n % by_n), bz = (int)(b / ((long long)bx_n * by_n));
        bool all = true;
        for (int e = lane; e < 512; e += 32) {
            const int x = bx * 8 + (e & 7), y = by * 8 + (e >> 3 & 7), z = bz * 8 + (e >> 6);
            if (x < cx && y < cy && z < cz) all = all && (flag[((long long)z * cy + y) * cx + x] & 1u) != 0;
        }
        if (!__all_sync(0xffffffffu, all)) continue;
        for (int e = lane; e < 512; e += 32) {
            const int x = bx * 8 + (e & 7), y = by * 8 + (e >> 3 & 7), z = bz * 8 + (e >> 6);
            if (x < cx && y < cy && z < cz) flag[((long long)z * cy + y) * cx + x] = 3u;
        }
    }
}

// value range of one brick slot (all (B+1)^3 voxels a sample owned by the brick can read): order-preserving keys
// of min and max over the finite voxels, and whether a non-finite voxel was seen.  r is zero-initialised to
// { key(+inf), key(-inf), 0 } by k_brick_range_init.
__global__ void __launch_bounds__(256) k_brick_range_init(BrickRangeK *r, unsigned long long n)
{
    const unsigned long long i = (unsigned long long)blockIdx.x * 256 + threadIdx.x;
    if (i < n) { r[i].enc_min = 0xff800000u; r[i].enc_max = 0x007fffffu; r[i].bad = 0u; r[i].pad = 0u; }
}

__global__ void __launch_bounds__(256) k_brick_range(const float *__restrict__ v, unsigned long long n, BrickRangeK *r)
{
    unsigned int kmin = 0xffffffffu, kmax = 0u, bad = 0u;
    for (unsigned long long i = (unsigned long long)blockIdx.x * 256 + threadIdx.x; i < n; i += (unsigned long long)gridDim.x * 256) {
        const float a = __ldg(v + i);
        if (fabsf(a) <= FLT_MAX) {
            const unsigned int b = __float_as_uint(a), k = (b & 0x80000000u) ? ~b : (b | 0x80000000u);
            kmin = min(kmin, k); kmax = max(kmax, k);
        } else bad = 1u;
    }
    kmin = __reduce_min_sync(0xffffffffu, kmin); kmax = __reduce_max_sync(0xffffffffu, kmax);
    bad = __reduce_or_sync(0xffffffffu, bad);
    if ((threadIdx.x & 31) == 0) {
        atomicMin(&r->enc_min, kmin); atomicMax(&r->enc_max, kmax);
        if (bad) atomicOr(&r->bad, 1u);
    }
}

}  // namespace

void launch_brick_range_init(BrickRangeK *r, unsigned long long n, cudaStream_t st)
{
    vr_launch(k_brick_range_init, (unsigned)((n + 255) / 256), 256, 0, st, r, n);
}

void launch_brick_range(const float *v, unsigned long long n, BrickRangeK *r, int grid, cudaStream_t st)
{
    vr_launch(k_brick_range, grid, 256, 0, st, v, n, r);
}

void launch_macro_blocks(unsigned char *flag, const MacroK &m, int grid, cudaStream_t st)
{
    vr_launch(k_macro_blocks, grid, 256, 0, st, flag, m.cx, m.cy, m.cz);
}

void launch_macro_minmax(const float *v, int nx, int ny, int nz, const MacroK &m, float2 *mm, cudaStream_t st)
{
    // gridDim.y <= 65535 cells along z (nz <= 524280 voxels): checked by the caller
    vr_launch(k_macro_minmax, dim3((unsigned)m.cy, (unsigned)m.cz), 256, 0, st, v, nx, ny, nz, m.cx, mm);
}

void launch_macro_flags(const float2 *mm, long long n_cells, const TfK &tf, unsigned char *flag, unsigned long long *n_skip,
                        int grid, cudaStream_t st)
{
    vr_launch(k_macro_flags, grid, 256, 0, st, mm, n_cells, tf, flag, n_skip);
}

}  // namespace vr
