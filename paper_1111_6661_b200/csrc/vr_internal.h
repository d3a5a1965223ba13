// vr_internal.h — host-side handle, error plumbing and kernel launcher declarations.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/vr.h"
#include "vr_math.cuh"

namespace vr {

void set_error(const char *fmt, ...);
vr_status cuda_fail(cudaError_t e, const char *what);

#define VR_CUDA(call)                                                  \
    do {                                                               \
        cudaError_t e__ = (call);                                      \
        if (e__ != cudaSuccess) return ::vr::cuda_fail(e__, #call);    \
    } while (0)

#define VR_REQUIRE(cond, ...)                                          \
    do {                                                               \
        if (!(cond)) { ::vr::set_error(__VA_ARGS__); return VR_ERR_INVALID_ARG; } \
    } while (0)

// ---------------------------------------------------------------- reductions (vr_reduce.cu)
// device scratch of one summary call
struct SummaryScratch {
    unsigned int enc_min, enc_max;        // order-preserving uint encodings of the running min / max
    float lo, hi, scale_h;                // histogram range decided on the device
    unsigned int pad;
    unsigned long long n_nonfinite, n_below, n_above;
    unsigned long long counts[4096];
};

struct BoxK {                             // a box of voxels inside a strided array
    const float *base;
    long long sy, sz;
    int ex, ey, ez;
};

void launch_summary_reset(SummaryScratch *s, cudaStream_t st);
void launch_minmax_flat(const float *v, unsigned long long n, SummaryScratch *s, int grid, cudaStream_t st);
void launch_minmax_box(BoxK b, SummaryScratch *s, int grid, cudaStream_t st);
// range_mode 0: lo/hi = the device min/max; 1: lo/hi given
void launch_summary_range(SummaryScratch *s, int range_mode, float lo, float hi, uint32_t nbins, cudaStream_t st);
void launch_hist_flat(const float *v, unsigned long long n, uint32_t nbins, SummaryScratch *s, int grid, cudaStream_t st);
void launch_hist_box(BoxK b, uint32_t nbins, SummaryScratch *s, int grid, cudaStream_t st);
// fused single pass (caller gave the range): min/max and histogram together
void launch_minmax_hist_flat(const float *v, unsigned long long n, uint32_t nbins, SummaryScratch *s, int grid,
                             cudaStream_t st);
void launch_minmax_hist_box(BoxK b, uint32_t nbins, SummaryScratch *s, int grid, cudaStream_t st);
void launch_summary_finish(const SummaryScratch *s, uint32_t nbins, vr_summary *out, cudaStream_t st);

// ---------------------------------------------------------------- ray casting (vr_raycast.cu)
struct TfK { const float4 *table; float scale, bias; };   // 257 float4 entries in global memory

// one brick as the kernels see it (per-frame table, visibility order)
struct BrickK {
    const float *base;          // voxel (ox,oy,oz)
    long long sy, sz;
    int ox, oy, oz;             // index origin of base
    int lo[3], hi[3];           // owned base-index range, inclusive (C.7): i0_a in [lo_a, hi_a]
    int x0, y0, x1, y1;         // screen rectangle, [x0,x1) x [y0,y1)
    unsigned long long frag_off;   // first fragment of this brick in the arena (sort-last)
};

struct WorkK { int brick, tx, ty, pad; };   // one CTA of the brick kernel: 16x8 pixel tile at (tx,ty)

struct BinsK { const unsigned int *offs; const unsigned int *list; int tiles_x, tile; };

void launch_march_full(int mode, bool ert, const CamK &cam, const VolK &vol, const TfK &tf, float *image,
                       long long pitch_f, cudaStream_t st);
void launch_march_bricks(int mode, bool wide, const CamK &cam, const VolK &vol, const TfK &tf, const BrickK *bricks,
                         const WorkK *work, int n_work, float *arena, cudaStream_t st);
void launch_composite(int mode, const CamK &cam, const BrickK *bricks, BinsK bins, const float *arena, float *image,
                      long long pitch_f, cudaStream_t st);
void launch_chain_init(int mode, int W, int H, float *image, long long pitch_f, cudaStream_t st);
void launch_chain_brick(int mode, bool ert, const CamK &cam, const VolK &vol, const TfK &tf, const BrickK &brick,
                        float *image, long long pitch_f, cudaStream_t st);
void launch_chain_finish(int W, int H, float *image, long long pitch_f, cudaStream_t st);

// ---------------------------------------------------------------- tile-wave ray casting (vr_tiles.cu)
// The volume is cut into staging tiles of TX x TY x TZ ownership cells (a finer brick grid, C.7).
// A persistent kernel stages one tile at a time in shared memory and marches every ray segment
// that crosses it; tiles are taken front to back (level = per-axis tile distance from the eye
// tile) and a tile starts once its <= 3 face neighbours towards the eye are complete, so the ray
// state carried in the image sees its samples in k order (exact C.5 / ERT).
struct TileWork {                // one entry of the per-frame work list (level-major)
    int x0, y0, x1, y1;          // conservative screen rectangle, [x0,x1) x [y0,y1); empty => no work
    unsigned short b[3];         // tile coordinates
    unsigned short flags;
};

struct TilePlanK {
    int nt[3];                   // tiles per axis
    int T[3];                    // tile edge per axis
    int persp;                   // 1: pure perspective (ou = ov = 0); 0: pure orthographic (du = dv = 0)
    int e[3];                    // perspective: tile index of the eye, floor(floor(o0 - 0.5) / T), unclamped
    int sgn[3];                  // orthographic: sign of d0 per axis
    int lvl0[3];                 // per-axis minimum raw level (subtracted so that levels start at 0)
    int n_tiles, n_levels;
};

__host__ __device__ inline int tile_axis_level(const TilePlanK &P, int a, int b)
{
    if (P.persp) return (b > P.e[a] ? b - P.e[a] : P.e[a] - b) - P.lvl0[a];
    return P.sgn[a] > 0 ? b : P.sgn[a] < 0 ? P.nt[a] - 1 - b : 0;
}
// tile coordinate of the face neighbour towards the eye on axis a, or -1
__host__ __device__ inline int tile_axis_pred(const TilePlanK &P, int a, int b)
{
    int p;
    if (P.persp) p = b > P.e[a] ? b - 1 : b < P.e[a] ? b + 1 : -1;
    else p = P.sgn[a] > 0 ? b - 1 : P.sgn[a] < 0 ? b + 1 : -1;
    return (p < 0 || p >= P.nt[a]) ? -1 : p;
}

enum { VR_TILE_32 = 1, VR_TILE_32x32x16 = 2, VR_TILE_32x16x16 = 3, VR_TILE_16 = 4, VR_TILE_KINDS = 5 };
void tile_dims(int kind, int T[3]);
// ctrl: [0] pop counter, [1 .. n_levels] per-level fill cursors (zeroed before each frame)
void launch_tile_plan(const CamK &cam, const TilePlanK &P, const VolK &vol, const unsigned int *lvl_off,
                      unsigned int *ctrl, TileWork *work, cudaStream_t st);
vr_status launch_tile_march(int kind, int mode, bool ert, const CamK &cam, const TilePlanK &P, const VolK &vol,
                            const TfK &tf, const TileWork *work, unsigned int *ctrl, unsigned int *done,
                            unsigned int serial, float *image, long long pitch_f, int sm_count, cudaStream_t st);


// ---------------------------------------------------------------- beam-slab ray casting (vr_beam.cu)
// One CTA per 16x16-pixel beam, ray state in registers, the beam's voxel box staged slab by slab in
// shared memory by TMA (double buffered).  *applied = false: camera / volume outside what the path
// handles (very wide beams, boxes larger than shared memory) — nothing was enqueued.
vr_status launch_beam(int mode, bool ert, const CamK &cam, const VolK &vol, const TfK &tf, unsigned int *overflow_dev,
                      float *image, long long pitch_f, cudaStream_t st, bool *applied);


// ---------------------------------------------------------------- sheared-plane beam ray casting (vr_shear.cu)
// Same beams, but every data plane of a slab is staged as its own rectangle at its own origin by 4-byte
// cp.async into a bank-conflict-aware layout.  *applied = false: nothing was enqueued.
struct ShearPlanCache;                       // per-handle cache of the per-frame host plans (camera -> plan)
ShearPlanCache *shear_cache_create();
void shear_cache_destroy(ShearPlanCache *c);
vr_status launch_shear(int mode, bool ert, bool sparse_direct, const CamK &cam, const VolK &vol, const TfK &tf,
                       unsigned int *overflow_dev, ShearPlanCache *cache, float *image, long long pitch_f,
                       cudaStream_t st, bool *applied);

}  // namespace vr
