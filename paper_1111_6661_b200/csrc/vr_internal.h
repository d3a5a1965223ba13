// vr_internal.h — host-side handle, error plumbing and kernel launcher declarations.
#pragma once
#ifndef VR_SIMT_HOST               // tests/simt/simt_host.h (force-included by the host emulation build) stands in
#include <cuda_runtime.h>
#endif
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/vr.h"
#include "vr_lanemap.h"
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

// Every kernel launch of the library goes through here (one place for the launch syntax; the host emulation
// build of the tests runs the same kernel function thread by thread instead).
template <typename... P, typename... A>
inline void vr_launch(void (*kernel)(P...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, A &&...args)
{
#ifdef VR_SIMT_HOST
    (void)st;
    ::simt::launch(grid, block, smem, [&] { kernel(static_cast<P>(args)...); });
#else
    kernel<<<grid, block, smem, st>>>(static_cast<P>(args)...);
#endif
}

// event counters for the host emulation of the tests (nothing in the product build)
#ifdef VR_SIMT_HOST
#define VR_TEST_COUNT(i) (++::simt::g_counters[i])
#else
#define VR_TEST_COUNT(i) ((void)0)
#endif
// memory-traffic model of the emulation (tests/simt/traffic_model.py): addresses of the four row pointers of a sample
#ifdef VR_SIMT_HOST
#define VR_TRACE_CORNER_LOADS(sampled, loads, base, p0, p1, p2, p3) \
    do { if (::simt::g_trace) ::simt::trace_corner_loads(sampled, loads, base, p0, p1, p2, p3); } while (0)
#else
#define VR_TRACE_CORNER_LOADS(sampled, loads, base, p0, p1, p2, p3) ((void)0)
#endif
enum { VR_CNT_LEAP_CELL = 0, VR_CNT_LEAP_BLOCK = 1, VR_CNT_LEAP_REJECTED = 2, VR_CNT_LAG_WAIT = 3, VR_CNT_FRAG_OUTSIDE = 4,
       VR_CNT_FRAG_NO_BRICK = 5 };

// dynamic shared memory of the CTA as an array of T
#ifdef VR_SIMT_HOST
#define VR_DYN_SHARED(T, name) T *name = reinterpret_cast<T *>(::simt::g_dyn_smem)
#else
#define VR_DYN_SHARED(T, name) extern __shared__ T name[]
#endif

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

// ---------------------------------------------------------------- mean / stddev / median (vr_stats.cu)
constexpr int kStatMaxGrid = 1024;            // CTAs per pass launch (one double slot per CTA)
struct StatScratch {
    unsigned int klo, khi;                    // key interval that holds the median (pass 0: key of min / max)
    unsigned int shift, done;                 // bin width 2^shift keys of the next select pass; 1: klo is the median
    unsigned long long n_finite, n_nonfinite, rank;
    double mean, m2, stddev;
    unsigned long long hist[256];
    unsigned long long part_n[kStatMaxGrid];
    double part[kStatMaxGrid], part_c[kStatMaxGrid];
};

void launch_stat_reset(StatScratch *s, cudaStream_t st);
// pass 0: count, sum, key range; 1: squared deviations + select; 2..4: select
void launch_stat_pass_flat(int pass, const float *v, unsigned long long n, StatScratch *s, int grid, cudaStream_t st);
void launch_stat_pass_box(int pass, BoxK b, StatScratch *s, int grid, cudaStream_t st);
void launch_stat_step(StatScratch *s, int pass, cudaStream_t st);       // one thread, after pass `pass`
void launch_stat_finish(const StatScratch *s, vr_statistics_result *out, cudaStream_t st);

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

// force_wide: 64-bit element offsets even where 32 bits would do (VR_OPT_FORCE_WIDE, for the tests)
void launch_march_full(int mode, bool ert, bool force_wide, const CamK &cam, const VolK &vol, const TfK &tf, float *image,
                       long long pitch_f, cudaStream_t st);
void launch_march_bricks(int mode, bool wide, const CamK &cam, const VolK &vol, const TfK &tf, const BrickK *bricks,
                         const WorkK *work, int n_work, float *arena, cudaStream_t st);
void launch_composite(int mode, const CamK &cam, const BrickK *bricks, BinsK bins, const float *arena, float *image,
                      long long pitch_f, cudaStream_t st);
void launch_chain_init(int mode, int W, int H, float *image, long long pitch_f, cudaStream_t st);
void launch_chain_brick(int mode, bool ert, bool force_wide, const CamK &cam, const VolK &vol, const TfK &tf,
                        const BrickK &brick, float *image, long long pitch_f, cudaStream_t st);
void launch_chain_finish(int W, int H, float *image, long long pitch_f, cudaStream_t st);

// ---------------------------------------------------------------- 8-bit frame for delivery (vr_encode.cu)
struct EncodeK { float bg[3]; float scale, bias; };
void launch_encode_rgba8(int mode, const float *img, long long pitch_f, int W, int H, const EncodeK &P, unsigned int *out,
                         long long out_pitch_w, cudaStream_t st);

// ---------------------------------------------------------------- lane-mapped ray casting (vr_lanes.cu)
// A resident volume as the kernel addresses it: one axis has element stride 1 (`fast`: 0 = the caller's
// x-fastest array, 2 = the library's z-fastest copy); sa, sb are the element strides of the other two
// axes in ascending axis order (fast 0: y, z; fast 2: x, y).
struct LaneVolK {
    const float *base;
    long long sa, sb;
    int nx, ny, nz;
};

// exact empty-space skipping (vr_macro.cu): one byte per macrocell of kMacroEdge^3 base indices; bit 0 = every
// sample based in the cell has opacity exactly 0 under the current transfer function, bit 1 = so has every cell
// of its block of 8 x 8 x 8 cells; n_skip = how many cells have bit 0 set
constexpr int kMacroEdge = 8;
struct MacroK {
    const unsigned char *flag;                // nullptr: no skipping
    const unsigned long long *n_skip;         // device counter written by the flag kernel
    unsigned long long min_skip;              // skipping is used iff *n_skip >= min_skip (decided on the device)
    int cx, cy, cz;                           // cells per axis
};

void launch_macro_minmax(const float *v, int nx, int ny, int nz, const MacroK &m, float2 *mm, cudaStream_t st);
void launch_macro_flags(const float2 *mm, long long n_cells, const TfK &tf, unsigned char *flag, unsigned long long *n_skip,
                        int grid, cudaStream_t st);
void launch_macro_blocks(unsigned char *flag, const MacroK &m, int grid, cudaStream_t st);

// value range of a brick slot as order-preserving keys (key(f) = bits ^ (sign ? ~0 : 0x80000000)); bad: non-finite seen
struct BrickRangeK { unsigned int enc_min, enc_max, bad, pad; };
void launch_brick_range_init(BrickRangeK *r, unsigned long long n, cudaStream_t st);
void launch_brick_range(const float *v, unsigned long long n, BrickRangeK *r, int grid, cudaStream_t st);

// sort-last partials written by the lane-mapped kernel: plan-ordered brick table, brick-grid -> plan index (-1:
// culled), fragment arena, brick edge and grid
struct PartK {
    const BrickK *bricks;
    const int *lut;
    float *arena;
    int B, nbx, nby;
};

// part != nullptr: write per-(ray, owner brick) fragments instead of pixels (no ERT, C.7).  Returns true iff the
// launch used 16-byte row loads.
bool launch_rows(int mode, bool ert, const CamK &cam, const LaneVolK &vol, int fast, const TfK &tf, const LaneMapK &map,
                 const MacroK &macro, const PartK *part, bool force_wide, bool quad_loads, int rows, float *image,
                 long long pitch_f, cudaStream_t st);
void launch_fragment_init(int mode, float *arena, unsigned long long n_frag, int grid, cudaStream_t st);
void launch_transpose_xz(const float *in, float *out, int nx, int ny, int nz, cudaStream_t st);

}  // namespace vr
