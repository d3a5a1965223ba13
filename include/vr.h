/*
 * vr.h — C ABI of libvr.so: B200-native bricked volume ray-casting of float32 spectral
 * cubes plus the data passes the paper names: min/max + histogram, mean / standard deviation /
 * median, and the 8-bit frame a thin client displays.
 *
 * What is computed.  The paper names the operations — interactive volume rendering of
 * larger-than-memory spectral cubes by sub-cube partitioning and a gather of partial images
 * and the "simple data analysis tasks" minimum/maximum
 * and histogram, the "global view" tasks median and standard deviation (L66),
 * a viewer that only displays results (L48, L70) — but gives no formulae.  The arithmetic is
 * therefore the set of readings C.0-C.8 of SURVEY.md §8(c) and C.13-C.14, S33-S41 of DESIGN.md §3.
 * Every entry point below cites the passage and the reading it implements.
 *
 * Conventions common to all calls
 *   - Plain C, no CUDA or torch types: a stream is passed as `void*` holding a cudaStream_t
 *     (NULL = the legacy default stream).  Pointers are marked HOST or DEVICE.
 *   - Every call returns vr_status; nothing throws, aborts or prints.  vr_last_error() gives a
 *     thread-local message for the last failing call on this thread.
 *   - Every struct starts with `struct_size` = sizeof(that struct) as the caller compiled it.
 *   - vr_render / vr_minmax_histogram / vr_statistics / vr_encode_rgba8 ENQUEUE work on `stream` and
 *     return; results are valid once `stream` reaches the point after the call.  With device-resident volumes and
 *     device outputs there is no host synchronisation inside.  Library-internal copy streams
 *     are joined to `stream` by events.
 *   - One host thread and one stream per handle at a time (the handle's device table, scratch and
 *     staging buffers are single instances; order calls on different streams yourself).  Different
 *     handles may be used concurrently.
 *   - There is no CPU fallback: without a CUDA device every compute call fails with VR_ERR_CUDA.
 */
#ifndef VR_H_
#define VR_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define VR_API __attribute__((visibility("default")))
#else
#define VR_API
#endif

typedef enum {
    VR_OK = 0,
    VR_ERR_INVALID_ARG = 1,   /* NULL, bad size/enum, non-finite or out-of-range value */
    VR_ERR_UNSUPPORTED = 2,   /* valid request this build cannot serve (message says why) */
    VR_ERR_OUT_OF_MEMORY = 3, /* host or device allocation failed */
    VR_ERR_CUDA = 4,          /* CUDA runtime error (message carries cudaGetErrorString) */
    VR_ERR_NOT_READY = 5      /* e.g. EA render before vr_set_transfer_function */
} vr_status;

enum { VR_LINEAR = 0,          /* float32[nz][ny][nx], x fastest (FITS order; z = spectral axis) */
       VR_BRICKED_HALO1 = 1 }; /* brick-major: brick id = bx + nbx*(by + nby*bz); each brick is
                                  float32[B+1][B+1][B+1] holding voxels [B*b, B*b+B] per axis clamped
                                  to the volume (one-voxel high-side halo, C.7) */
enum { VR_DEVICE = 0, VR_HOST_PINNED = 1 };
enum { VR_EA = 0,              /* emission-absorption, premultiplied RGBA, 4 channels */
       VR_MIP = 1 };           /* maximum intensity projection, 1 channel */
enum { VR_SORT_LAST = 1u };    /* vr_camera.flags: render per-brick partial images and merge them
                                  with the sort-last compositor even when a single march would do */
/* vr_camera.flags: progressive pass — render only the pixels (i,j) with i % stride == phase_x and j % stride ==
   phase_y, IN PLACE in the full-resolution image; stride 1..255, phases below the stride (see vr_render) */
#define VR_SUBSAMPLE(stride, phase_x, phase_y) \
    (((uint32_t)(stride) << 8) | ((uint32_t)(phase_x) << 16) | ((uint32_t)(phase_y) << 24))

typedef struct vr_volume vr_volume; /* opaque; created and destroyed only by the library */

/* ------------------------------------------------------------------------------------------
 * vr_create_volume — brick decomposition + residency (
 * PAPER.md:L24, L66 "partitioning the cube into ... sub-cubes, with a different data loading
 * for each"; reading C.7 for the brick grid).
 *
 *   nx,ny,nz   voxels per axis, each >= 2.
 *   brick      brick edge B in voxels; 0 = one brick = the whole cube.  The grid is
 *              nb_a = ceil(n_a / B); at most 65535 bricks per axis.
 *   layout     VR_LINEAR or VR_BRICKED_HALO1 (requires brick > 0).
 *   location   VR_DEVICE: `data` is a DEVICE pointer, 16-byte aligned, used in place.
 *              VR_HOST_PINNED: `data` is a HOST pointer to page-locked memory (checked with
 *              cudaPointerGetAttributes; pageable memory => VR_ERR_INVALID_ARG).  The library
 *              then owns a device-side copy policy:
 *                - resident_bytes == 0 or >= the volume's bytes: the whole volume is mirrored
 *                  on the device on first use (uploaded once on the copy streams);
 *                - otherwise (out of core; "multiple execution
 *                  queues (or streams) to overlap GPU computation with data I/O"): a pool of
 *                  floor(resident_bytes / brick_bytes) brick slots; bricks are streamed per
 *                  frame in view order on n_copy_streams streams.  Requires VR_BRICKED_HALO1.
 *   data       BORROWED until vr_destroy_volume; never written by the library; its contents must
 *              not change while the handle exists (the library may hold derived copies).
 *   n_copy_streams  1..8 (0 => 4).  Only used for VR_HOST_PINNED.
 * Errors: VR_ERR_INVALID_ARG (NULL, dims < 2, bad enums, brick grid too large, pageable host
 * memory, misaligned device pointer), VR_ERR_OUT_OF_MEMORY, VR_ERR_CUDA.
 * ------------------------------------------------------------------------------------------ */
typedef struct {
    uint32_t struct_size;
    uint32_t nx, ny, nz;
    uint32_t brick;
    uint32_t layout;
    uint32_t location;
    uint32_t n_copy_streams;
    const float *data;          /* DEVICE or pinned HOST, see location */
    uint64_t resident_bytes;
} vr_volume_desc;

VR_API vr_status vr_create_volume(const vr_volume_desc *desc, vr_volume **out);

/* Synchronises the library's own streams, frees everything the handle owns.  The caller's
 * data, image and summary buffers are untouched.  NULL is accepted. */
VR_API vr_status vr_destroy_volume(vr_volume *vol);

/* ------------------------------------------------------------------------------------------
 * vr_set_transfer_function — SURVEY.md row A3; reading C.4 (S8-S11).
 *   rgba   HOST, 256*4 floats, copied before return.  Entry i sits at u = i/255; rgb is
 *          non-premultiplied; alpha is the per-SAMPLE opacity at the step the caller will
 *          render with (no opacity correction inside the library).  Every value must be
 *          finite and in [0,1].
 *   vmin,vmax  scalar range mapped to u in [0,1]: scale = 1/(vmax-vmin), bias = -vmin*scale,
 *          both rounded to float32 once (C.4).  Must be finite with vmax > vmin.  Normally
 *          the vmin/vmax produced by vr_minmax_histogram.
 * Host work only: the table reaches the device on the stream of the next vr_render that needs it, so renders
 * already enqueued keep the table they were launched with.  A handle is used on ONE stream at a time: calls
 * on different streams must be ordered by the caller (event or synchronisation), because the handle's device
 * table, summary scratch and staging buffers are single instances.
 * Errors: VR_ERR_INVALID_ARG.
 * ------------------------------------------------------------------------------------------ */
VR_API vr_status vr_set_transfer_function(vr_volume *vol, const float *rgba, float vmin, float vmax);

/* ------------------------------------------------------------------------------------------
 * vr_render — SURVEY.md rows A4-A10: per-frame brick ordering, ray generation and entry/exit
 * (C.1, C.2), trilinear sampling (C.3), classification (C.4), front-to-back compositing with
 * early ray termination (C.5), MIP (C.6), per-brick partial images and the sort-last
 * compositor (C.7).  This is the kernel the paper calls "the GPU part" of its case study
 * and the gather of partial results.
 *
 * Camera (C.1):  origin(i,j) = o0 + (i+.5)*ou + (j+.5)*ov
 *                dir(i,j)    = normalize(d0 + (i+.5)*du + (j+.5)*dv)
 *   in voxel units of the box [0,nx]x[0,ny]x[0,nz]; voxel (ix,iy,iz) has its value at its
 *   centre (ix+.5, iy+.5, iz+.5); reconstruction is clamp-to-edge (C.0).  Perspective:
 *   ou = ov = 0.  Orthographic: du = dv = 0.
 *   step       sample spacing in voxels along the unit direction, > 0.  Samples sit on one
 *              lattice per ray anchored at the VOLUME entry: t_k = t_enter + (k+.5)*step.
 *   ert_alpha  0 = off; otherwise in (0,1): a ray stops after the sample at which its
 *              transmittance T <= 1 - ert_alpha (that sample included).  EA only.
 *   flags      VR_SORT_LAST: per-brick partial images + compositor.  Needs brick > 0, a pure
 *              perspective or pure orthographic camera, and ert_alpha == 0 (early termination
 *              is not defined for independent partials, reading S15) => else VR_ERR_UNSUPPORTED.
 *              VR_SUBSAMPLE(s, px, py): a progressive pass (the "interactive" of
 *              PAPER.md:L34): only the pixels with i % s == px and j % s == py are rendered, into their own
 *              places of the full-resolution image; every other pixel of the buffer is left untouched.  A rendered
 *              pixel is bit-identical to the same pixel of a full render (the ray of pixel (i,j) is C.1's, whatever
 *              the pass), so a viewer can show the s = 4 lattice while the camera moves (1/16 of the rays) and fill
 *              in the remaining phases when it rests: after all s^2 phases the image IS the full render.  Single
 *              march of a resident VR_LINEAR volume into a DEVICE image only (else VR_ERR_UNSUPPORTED).
 * Image: `pixels` is caller-owned, DEVICE (location VR_DEVICE) or pinned HOST (VR_HOST_PINNED;
 *   the library renders into an internal device image and enqueues the device-to-host copy on
 *   `stream`).  Row j = 0 is the v-minimum row; row_pitch_bytes >= width*channels*4 and a
 *   multiple of 16 (EA) / 4 (MIP); 0 means tightly packed.
 *   VR_EA : channels = 4: premultiplied (C.r, C.g, C.b, 1-T); a miss is (0,0,0,0).
 *   VR_MIP: channels = 1: max of the interpolated samples in data units; no sample = -INFINITY.
 * Out-of-core volumes are rendered brick by brick in view order with the ray state carried in
 * the image (so ERT stays exact); uploads run on the copy streams and overlap rendering.  Once the
 * value ranges gathered by the first vr_minmax_histogram of a brick-major volume have reached the
 * host, an EA render drops every brick whose whole range maps to opacity exactly 0 before it is
 * uploaded or marched (exact: such samples change nothing; VR_OPT_EMPTY_SKIP = 0 turns it off).
 * Errors: VR_ERR_INVALID_ARG (NULL, width/height 0, step <= 0 or non-finite, ert_alpha not in
 * [0,1), channels not matching mode, bad pitch), VR_ERR_NOT_READY (EA before a transfer
 * function was set), VR_ERR_UNSUPPORTED, VR_ERR_OUT_OF_MEMORY, VR_ERR_CUDA.
 * ------------------------------------------------------------------------------------------ */
typedef struct {
    uint32_t struct_size, width, height;
    float o0[3], ou[3], ov[3];
    float d0[3], du[3], dv[3];
    float step;
    float ert_alpha;
    uint32_t flags;
} vr_camera;

typedef struct {
    uint32_t struct_size;
    uint32_t channels;          /* 4 for VR_EA, 1 for VR_MIP */
    uint32_t location;          /* VR_DEVICE or VR_HOST_PINNED */
    uint32_t reserved;
    float *pixels;
    uint64_t row_pitch_bytes;
} vr_image;

VR_API vr_status vr_render(vr_volume *vol, const vr_camera *cam, int mode, const vr_image *image, void *stream);

/* ------------------------------------------------------------------------------------------
 * vr_minmax_histogram — SURVEY.md rows A1, A2; reading C.8 (S22-S26).
 * ("calculating a histogram or computing data minimum/maximum"), L66 ("a single-pass
 * accumulative operation like calculating the data minimum and maximum").
 *
 *   vmin, vmax   min and max over the voxels with isfinite(v); n_nonfinite counts the rest.
 *   histogram    lo,hi = range[0],range[1] if range != NULL else (vmin,vmax);
 *                scale_h = (float)nbins / (hi - lo)  (0 if hi == lo); for each finite v:
 *                v < lo => n_below; v > hi => n_above; else b = (int)((v - lo) * scale_h),
 *                clamped to nbins-1; counts[b]++.  All float32, subtract then multiply, no FMA.
 *                Invariant: sum(counts) + n_below + n_above + n_nonfinite == nx*ny*nz.
 *                Halo voxels of a bricked layout are not counted.
 *   nbins        1..4096.
 *   range        HOST pointer to two floats (finite, range[1] >= range[0]) or NULL.  With NULL
 *                the cube is read twice (8 B/voxel), else once for min/max and histogram together.
 *   out          vr_summary followed by nbins uint64 counts: DEVICE memory (out_location
 *                VR_DEVICE) or pinned HOST (VR_HOST_PINNED), 8-byte aligned,
 *                VR_SUMMARY_BYTES(nbins) bytes, written on `stream`.
 * Out-of-core volumes are streamed through the brick pool (both passes ride the streamer).
 * Errors: VR_ERR_INVALID_ARG, VR_ERR_OUT_OF_MEMORY, VR_ERR_CUDA.
 * ------------------------------------------------------------------------------------------ */
typedef struct {
    float vmin, vmax;
    uint64_t n_nonfinite, n_below, n_above;
    uint64_t counts[1];         /* nbins entries */
} vr_summary;
#define VR_SUMMARY_BYTES(nbins) (32u + 8u * (uint64_t)(nbins))

VR_API vr_status vr_minmax_histogram(vr_volume *vol, uint32_t nbins, const float *range, vr_summary *out,
                                     uint32_t out_location, void *stream);

/* ------------------------------------------------------------------------------------------
 * vr_statistics — the multi-pass "global view" statistics of the whole cube (
 * PAPER.md:L66 "global view data analysis tasks ... [like] median and standard deviation", which need
 * every voxel and several passes over the data; readings S35-S37 of DESIGN.md §3).  Over the voxels
 * with isfinite(v) (n_finite of them; n_nonfinite counts the rest; halo voxels of a bricked layout are
 * not counted):
 *   mean     sum(v) / n_finite, accumulated in float64 (compensated; S35).
 *   stddev   POPULATION standard deviation sqrt(sum((v - mean)^2) / n_finite), second pass, float64 (S36).
 *   median   the LOWER median: the voxel value of rank floor((n_finite - 1) / 2) (0-based) in ascending
 *            IEEE totalOrder (-0 before +0).  A data value, found exactly by a 4-pass radix select on the
 *            order-preserving bit pattern (S37); no sorting, no approximation.
 *   n_finite == 0: mean, stddev and median are NaN.
 * Five streams of the cube (4 B/voxel each) enqueued on `stream`, nothing read back in between; float64
 * sums are deterministic for a given device (fixed reduction order), and equal to any other correct
 * summation within a few units of 1e-16 * mean(|v|).  Out-of-core volumes ride the brick streamer.
 *   out   DEVICE (out_location VR_DEVICE) or pinned HOST (VR_HOST_PINNED), 8-byte aligned.
 * Errors: VR_ERR_INVALID_ARG, VR_ERR_OUT_OF_MEMORY, VR_ERR_CUDA.
 * ------------------------------------------------------------------------------------------ */
typedef struct {
    uint64_t n_finite, n_nonfinite;
    double mean, stddev;
    float median;
    uint32_t reserved;
} vr_statistics_result;

VR_API vr_status vr_statistics(vr_volume *vol, vr_statistics_result *out, uint32_t out_location, void *stream);

/* ------------------------------------------------------------------------------------------
 * vr_encode_rgba8 — the 8-bit frame a thin client displays ("remote
 * ... viewer ... is only responsible for ... result display", L70; reading S40 / C.14).  No graphics API
 * is involved: the frame is a byte buffer.
 *   src        a rendered image of this library: DEVICE float32, VR_EA (4 channels, premultiplied C and
 *              opacity A) or VR_MIP (1 channel); src->row_pitch_bytes as in vr_render.
 *   VR_EA      x_c = fmaf(1 - A, background_c, C_c), clamped to [0,1] (NaN -> 0);
 *              byte_c = round-half-even(x_c * 255); alpha byte 255.
 *   VR_MIP     u = sat(fmaf(m, scale, bias)) with scale = 1/(vmax - vmin), bias = -vmin * scale (float32, as
 *              C.4); byte = round-half-even(u * 255) in r, g and b; a miss (-INFINITY) gives 0; alpha 255.
 *   out        width*height RGBA8 pixels, rows of out_pitch_bytes (>= 4*width, multiple of 4; 0 = tight), DEVICE
 *              (out_location VR_DEVICE) or pinned HOST (VR_HOST_PINNED: encoded into an internal device buffer
 *              and copied on `stream`), 4-byte aligned.
 * Enqueued on `stream` after whatever produced `src` there.
 * Errors: VR_ERR_INVALID_ARG (NULL, bad sizes / mode / pitch, non-finite background, vmax <= vmin for VR_MIP),
 * VR_ERR_OUT_OF_MEMORY, VR_ERR_CUDA.
 * ------------------------------------------------------------------------------------------ */
typedef struct {
    uint32_t struct_size;
    uint32_t width, height;
    uint32_t mode;               /* VR_EA or VR_MIP: what `src` holds */
    float background[3];         /* VR_EA: opaque background colour, each in [0,1] */
    float vmin, vmax;            /* VR_MIP: scalar range of the grey ramp */
} vr_encode_desc;

VR_API vr_status vr_encode_rgba8(vr_volume *vol, const vr_encode_desc *desc, const vr_image *src, uint8_t *out,
                                 uint64_t out_pitch_bytes, uint32_t out_location, void *stream);

/* ------------------------------------------------------------------------------------------
 * vr_get_stats — counters of the last vr_render / vr_minmax_histogram on this handle
 * (SURVEY.md §5 "metrics"): host-side values only, no synchronisation.
 * ------------------------------------------------------------------------------------------ */
typedef struct {
    uint32_t struct_size;
    uint32_t n_bricks;              /* bricks in the grid */
    uint32_t bricks_drawn;          /* bricks that produced work in the last render */
    uint32_t bricks_culled;         /* bricks outside the view (empty screen rectangle) */
    uint32_t path;                  /* last render: 0 none, 1 ray-major tiles, 2 sort-last, 3 brick chain, 7 lane-mapped rows */
    uint32_t kernel_launches;       /* library kernels launched by the last call */
    uint64_t fragments;             /* (brick,pixel) partial fragments written (sort-last) */
    uint64_t h2d_bytes;             /* host-to-device bytes enqueued by the last call */
    uint64_t d2h_bytes;             /* device-to-host bytes enqueued by the last call */
    uint64_t total_kernel_launches; /* since vr_create_volume */
    uint64_t resident_bytes;        /* device bytes owned by the handle */
    uint32_t zfast_copy;            /* 1: the handle holds a z-fastest copy of the volume (VR_OPT_ZFAST_COPY) */
    uint32_t skip_variant;          /* 1: the last render launched the empty-space-skipping kernel variant */
    uint32_t bricks_empty;          /* bricks of a brick-major volume dropped by the last render because their whole value
                                       range has opacity 0 (neither uploaded nor marched) */
    uint32_t quad_launches;         /* lane-mapped launches of the last render that used 16-byte row loads (VR_OPT_ROW_LOADS) */
    uint64_t macro_cells;           /* macrocells of the skipping grid (0: none built) */
    uint64_t empty_cells;           /* cells whose samples all have opacity 0 under the current transfer function,
                                       as of the last flag pass that has COMPLETED on its stream */
} vr_stats;

VR_API vr_status vr_get_stats(vr_volume *vol, vr_stats *stats);

/* ------------------------------------------------------------------------------------------
 * vr_set_option — implementation choices that never change results (all paths evaluate the same
 * canonical arithmetic, C.1-C.7, and are bit-identical); used by the parity tests and by bench.py.
 *   VR_OPT_RENDER_PATH  how a resident VR_LINEAR volume is marched when VR_SORT_LAST is not requested:
 *                       0 = auto: lane-mapped rows (one thread per ray; warps formed per frame so that their
 *                       samples run along the memory-fast axis), 1 = ray-major (fixed 8x4-pixel warps).
 *   VR_OPT_ZFAST_COPY   1 (default): the first view with rays that travel mostly along x makes the library
 *                       allocate a z-fastest copy of a resident VR_LINEAR volume (same size as the volume,
 *                       transposed once on the render's stream) when the device has that much free memory,
 *                       and such rays are rendered from it; 0: never (they are rendered from the x-fastest
 *                       array, slower).  The voxel data must not change while a handle holds a copy.
 *   VR_OPT_LANE_LAG     lane-mapped path: a ray more than this many voxel planes (along the view's principal
 *                       axis) ahead of the slowest ray of its warp waits; 0 = off; default 1.
 *   VR_OPT_EMPTY_SKIP   1 (default): exact transfer-function-aware empty-space skipping on the lane-mapped path
 *                       (SURVEY.md §8(f) #2).  When the table has an interval of opacity exactly 0, the library
 *                       keeps min / max per macrocell of 8^3 voxels (one extra read of the volume, once per
 *                       handle) and one byte per cell and transfer function; a sample based in a cell whose
 *                       whole value range maps to opacity 0 is not read (compositing it would change nothing,
 *                       C.5), so images are bit-identical.  Used only while at least 1/64 of the cells are
 *                       empty (decided on the device, no read-back).  0: never.
 *   VR_OPT_ROW_LOADS    lane-mapped path: how the two voxels (u, u+1) a sample reads from each of its four rows are
 *                       fetched.  0: two 4-byte loads.  1: ONE aligned 16-byte load of the quad that holds u, plus a
 *                       4-byte load of u+1 for the lanes whose u ends its quad — fewer cache lines touched per sample,
 *                       more select instructions.  2 (default): 1 for the launches whose rays can enter the volume
 *                       through a face perpendicular to the memory-fast axis (oblique views: bound by lines touched),
 *                       0 for the others (bound by instruction issue); see profiles/r2_lane_traffic_model.md.  Quads
 *                       need a memory-fast dimension that is a multiple of 4 and are not used by the empty-space
 *                       skipping variant.
 *   VR_OPT_TILE_SHEAR   lane-mapped path: 1 (default): every tile of 32 x 64 pixels shears its rows by its own slope (under
 *                       perspective the slope that keeps a warp on one voxel row changes several-fold across the image);
 *                       0: one slope per frame, taken at the image centre.
 *   VR_OPT_FORCE_WIDE   1: the render kernels form 64-bit voxel offsets even for volumes of fewer than 2^32
 *                       voxels (the code the largest volumes run; lets the tests cover it at small size).  Default 0.
 * Errors: VR_ERR_INVALID_ARG (NULL handle, unknown option, value out of range).
 * ------------------------------------------------------------------------------------------ */
enum { VR_OPT_RENDER_PATH = 1, VR_OPT_ZFAST_COPY = 2, VR_OPT_LANE_LAG = 3, VR_OPT_EMPTY_SKIP = 4, VR_OPT_FORCE_WIDE = 5,
       VR_OPT_ROW_LOADS = 6, VR_OPT_TILE_SHEAR = 7 };
VR_API vr_status vr_set_option(vr_volume *vol, uint32_t option, int64_t value);

/* Thread-local message of the last failing call on this thread ("" if none). */
VR_API const char *vr_last_error(void);

/* Library version and the CUDA architecture it was built for, e.g. "vr-b200 0.1 sm_100a". */
VR_API const char *vr_version(void);

#ifdef __cplusplus
}
#endif
#endif /* VR_H_ */
