// vr_api.cu — the C ABI of include/vr.h and the host runtime behind it: brick table and
// residency, per-frame brick ordering / culling / screen rectangles (A4),
// the out-of-core brick streamer (A5) and launch planning for the kernels of vr_raycast.cu and
// vr_reduce.cu.  No host synchronisation on the in-HBM paths; everything is enqueued on the
// caller's stream, library copy streams are joined to it by events.
#include <algorithm>
#include <cfloat>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>

#include "vr_internal.h"
#include "vr_plan.h"

namespace vr {

// ------------------------------------------------------------------ error plumbing
static thread_local char g_err[512] = "";

void set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

vr_status cuda_fail(cudaError_t e, const char *what)
{
    set_error("CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
    if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return VR_ERR_OUT_OF_MEMORY; }
    return VR_ERR_CUDA;
}

// ------------------------------------------------------------------ small helpers
template <typename T>
struct DevBuf {                       // grow-only device buffer
    T *p = nullptr;
    size_t cap = 0;
    vr_status reserve(size_t n)
    {
        if (n <= cap) return VR_OK;
        if (p) { VR_CUDA(cudaFree(p)); p = nullptr; cap = 0; }
        size_t want = n + n / 4;
        VR_CUDA(cudaMalloc(&p, want * sizeof(T)));
        cap = want;
        return VR_OK;
    }
    void release() { if (p) cudaFree(p); p = nullptr; cap = 0; }
};

struct Staging {                      // one slot of the per-frame table ring (pinned host + device)
    unsigned char *h = nullptr, *d = nullptr;
    size_t cap = 0;
    cudaEvent_t done = nullptr;       // recorded after the last kernel that reads d
    bool in_flight = false;
};

constexpr int kStagingRing = 4;
constexpr int kMaxCopyStreams = 8;

}  // namespace vr

using namespace vr;

struct vr_volume {
    vr_volume_desc desc;
    int device = 0, sm_count = 0;
    uint32_t B = 0, E = 0;                    // brick edge; E = B + 1 (bricked layouts)
    uint32_t nb[3] = { 1, 1, 1 };
    uint64_t n_vox = 0, n_bricks = 1, brick_elems = 0, total_elems = 0;
    bool out_of_core = false;

    // device views
    const float *dev_data = nullptr;          // whole volume on the device in desc.layout (borrowed or mirror)
    float *mirror = nullptr;                  // owned copy of a host volume (fully resident case)
    bool mirror_valid = false;
    std::vector<cudaEvent_t> mirror_ev;       // one per copy stream used by the upload

    // out-of-core pool
    float *pool = nullptr;
    uint32_t n_slots = 0, n_fixed = 0, n_ring = 0;
    uint64_t ring_pos = 0, copy_rr = 0;
    std::vector<uint8_t> fixed_loaded;
    std::vector<cudaEvent_t> ev_up, ev_free;  // per slot
    std::vector<uint8_t> slot_used;

    cudaStream_t copy[kMaxCopyStreams] = {};
    int n_copy = 0;

    // transfer function: host copy; uploaded on the stream of the next render that needs it
    float4 *d_tf = nullptr;
    float tf_tab[257 * 4];
    bool tf_set = false, tf_dirty = false, tf_has_zero = false;
    float tf_scale = 0.0f, tf_bias = 0.0f;

    // exact empty-space skipping (vr_macro.cu): macrocell min/max (made once), per-transfer-function flags
    float2 *macro_mm = nullptr;
    unsigned char *macro_flag = nullptr;
    unsigned long long *d_nskip = nullptr, *h_nskip = nullptr;
    cudaEvent_t nskip_ev = nullptr;           // recorded after the count of empty cells was copied to h_nskip
    bool macro_failed = false, macro_flags_dirty = true;
    int mc[3] = { 0, 0, 0 };
    int opt_skip = 1;

    // value range of every brick slot of a brick-major volume, gathered by the first summary pass (device, pinned
    // host copy, event recorded after the copy): lets the chain and sort-last paths drop bricks whose samples all
    // have opacity 0 BEFORE they are uploaded or marched (S38)
    BrickRangeK *d_brick_rng = nullptr, *h_brick_rng = nullptr;
    cudaEvent_t brick_rng_ev = nullptr;
    bool brick_rng_issued = false;

    // scratch
    SummaryScratch *d_sum = nullptr;
    vr_summary *d_sum_out = nullptr;          // staging for host outputs
    StatScratch *d_stat = nullptr;            // vr_statistics (allocated on first use)
    vr_statistics_result *d_stat_out = nullptr;
    DevBuf<float> arena, host_image;
    DevBuf<unsigned int> host_frame;          // vr_encode_rgba8 with a pinned-host output

    // lane-mapped path: the library's z-fastest copy of a resident linear volume (vr_lanes.cu)
    float *zfast = nullptr;
    bool zfast_failed = false;                // allocation refused once: not retried
    cudaEvent_t zfast_ev = nullptr;           // recorded after the transposition
    int opt_path = 0, opt_zcopy = 1, opt_lag = 1, opt_wide = 0, opt_quad = 2, opt_tile_shear = 1;   // vr_set_option
    Staging staging[kStagingRing];
    int staging_next = 0;

    vr_stats stats;
};

namespace vr {

static void free_volume(vr_volume *v)
{
    if (!v) return;
    cudaSetDevice(v->device);
    for (int i = 0; i < v->n_copy; ++i) if (v->copy[i]) { cudaStreamSynchronize(v->copy[i]); cudaStreamDestroy(v->copy[i]); }
    for (auto e : v->mirror_ev) cudaEventDestroy(e);
    for (auto e : v->ev_up) cudaEventDestroy(e);
    for (auto e : v->ev_free) cudaEventDestroy(e);
    for (auto &s : v->staging) {
        if (s.done) { if (s.in_flight) cudaEventSynchronize(s.done); cudaEventDestroy(s.done); }
        if (s.h) cudaFreeHost(s.h);
        if (s.d) cudaFree(s.d);
    }
    if (v->mirror) cudaFree(v->mirror);
    if (v->pool) cudaFree(v->pool);
    if (v->d_tf) cudaFree(v->d_tf);
    if (v->d_sum) cudaFree(v->d_sum);
    if (v->d_sum_out) cudaFree(v->d_sum_out);
    if (v->d_stat) cudaFree(v->d_stat);
    if (v->d_stat_out) cudaFree(v->d_stat_out);
    if (v->zfast) cudaFree(v->zfast);
    if (v->macro_mm) cudaFree(v->macro_mm);
    if (v->macro_flag) cudaFree(v->macro_flag);
    if (v->d_nskip) cudaFree(v->d_nskip);
    if (v->h_nskip) cudaFreeHost(v->h_nskip);
    if (v->nskip_ev) cudaEventDestroy(v->nskip_ev);
    if (v->d_brick_rng) cudaFree(v->d_brick_rng);
    if (v->h_brick_rng) cudaFreeHost(v->h_brick_rng);
    if (v->brick_rng_ev) cudaEventDestroy(v->brick_rng_ev);
    if (v->zfast_ev) cudaEventDestroy(v->zfast_ev);
    v->arena.release();
    v->host_image.release();
    v->host_frame.release();
    delete v;
}

static inline uint64_t brick_id(const vr_volume *v, uint32_t bx, uint32_t by, uint32_t bz)
{
    return bx + (uint64_t)v->nb[0] * (by + (uint64_t)v->nb[1] * bz);
}

// owned base-index range of brick b on axis a (C.7): i0 in [B*b, min(B*b + B - 1, n - 2)]
static inline void owned_range(const vr_volume *v, int a, uint32_t b, int &lo, int &hi)
{
    const int n = (int)(a == 0 ? v->desc.nx : a == 1 ? v->desc.ny : v->desc.nz);
    lo = (int)(v->B * b);
    hi = std::min((int)(v->B * b + v->B - 1), n - 2);
}

// make sure a fully-resident host volume is on the device; `st` then waits for the upload
static vr_status ensure_mirror(vr_volume *v, cudaStream_t st)
{
    if (v->desc.location != VR_HOST_PINNED || v->out_of_core) return VR_OK;
    if (!v->mirror_valid) {
        const size_t bytes = v->total_elems * sizeof(float);
        const size_t chunk = std::max<size_t>((bytes / (size_t)v->n_copy + 255) & ~(size_t)255, 256);
        size_t off = 0;
        for (int i = 0; i < v->n_copy && off < bytes; ++i, off += chunk) {
            const size_t nby = std::min(chunk, bytes - off);
            VR_CUDA(cudaMemcpyAsync((char *)v->mirror + off, (const char *)v->desc.data + off, nby,
                                    cudaMemcpyHostToDevice, v->copy[i]));
            VR_CUDA(cudaEventRecord(v->mirror_ev[i], v->copy[i]));
        }
        v->mirror_valid = true;
        v->stats.h2d_bytes += bytes;
    }
    for (auto e : v->mirror_ev) VR_CUDA(cudaStreamWaitEvent(st, e, 0));
    return VR_OK;
}

// device pointer + strides + origin of brick (bx,by,bz) for the resident layouts
static void resident_brick_view(const vr_volume *v, uint32_t bx, uint32_t by, uint32_t bz, BrickK &k)
{
    if (v->desc.layout == VR_LINEAR) {
        k.base = v->dev_data; k.sy = v->desc.nx; k.sz = (long long)v->desc.nx * v->desc.ny;
        k.ox = k.oy = k.oz = 0;
    } else {
        k.base = v->dev_data + brick_id(v, bx, by, bz) * v->brick_elems;
        k.sy = v->E; k.sz = (long long)v->E * v->E;
        k.ox = (int)(bx * v->B); k.oy = (int)(by * v->B); k.oz = (int)(bz * v->B);
    }
}

// ------------------------------------------------------------------ out-of-core streamer (A5)
// Returns the device pointer of brick `b` for work enqueued on `st` right after this call and
// makes `st` wait for its upload.  Bricks [0, n_fixed) live permanently in slot b; the others
// pass through a ring of n_ring slots fed round-robin by the copy streams, so uploads of the
// next bricks overlap the kernels of the current one (last sentence).
static vr_status stream_brick_acquire(vr_volume *v, uint64_t b, cudaStream_t st, const float **ptr, uint32_t *slot_out)
{
    uint32_t slot;
    bool upload;
    if (b < v->n_fixed) { slot = (uint32_t)b; upload = !v->fixed_loaded[b]; v->fixed_loaded[b] = 1; }
    else { slot = v->n_fixed + (uint32_t)(v->ring_pos++ % v->n_ring); upload = true; }
    float *dst = v->pool + (size_t)slot * v->brick_elems;
    if (upload) {
        cudaStream_t cs = v->copy[v->copy_rr++ % (uint64_t)v->n_copy];
        if (v->slot_used[slot]) VR_CUDA(cudaStreamWaitEvent(cs, v->ev_free[slot], 0));
        const size_t bytes = v->brick_elems * sizeof(float);
        VR_CUDA(cudaMemcpyAsync(dst, v->desc.data + b * v->brick_elems, bytes, cudaMemcpyHostToDevice, cs));
        VR_CUDA(cudaEventRecord(v->ev_up[slot], cs));
        v->stats.h2d_bytes += bytes;
        v->slot_used[slot] = 1;
    }
    if (v->slot_used[slot]) VR_CUDA(cudaStreamWaitEvent(st, v->ev_up[slot], 0));
    *ptr = dst; *slot_out = slot;
    return VR_OK;
}

static vr_status stream_brick_release(vr_volume *v, uint32_t slot, cudaStream_t st)
{
    if (slot >= v->n_fixed) VR_CUDA(cudaEventRecord(v->ev_free[slot], st));
    return VR_OK;
}

// ------------------------------------------------------------------ per-frame brick planning (A4)
struct PlannedBrick { BrickK k; double key; uint32_t b[3]; uint64_t id; };

// bricks that own samples and touch the screen, in visibility order (C.7)
static void plan_bricks(const vr_volume *v, const vr_camera *c, std::vector<PlannedBrick> &out, uint32_t &culled)
{
    const bool perspective = zero3(c->ou) && zero3(c->ov);
    const int n[3] = { (int)v->desc.nx, (int)v->desc.ny, (int)v->desc.nz };
    out.clear();
    culled = 0;
    for (uint32_t bz = 0; bz < v->nb[2]; ++bz)
        for (uint32_t by = 0; by < v->nb[1]; ++by)
            for (uint32_t bx = 0; bx < v->nb[0]; ++bx) {
                PlannedBrick p;
                p.b[0] = bx; p.b[1] = by; p.b[2] = bz; p.id = brick_id(v, bx, by, bz);
                bool empty = false;
                double lo[3], hi[3];
                p.key = 0.0;
                for (int a = 0; a < 3; ++a) {
                    owned_range(v, a, p.b[a], p.k.lo[a], p.k.hi[a]);
                    if (p.k.lo[a] > p.k.hi[a]) empty = true;
                    brick_cell(p.k.lo[a], p.k.hi[a], n[a], lo[a], hi[a]);
                    p.key += brick_key_term(perspective, (double)v->B, p.b[a], (double)c->o0[a], (double)c->d0[a]);
                }
                if (empty) continue;
                box_rect(c, perspective, lo, hi, p.k.x0, p.k.y0, p.k.x1, p.k.y1);
                if (p.k.x1 <= p.k.x0 || p.k.y1 <= p.k.y0) { ++culled; continue; }
                p.k.frag_off = 0;
                p.k.base = nullptr; p.k.sy = p.k.sz = 0; p.k.ox = p.k.oy = p.k.oz = 0;
                out.push_back(p);
            }
    std::stable_sort(out.begin(), out.end(), [](const PlannedBrick &a, const PlannedBrick &b) { return a.key < b.key; });
}

static vr_status staging_acquire(vr_volume *v, size_t bytes, Staging **out)
{
    Staging &s = v->staging[v->staging_next];
    v->staging_next = (v->staging_next + 1) % kStagingRing;
    if (!s.done) VR_CUDA(cudaEventCreateWithFlags(&s.done, cudaEventDisableTiming));
    if (s.in_flight) { VR_CUDA(cudaEventSynchronize(s.done)); s.in_flight = false; }
    if (bytes > s.cap) {
        if (s.h) { VR_CUDA(cudaFreeHost(s.h)); s.h = nullptr; }
        if (s.d) { VR_CUDA(cudaFree(s.d)); s.d = nullptr; }
        s.cap = 0;
        const size_t want = bytes + bytes / 2 + 4096;
        VR_CUDA(cudaMallocHost(&s.h, want));
        VR_CUDA(cudaMalloc(&s.d, want));
        s.cap = want;
    }
    *out = &s;
    return VR_OK;
}

static CamK to_camk(const vr_camera *c)
{
    CamK k;
    for (int a = 0; a < 3; ++a) {
        k.o0[a] = c->o0[a]; k.ou[a] = c->ou[a]; k.ov[a] = c->ov[a];
        k.d0[a] = c->d0[a]; k.du[a] = c->du[a]; k.dv[a] = c->dv[a];
    }
    k.step = c->step;
    k.t_min = 1.0f - c->ert_alpha;        // one float32 subtraction (C.5)
    k.width = (int)c->width; k.height = (int)c->height;
    k.sub = 1; k.sx = k.sy = 0;
    return k;
}

// ------------------------------------------------------------------ render paths
static vr_status render_single(vr_volume *v, const CamK &cam, int mode, bool ert, const TfK &tf, float *img,
                               long long pitch_f, cudaStream_t st)
{
    VolK V;
    V.base = v->dev_data; V.sy = v->desc.nx; V.sz = (long long)v->desc.nx * v->desc.ny;
    V.nx = (int)v->desc.nx; V.ny = (int)v->desc.ny; V.nz = (int)v->desc.nz; V.ox = V.oy = V.oz = 0;
    launch_march_full(mode, ert, v->opt_wide != 0, cam, V, tf, img, pitch_f, st);
    v->stats.kernel_launches += 1;
    v->stats.path = 1;
    v->stats.bricks_drawn = (uint32_t)v->n_bricks;
    return VR_OK;
}

static vr_status render_lanes(vr_volume *v, const vr_camera *c, const CamK &cam, int mode, bool ert, const TfK &tf,
                              const PartK *part, float *img, long long pitch_f, cudaStream_t st);
static bool lanes_addressable(const vr_volume *v);

// ------------------------------------------------------------------ empty bricks (S38)
// C.4 table index of a scalar, the float32 sequence of classify() (host code is built without contraction)
static inline int tf_index_host(float s, float scale, float bias)
{
    float u = fmaf(s, scale, bias);
    u = u != u ? 0.0f : fminf(fmaxf(u, 0.0f), 1.0f);
    const int i = (int)(u * 255.0f);
    return i > 254 ? 254 : i;
}

// every sample that reads only voxels of [mn, mx] has opacity exactly 0 under the handle's transfer function
// (same argument and same dilation as k_macro_flags, vr_macro.cu)
static bool range_is_empty(const vr_volume *v, float mn, float mx)
{
    if (!(mn >= -FLT_MAX && mx <= FLT_MAX && mn <= mx)) return false;
    const float e = fmaf(fmaxf(fabsf(mn), fabsf(mx)), 4.76837158203125e-7f, FLT_MIN);
    const int lo = tf_index_host(mn - e, v->tf_scale, v->tf_bias), hi = tf_index_host(mx + e, v->tf_scale, v->tf_bias);
    for (int j = lo; j <= hi + 1; ++j)
        if (v->tf_tab[4 * j + 3] != 0.0f) return false;
    return true;
}

static inline float key_to_float(unsigned int k)
{
    const unsigned int b = (k & 0x80000000u) ? (k & 0x7fffffffu) : ~k;
    float f; memcpy(&f, &b, 4); return f;
}

// drops the bricks of a brick-major volume whose slot range maps to opacity 0 (EA only; needs the ranges of the
// first summary pass to have ARRIVED on the host: no waiting here)
static void cull_empty_bricks(vr_volume *v, int mode, std::vector<PlannedBrick> &plan)
{
    v->stats.bricks_empty = 0;
    if (mode != VR_EA || !v->opt_skip || !v->tf_has_zero || !v->brick_rng_issued) return;
    if (cudaEventQuery(v->brick_rng_ev) != cudaSuccess) { cudaGetLastError(); return; }
    size_t keep = 0;
    for (size_t i = 0; i < plan.size(); ++i) {
        const BrickRangeK &r = v->h_brick_rng[plan[i].id];
        const bool empty = !r.bad && range_is_empty(v, key_to_float(r.enc_min), key_to_float(r.enc_max));
        if (empty) { v->stats.bricks_empty++; continue; }
        if (keep != i) plan[keep] = plan[i];
        ++keep;
    }
    plan.resize(keep);
}

// Sort-last (C.7, A10): per-(pixel, brick) fragments over each brick's screen rectangle, folded per pixel in
// visibility order by k_composite.  Fragments of a VR_LINEAR volume come from ONE lane-mapped march per frame
// that flushes the ray state at every change of owner brick; bricks of a resident VR_BRICKED_HALO1 volume are
// marched one (brick, pixel tile) per CTA.  Both produce the same fragments bit for bit.
static vr_status render_sort_last(vr_volume *v, const vr_camera *c, const CamK &cam, int mode, const TfK &tf,
                                  float *img, long long pitch_f, cudaStream_t st)
{
    std::vector<PlannedBrick> plan;
    uint32_t culled = 0;
    plan_bricks(v, c, plan, culled);
    cull_empty_bricks(v, mode, plan);
    const int W = cam.width, H = cam.height;
    const int bins_x = (W + 15) / 16, bins_y = (H + 15) / 16;
    // fragments, work items, bins
    uint64_t n_frag = 0;
    size_t n_work = 0;
    std::vector<uint32_t> bin_cnt((size_t)bins_x * bins_y + 1, 0);
    for (auto &p : plan) {
        resident_brick_view(v, p.b[0], p.b[1], p.b[2], p.k);
        p.k.frag_off = n_frag;
        const int w = p.k.x1 - p.k.x0, h = p.k.y1 - p.k.y0;
        n_frag += (uint64_t)w * h;
        n_work += (size_t)((w + 15) / 16) * ((h + 7) / 8);
        for (int ty = p.k.y0 / 16; ty <= (p.k.y1 - 1) / 16; ++ty)
            for (int tx = p.k.x0 / 16; tx <= (p.k.x1 - 1) / 16; ++tx) bin_cnt[(size_t)ty * bins_x + tx]++;
    }
    size_t n_list = 0;
    for (size_t i = 0; i < bin_cnt.size(); ++i) { const uint32_t c2 = bin_cnt[i]; bin_cnt[i] = (uint32_t)n_list; n_list += c2; }
    if (n_work > 0x7fffffffull) { set_error("too many (brick, tile) work items: %zu", n_work); return VR_ERR_UNSUPPORTED; }

    const bool lanes = v->desc.layout == VR_LINEAR && v->opt_path == 0 && lanes_addressable(v);
    // the lane-mapped march needs no work items: a brick-grid -> plan-index table takes their place
    const size_t work_bytes = lanes ? (size_t)v->n_bricks * sizeof(int) : n_work * sizeof(WorkK);
    const size_t off_bricks = 0;
    const size_t off_work = (off_bricks + plan.size() * sizeof(BrickK) + 255) & ~(size_t)255;
    const size_t off_offs = (off_work + work_bytes + 255) & ~(size_t)255;
    const size_t off_list = (off_offs + bin_cnt.size() * sizeof(uint32_t) + 255) & ~(size_t)255;
    const size_t total = off_list + n_list * sizeof(uint32_t) + 256;
    Staging *s;
    vr_status rc = staging_acquire(v, total, &s);
    if (rc != VR_OK) return rc;
    BrickK *hb = reinterpret_cast<BrickK *>(s->h + off_bricks);
    WorkK *hw = reinterpret_cast<WorkK *>(s->h + off_work);
    uint32_t *ho = reinterpret_cast<uint32_t *>(s->h + off_offs);
    uint32_t *hl = reinterpret_cast<uint32_t *>(s->h + off_list);
    std::vector<uint32_t> fill(bin_cnt.begin(), bin_cnt.end() - 1);
    size_t wi = 0;
    for (size_t bi = 0; bi < plan.size(); ++bi) {
        const BrickK &k = plan[bi].k;
        hb[bi] = k;
        const int tw = (k.x1 - k.x0 + 15) / 16, th = (k.y1 - k.y0 + 7) / 8;
        for (int ty = 0; ty < th && !lanes; ++ty)
            for (int tx = 0; tx < tw; ++tx) { hw[wi].brick = (int)bi; hw[wi].tx = tx; hw[wi].ty = ty; hw[wi].pad = 0; ++wi; }
        for (int ty = k.y0 / 16; ty <= (k.y1 - 1) / 16; ++ty)
            for (int tx = k.x0 / 16; tx <= (k.x1 - 1) / 16; ++tx) hl[fill[(size_t)ty * bins_x + tx]++] = (uint32_t)bi;
    }
    memcpy(ho, bin_cnt.data(), bin_cnt.size() * sizeof(uint32_t));
    if (lanes) {
        int *lut = reinterpret_cast<int *>(hw);
        for (uint64_t b = 0; b < v->n_bricks; ++b) lut[b] = -1;
        for (size_t bi = 0; bi < plan.size(); ++bi) lut[plan[bi].id] = (int)bi;
    }

    rc = v->arena.reserve((size_t)n_frag * (mode == VR_EA ? 4 : 1) + 4);
    if (rc != VR_OK) return rc;
    VR_CUDA(cudaMemcpyAsync(s->d, s->h, total, cudaMemcpyHostToDevice, st));
    v->stats.h2d_bytes += total;

    VolK Vdims;                               // dims only; base / strides / origin come from each BrickK
    Vdims.nx = (int)v->desc.nx; Vdims.ny = (int)v->desc.ny; Vdims.nz = (int)v->desc.nz;
    Vdims.base = nullptr; Vdims.sy = Vdims.sz = 0; Vdims.ox = Vdims.oy = Vdims.oz = 0;
    // 64-bit element offsets only when a linear volume exceeds 2^32-1 voxels; slots never do
    const bool wide = v->opt_wide != 0 || (v->desc.layout == VR_LINEAR && v->n_vox > 0xffffffffull);
    if (lanes) {
        launch_fragment_init(mode, v->arena.p, n_frag, v->sm_count * 8, st);
        PartK P;
        P.bricks = reinterpret_cast<const BrickK *>(s->d + off_bricks);
        P.lut = reinterpret_cast<const int *>(s->d + off_work);
        P.arena = v->arena.p; P.B = (int)v->B; P.nbx = (int)v->nb[0]; P.nby = (int)v->nb[1];
        if (n_frag) v->stats.kernel_launches += 1;
        rc = render_lanes(v, c, cam, mode, false, tf, &P, img, pitch_f, st);      // counts its own one or two launches
        if (rc != VR_OK) return rc;
    } else {
        launch_march_bricks(mode, wide, cam, Vdims, tf, reinterpret_cast<const BrickK *>(s->d + off_bricks),
                            reinterpret_cast<const WorkK *>(s->d + off_work), (int)n_work, v->arena.p, st);
        if (n_work) v->stats.kernel_launches += 1;
    }
    BinsK bins;
    bins.offs = reinterpret_cast<const unsigned int *>(s->d + off_offs);
    bins.list = reinterpret_cast<const unsigned int *>(s->d + off_list);
    bins.tiles_x = bins_x; bins.tile = 16;
    launch_composite(mode, cam, reinterpret_cast<const BrickK *>(s->d + off_bricks), bins, v->arena.p, img, pitch_f, st);
    VR_CUDA(cudaEventRecord(s->done, st));
    s->in_flight = true;
    v->stats.kernel_launches += 1;
    v->stats.path = 2;
    v->stats.fragments = n_frag;
    v->stats.bricks_drawn = (uint32_t)plan.size();
    v->stats.bricks_culled = culled;
    return VR_OK;
}

// brick-by-brick front to back, ray state carried in the image (exact ERT).  Used for every
// out-of-core volume and for resident VR_BRICKED_HALO1 volumes without VR_SORT_LAST.
static vr_status render_chain(vr_volume *v, const vr_camera *c, const CamK &cam, int mode, bool ert, const TfK &tf,
                              float *img, long long pitch_f, cudaStream_t st)
{
    std::vector<PlannedBrick> plan;
    uint32_t culled = 0;
    plan_bricks(v, c, plan, culled);
    cull_empty_bricks(v, mode, plan);
    VolK V;
    V.nx = (int)v->desc.nx; V.ny = (int)v->desc.ny; V.nz = (int)v->desc.nz;
    V.base = nullptr; V.sy = V.sz = 0; V.ox = V.oy = V.oz = 0;
    launch_chain_init(mode, cam.width, cam.height, img, pitch_f, st);
    v->stats.kernel_launches += 1;
    for (auto &p : plan) {
        uint32_t slot = 0;
        if (v->out_of_core) {
            const float *ptr;
            vr_status rc = stream_brick_acquire(v, p.id, st, &ptr, &slot);
            if (rc != VR_OK) return rc;
            p.k.base = ptr; p.k.sy = v->E; p.k.sz = (long long)v->E * v->E;
            p.k.ox = (int)(p.b[0] * v->B); p.k.oy = (int)(p.b[1] * v->B); p.k.oz = (int)(p.b[2] * v->B);
        } else resident_brick_view(v, p.b[0], p.b[1], p.b[2], p.k);
        launch_chain_brick(mode, ert, v->opt_wide != 0, cam, V, tf, p.k, img, pitch_f, st);
        v->stats.kernel_launches += 1;
        if (v->out_of_core) { vr_status rc = stream_brick_release(v, slot, st); if (rc != VR_OK) return rc; }
    }
    if (mode == VR_EA) { launch_chain_finish(cam.width, cam.height, img, pitch_f, st); v->stats.kernel_launches += 1; }
    v->stats.path = 3;
    v->stats.bricks_drawn = (uint32_t)plan.size();
    v->stats.bricks_culled = culled;
    return VR_OK;
}

// ------------------------------------------------------------------ lane-mapped single march (vr_lanes.cu)
// The z-fastest copy is made lazily, the first time a view has pixels that travel mostly along x, when
// the option allows it and the device has room; without it such pixels are rendered from the x-fastest
// array (same results, slower).
static vr_status ensure_zfast(vr_volume *v, cudaStream_t st, bool *have)
{
    *have = false;
    if (!v->opt_zcopy || v->desc.layout != VR_LINEAR || v->out_of_core || v->zfast_failed) return VR_OK;
    if (!v->zfast) {
        const size_t bytes = (size_t)v->n_vox * sizeof(float);
        size_t free_b = 0, total_b = 0;
        VR_CUDA(cudaMemGetInfo(&free_b, &total_b));
        if ((v->desc.nz + 31) / 32 > 65535u || free_b < bytes + ((size_t)512 << 20)) { v->zfast_failed = true; return VR_OK; }
        float *p = nullptr;
        if (cudaMalloc(&p, bytes) != cudaSuccess) { cudaGetLastError(); v->zfast_failed = true; return VR_OK; }
        v->zfast = p;
        if (!v->zfast_ev) VR_CUDA(cudaEventCreateWithFlags(&v->zfast_ev, cudaEventDisableTiming));
        launch_transpose_xz(v->dev_data, v->zfast, (int)v->desc.nx, (int)v->desc.ny, (int)v->desc.nz, st);
        VR_CUDA(cudaEventRecord(v->zfast_ev, st));
        v->stats.kernel_launches += (v->desc.ny + 65534) / 65535;
        v->stats.resident_bytes += bytes;
    }
    VR_CUDA(cudaStreamWaitEvent(st, v->zfast_ev, 0));
    *have = true;
    return VR_OK;
}

// The table set by vr_set_transfer_function reaches the device on the stream of the first render that uses it
// (stream order: renders already enqueued on that stream keep the table they were launched with).
static vr_status upload_tf(vr_volume *v, cudaStream_t st)
{
    if (!v->tf_dirty) return VR_OK;
    Staging *s;
    vr_status rc = staging_acquire(v, sizeof(v->tf_tab), &s);
    if (rc != VR_OK) return rc;
    memcpy(s->h, v->tf_tab, sizeof(v->tf_tab));
    VR_CUDA(cudaMemcpyAsync(v->d_tf, s->h, sizeof(v->tf_tab), cudaMemcpyHostToDevice, st));
    VR_CUDA(cudaEventRecord(s->done, st));
    s->in_flight = true;
    v->stats.h2d_bytes += sizeof(v->tf_tab);
    v->tf_dirty = false;
    return VR_OK;
}

// Macrocell grid of a resident linear volume (made once, on the render's stream) and the per-transfer-function
// flags (remade after every vr_set_transfer_function).  Leaves M.flag == nullptr when skipping cannot be used.
static vr_status ensure_macro(vr_volume *v, const TfK &tf, cudaStream_t st, MacroK &M)
{
    M.flag = nullptr; M.n_skip = nullptr; M.min_skip = ~0ull; M.cx = M.cy = M.cz = 0;
    v->stats.skip_variant = 0;
    if (!v->opt_skip || !v->tf_has_zero || v->macro_failed || v->desc.layout != VR_LINEAR || v->out_of_core) return VR_OK;
    const int n[3] = { (int)v->desc.nx, (int)v->desc.ny, (int)v->desc.nz };
    if (!v->macro_mm) {
        for (int a = 0; a < 3; ++a) v->mc[a] = (n[a] - 2) / kMacroEdge + 1;       // base indices 0 .. n-2
        const size_t cells = (size_t)v->mc[0] * v->mc[1] * v->mc[2];
        if (v->mc[2] > 65535 || cells > 0x7fffffffull) { v->macro_failed = true; return VR_OK; }
        float2 *mm = nullptr; unsigned char *fl = nullptr;
        if (cudaMalloc(&mm, cells * sizeof(float2)) != cudaSuccess) { cudaGetLastError(); v->macro_failed = true; return VR_OK; }
        if (cudaMalloc(&fl, cells) != cudaSuccess) { cudaGetLastError(); cudaFree(mm); v->macro_failed = true; return VR_OK; }
        v->macro_mm = mm; v->macro_flag = fl;
        VR_CUDA(cudaMalloc(&v->d_nskip, sizeof(unsigned long long)));
        VR_CUDA(cudaMallocHost(&v->h_nskip, sizeof(unsigned long long)));
        VR_CUDA(cudaEventCreateWithFlags(&v->nskip_ev, cudaEventDisableTiming));
        *v->h_nskip = 0;
        MacroK G; G.flag = nullptr; G.n_skip = nullptr; G.min_skip = 0; G.cx = v->mc[0]; G.cy = v->mc[1]; G.cz = v->mc[2];
        launch_macro_minmax(v->dev_data, n[0], n[1], n[2], G, v->macro_mm, st);
        v->stats.kernel_launches += 1;
        v->stats.resident_bytes += cells * (sizeof(float2) + 1);
        v->macro_flags_dirty = true;
    }
    const long long cells = (long long)v->mc[0] * v->mc[1] * v->mc[2];
    if (v->macro_flags_dirty) {
        VR_CUDA(cudaMemsetAsync(v->d_nskip, 0, sizeof(unsigned long long), st));
        launch_macro_flags(v->macro_mm, cells, tf, v->macro_flag, v->d_nskip,
                           (int)std::min<long long>((cells + 255) / 256, (long long)v->sm_count * 8), st);
        VR_CUDA(cudaMemcpyAsync(v->h_nskip, v->d_nskip, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
        VR_CUDA(cudaEventRecord(v->nskip_ev, st));
        MacroK G; G.flag = nullptr; G.n_skip = nullptr; G.min_skip = 0; G.cx = v->mc[0]; G.cy = v->mc[1]; G.cz = v->mc[2];
        launch_macro_blocks(v->macro_flag, G, (int)std::min<long long>((cells / 512 + 8) / 8, (long long)v->sm_count * 8), st);
        v->stats.kernel_launches += 2;
        v->macro_flags_dirty = false;
    }
    const unsigned long long min_skip = (unsigned long long)std::max<long long>(1, cells / 64);   // worth a byte load per sample from ~1.6 % empty cells
    // once the count of this transfer function has reached the host (no waiting), a grid with too few empty cells
    // is not consulted at all: the plain kernel variant is launched
    if (cudaEventQuery(v->nskip_ev) == cudaSuccess) { if (*v->h_nskip < min_skip) return VR_OK; }
    else cudaGetLastError();
    M.flag = v->macro_flag; M.n_skip = v->d_nskip;
    M.min_skip = min_skip;
    M.cx = v->mc[0]; M.cy = v->mc[1]; M.cz = v->mc[2];
    v->stats.skip_variant = 1;
    v->stats.macro_cells = (uint64_t)cells;
    return VR_OK;
}

// the lane-mapped kernel forms offsets inside one plane of either volume copy in 32 bits
static bool lanes_addressable(const vr_volume *v)
{
    return (uint64_t)v->desc.nx * v->desc.ny <= 0xffffffffull && (uint64_t)v->desc.ny * v->desc.nz <= 0xffffffffull;
}

// VR_OPT_ROW_LOADS = 2 (auto): 16-byte row loads for the launches whose rays can enter the volume through a face
// perpendicular to the memory-fast axis of the copy they read.  Those are the oblique views, where the lanes of a
// warp sit on rows of their own and the corner loads are bound by cache lines touched (3.5-4.6 lines per sample
// with two scalar loads per row, 2.6-3.1 with one quad: profiles/r2_lane_traffic_model.md); on the other views the
// lanes share rows, issue binds, and the selects of the quad variant cost more than its lines save.  A face is
// visible iff the eye is beyond it (perspective) or the direction has a component along its axis (orthographic).
static bool launch_quad(const vr_volume *v, const vr_camera *c, int fast)
{
    if (v->opt_quad != 2) return v->opt_quad == 1;
    const float n_fast = (float)(fast == 0 ? v->desc.nx : v->desc.nz);
    if (zero3(c->ou) && zero3(c->ov)) return c->o0[fast] < 0.0f || c->o0[fast] > n_fast;
    if (zero3(c->du) && zero3(c->dv)) return c->d0[fast] != 0.0f;
    return true;
}

// part != nullptr: per-(ray, owner brick) fragments for the sort-last compositor instead of pixels
static vr_status render_lanes(vr_volume *v, const vr_camera *c, const CamK &cam, int mode, bool ert, const TfK &tf,
                              const PartK *part, float *img, long long pitch_f, cudaStream_t st)
{
    const int n[3] = { (int)v->desc.nx, (int)v->desc.ny, (int)v->desc.nz };
    MacroK Mc;
    Mc.flag = nullptr; Mc.n_skip = nullptr; Mc.min_skip = ~0ull; Mc.cx = Mc.cy = Mc.cz = 0;
    if (mode == VR_EA && !part) { vr_status rc = ensure_macro(v, tf, st, Mc); if (rc != VR_OK) return rc; }
    else v->stats.skip_variant = 0;
    // how many of 9 probe pixels (corners, edge midpoints, centre) travel mostly along x
    int n_x = 0;
    for (int py = 0; py < 3; ++py)
        for (int px = 0; px < 3; ++px) {
            const double x = 0.5 * px * cam.width, y = 0.5 * py * cam.height;
            const double gx = (double)c->d0[0] + x * (double)c->du[0] + y * (double)c->dv[0];
            const double gz = (double)c->d0[2] + x * (double)c->du[2] + y * (double)c->dv[2];
            if (std::fabs(gx) > std::fabs(gz)) ++n_x;
        }
    bool have_z = false;
    if (n_x > 0) { vr_status rc = ensure_zfast(v, st, &have_z); if (rc != VR_OK) return rc; }
    LaneVolK A, Z;
    A.base = v->dev_data; A.sa = n[0]; A.sb = (long long)n[0] * n[1]; A.nx = n[0]; A.ny = n[1]; A.nz = n[2];
    Z = A; Z.base = v->zfast; Z.sa = (long long)n[1] * n[2]; Z.sb = n[2];
    LaneMapK M;
    int rows;
    if (!have_z || n_x == 0) {
        make_lane_map(c, n, 0, 0, v->opt_lag, v->opt_tile_shear, M, rows);
        v->stats.quad_launches += launch_rows(mode, ert, cam, A, 0, tf, M, Mc, part, v->opt_wide != 0, launch_quad(v, c, 0), rows, img, pitch_f, st);
        v->stats.kernel_launches += 1;
    } else if (n_x == 9) {
        make_lane_map(c, n, 2, 0, v->opt_lag, v->opt_tile_shear, M, rows);
        v->stats.quad_launches += launch_rows(mode, ert, cam, Z, 2, tf, M, Mc, part, v->opt_wide != 0, launch_quad(v, c, 2), rows, img, pitch_f, st);
        v->stats.kernel_launches += 1;
    } else {
        make_lane_map(c, n, 0, 1, v->opt_lag, v->opt_tile_shear, M, rows);
        v->stats.quad_launches += launch_rows(mode, ert, cam, A, 0, tf, M, Mc, part, v->opt_wide != 0, launch_quad(v, c, 0), rows, img, pitch_f, st);
        make_lane_map(c, n, 2, 2, v->opt_lag, v->opt_tile_shear, M, rows);
        v->stats.quad_launches += launch_rows(mode, ert, cam, Z, 2, tf, M, Mc, part, v->opt_wide != 0, launch_quad(v, c, 2), rows, img, pitch_f, st);
        v->stats.kernel_launches += 2;
    }
    v->stats.path = 7;
    v->stats.zfast_copy = v->zfast ? 1u : 0u;
    v->stats.bricks_drawn = (uint32_t)v->n_bricks;
    return VR_OK;
}

// ------------------------------------------------------------------ one pass over every voxel (A1, A2, statistics)
// VR_LINEAR: one launch on the flat array; VR_BRICKED_HALO1: one launch per brick on its box without the halo,
// out of core through the brick streamer (uploads of the next bricks overlap the kernel of the current one).
template <typename Flat, typename Box>
static vr_status sweep_volume(vr_volume *v, cudaStream_t st, int grid, Flat &&flat, Box &&box_fn)
{
    if (v->desc.layout == VR_LINEAR) {
        flat(v->dev_data, (unsigned long long)v->n_vox, grid);
        v->stats.kernel_launches += 1;
        return VR_OK;
    }
    const uint32_t n[3] = { v->desc.nx, v->desc.ny, v->desc.nz };
    for (uint32_t bz = 0; bz < v->nb[2]; ++bz)
        for (uint32_t by = 0; by < v->nb[1]; ++by)
            for (uint32_t bx = 0; bx < v->nb[0]; ++bx) {
                const uint64_t id = brick_id(v, bx, by, bz);
                BoxK box;
                uint32_t slot = 0;
                if (v->out_of_core) {
                    const float *ptr;
                    vr_status rc = stream_brick_acquire(v, id, st, &ptr, &slot);
                    if (rc != VR_OK) return rc;
                    box.base = ptr;
                } else box.base = v->dev_data + id * v->brick_elems;
                box.sy = v->E; box.sz = (long long)v->E * v->E;
                const uint32_t bb[3] = { bx, by, bz };
                int ext[3];
                for (int a = 0; a < 3; ++a) ext[a] = (int)std::min(v->B, n[a] - bb[a] * v->B);   // halo excluded
                box.ex = ext[0]; box.ey = ext[1]; box.ez = ext[2];
                const int bgrid = (int)std::max<long long>(1, std::min<long long>(grid, ((long long)box.ey * box.ez + 15) / 16));
                box_fn(box, bgrid, id);
                v->stats.kernel_launches += 1;
                if (v->out_of_core) { vr_status rc = stream_brick_release(v, slot, st); if (rc != VR_OK) return rc; }
            }
    return VR_OK;
}

}  // namespace vr

// ====================================================================== C ABI
extern "C" {

VR_API const char *vr_last_error(void) { return g_err; }
VR_API const char *vr_version(void) { return "vr-b200 0.1 sm_100a"; }

VR_API vr_status vr_create_volume(const vr_volume_desc *d, vr_volume **out)
{
    g_err[0] = 0;
    VR_REQUIRE(d && out, "vr_create_volume: NULL argument");
    *out = nullptr;
    VR_REQUIRE(d->struct_size == sizeof(vr_volume_desc), "vr_volume_desc.struct_size %u != %zu", d->struct_size, sizeof(vr_volume_desc));
    VR_REQUIRE(d->nx >= 2 && d->ny >= 2 && d->nz >= 2, "each dimension must be >= 2 (got %ux%ux%u)", d->nx, d->ny, d->nz);
    VR_REQUIRE(d->nx <= 0x7fffffffu && d->ny <= 0x7fffffffu && d->nz <= 0x7fffffffu, "dimension too large");
    VR_REQUIRE(d->layout == VR_LINEAR || d->layout == VR_BRICKED_HALO1, "bad layout %u", d->layout);
    VR_REQUIRE(d->location == VR_DEVICE || d->location == VR_HOST_PINNED, "bad location %u", d->location);
    VR_REQUIRE(d->data != nullptr, "data is NULL");
    VR_REQUIRE(d->layout == VR_LINEAR || d->brick > 0, "VR_BRICKED_HALO1 needs brick > 0");
    VR_REQUIRE(d->n_copy_streams <= (uint32_t)kMaxCopyStreams, "n_copy_streams must be <= %d", kMaxCopyStreams);
    VR_REQUIRE(((uintptr_t)d->data & 15u) == 0, "data must be 16-byte aligned");

    vr_volume *v = new (std::nothrow) vr_volume();
    if (!v) { set_error("host allocation failed"); return VR_ERR_OUT_OF_MEMORY; }
    v->desc = *d;
    memset(&v->stats, 0, sizeof(v->stats));
    v->stats.struct_size = sizeof(vr_stats);
    const uint32_t maxdim = std::max(d->nx, std::max(d->ny, d->nz));
    v->B = d->brick ? d->brick : maxdim;
    v->E = v->B + 1;
    const uint32_t n[3] = { d->nx, d->ny, d->nz };
    for (int a = 0; a < 3; ++a) v->nb[a] = d->brick ? (n[a] + v->B - 1) / v->B : 1;
    if (v->nb[0] > 65535 || v->nb[1] > 65535 || v->nb[2] > 65535) {
        delete v; set_error("brick grid exceeds 65535 bricks on an axis"); return VR_ERR_INVALID_ARG;
    }
    v->n_bricks = (uint64_t)v->nb[0] * v->nb[1] * v->nb[2];
    v->n_vox = (uint64_t)d->nx * d->ny * d->nz;
    v->brick_elems = (uint64_t)v->E * v->E * v->E;
    v->total_elems = d->layout == VR_LINEAR ? v->n_vox : v->n_bricks * v->brick_elems;
    v->stats.n_bricks = (uint32_t)std::min<uint64_t>(v->n_bricks, 0xffffffffu);

#define VR_FAIL_CUDA(call)                                                   \
    do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { vr_status r__ = cuda_fail(e__, #call); free_volume(v); return r__; } } while (0)

    VR_FAIL_CUDA(cudaGetDevice(&v->device));
    cudaPointerAttributes attr;
    VR_FAIL_CUDA(cudaPointerGetAttributes(&attr, d->data));
    if (d->location == VR_DEVICE) {
        if (attr.type != cudaMemoryTypeDevice && attr.type != cudaMemoryTypeManaged) {
            free_volume(v); set_error("location VR_DEVICE but data is not a device pointer"); return VR_ERR_INVALID_ARG;
        }
        // the handle lives on the device that owns the data, whatever device is current in the calling thread
        if (attr.type == cudaMemoryTypeDevice && attr.device != v->device) {
            v->device = attr.device;
            VR_FAIL_CUDA(cudaSetDevice(v->device));
        }
        v->dev_data = d->data;
    }
    VR_FAIL_CUDA(cudaDeviceGetAttribute(&v->sm_count, cudaDevAttrMultiProcessorCount, v->device));
    if (d->location != VR_DEVICE) {
        if (attr.type != cudaMemoryTypeHost) {
            free_volume(v); set_error("location VR_HOST_PINNED but data is not page-locked host memory"); return VR_ERR_INVALID_ARG;
        }
        v->n_copy = d->n_copy_streams ? (int)d->n_copy_streams : 4;
        for (int i = 0; i < v->n_copy; ++i) VR_FAIL_CUDA(cudaStreamCreateWithFlags(&v->copy[i], cudaStreamNonBlocking));
        const uint64_t bytes = v->total_elems * sizeof(float);
        if (d->resident_bytes == 0 || d->resident_bytes >= bytes) {
            VR_FAIL_CUDA(cudaMalloc(&v->mirror, bytes));
            v->dev_data = v->mirror;
            v->mirror_ev.resize(v->n_copy);
            for (auto &e : v->mirror_ev) VR_FAIL_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
            v->stats.resident_bytes = bytes;
        } else {
            if (d->layout != VR_BRICKED_HALO1) {
                free_volume(v); set_error("out-of-core streaming (resident_bytes < volume bytes) needs VR_BRICKED_HALO1");
                return VR_ERR_UNSUPPORTED;
            }
            const uint64_t bb = v->brick_elems * sizeof(float);
            v->n_slots = (uint32_t)std::min<uint64_t>(d->resident_bytes / bb, v->n_bricks);
            if (v->n_slots < 2) { free_volume(v); set_error("resident_bytes holds fewer than 2 bricks of %llu bytes", (unsigned long long)bb); return VR_ERR_INVALID_ARG; }
            v->n_ring = std::min<uint32_t>(v->n_slots, std::max<uint32_t>(2u, 2u * (uint32_t)v->n_copy));
            v->n_fixed = v->n_slots - v->n_ring;
            v->out_of_core = true;
            VR_FAIL_CUDA(cudaMalloc(&v->pool, (size_t)v->n_slots * bb));
            v->fixed_loaded.assign(v->n_fixed, 0);
            v->slot_used.assign(v->n_slots, 0);
            v->ev_up.resize(v->n_slots); v->ev_free.resize(v->n_slots);
            for (auto &e : v->ev_up) VR_FAIL_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
            for (auto &e : v->ev_free) VR_FAIL_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
            v->stats.resident_bytes = (uint64_t)v->n_slots * bb;
        }
    }
    VR_FAIL_CUDA(cudaMalloc(&v->d_tf, 257 * sizeof(float4)));
    VR_FAIL_CUDA(cudaMalloc(&v->d_sum, sizeof(SummaryScratch)));
    VR_FAIL_CUDA(cudaMalloc(&v->d_sum_out, VR_SUMMARY_BYTES(4096)));
#undef VR_FAIL_CUDA
    *out = v;
    return VR_OK;
}

VR_API vr_status vr_destroy_volume(vr_volume *v)
{
    g_err[0] = 0;
    free_volume(v);
    return VR_OK;
}

VR_API vr_status vr_set_transfer_function(vr_volume *v, const float *rgba, float vmin, float vmax)
{
    g_err[0] = 0;
    VR_REQUIRE(v && rgba, "vr_set_transfer_function: NULL argument");
    VR_REQUIRE(std::isfinite(vmin) && std::isfinite(vmax) && vmax > vmin, "need finite vmin < vmax (got %g, %g)", vmin, vmax);
    bool has_zero = false;
    for (int i = 0; i < 1024; ++i)
        VR_REQUIRE(std::isfinite(rgba[i]) && rgba[i] >= 0.0f && rgba[i] <= 1.0f, "table entry %d = %g is outside [0,1]", i, rgba[i]);
    const float scale = 1.0f / (vmax - vmin), bias = -vmin * scale;   // C.4, float32
    if (v->tf_set && scale == v->tf_scale && bias == v->tf_bias && memcmp(v->tf_tab, rgba, 1024 * sizeof(float)) == 0)
        return VR_OK;                                               // the same table and range again: nothing to redo
    for (int i = 0; i < 1024; ++i) v->tf_tab[i] = rgba[i];
    for (int c = 0; c < 4; ++c) v->tf_tab[1024 + c] = rgba[1020 + c];      // pad entry (never weighted: i <= 254)
    for (int i = 0; i < 255; ++i) has_zero = has_zero || (rgba[4 * i + 3] == 0.0f && rgba[4 * i + 7] == 0.0f);
    v->tf_has_zero = has_zero;                                       // some table interval has opacity exactly 0
    v->tf_scale = scale;
    v->tf_bias = bias;
    v->tf_dirty = true;                                             // uploaded on the stream of the next render
    v->macro_flags_dirty = true;
    v->tf_set = true;
    return VR_OK;
}

VR_API vr_status vr_render(vr_volume *v, const vr_camera *c, int mode, const vr_image *im, void *stream)
{
    g_err[0] = 0;
    VR_REQUIRE(v && c && im, "vr_render: NULL argument");
    VR_REQUIRE(c->struct_size == sizeof(vr_camera), "vr_camera.struct_size %u != %zu", c->struct_size, sizeof(vr_camera));
    VR_REQUIRE(im->struct_size == sizeof(vr_image), "vr_image.struct_size %u != %zu", im->struct_size, sizeof(vr_image));
    VR_REQUIRE(mode == VR_EA || mode == VR_MIP, "bad mode %d", mode);
    VR_REQUIRE(c->width > 0 && c->height > 0 && c->width <= 65536 && c->height <= 65536, "bad image size %ux%u", c->width, c->height);
    VR_REQUIRE(std::isfinite(c->step) && c->step > 0.0f, "step must be finite and > 0 (got %g)", c->step);
    VR_REQUIRE(c->ert_alpha >= 0.0f && c->ert_alpha < 1.0f, "ert_alpha must be in [0,1) (got %g)", c->ert_alpha);
    for (int a = 0; a < 3; ++a)
        VR_REQUIRE(std::isfinite(c->o0[a]) && std::isfinite(c->ou[a]) && std::isfinite(c->ov[a]) && std::isfinite(c->d0[a]) &&
                   std::isfinite(c->du[a]) && std::isfinite(c->dv[a]), "camera vectors must be finite");
    const uint32_t ch = mode == VR_EA ? 4u : 1u;
    VR_REQUIRE(im->channels == ch, "image.channels %u does not match mode (%u expected)", im->channels, ch);
    VR_REQUIRE(im->pixels != nullptr, "image.pixels is NULL");
    VR_REQUIRE(im->location == VR_DEVICE || im->location == VR_HOST_PINNED, "bad image.location %u", im->location);
    const uint64_t row_bytes = (uint64_t)c->width * ch * 4;
    const uint64_t pitch = im->row_pitch_bytes ? im->row_pitch_bytes : row_bytes;
    VR_REQUIRE(pitch >= row_bytes && pitch % (mode == VR_EA ? 16 : 4) == 0, "bad row_pitch_bytes %llu", (unsigned long long)pitch);
    VR_REQUIRE(((uintptr_t)im->pixels & (mode == VR_EA ? 15u : 3u)) == 0, "image.pixels is misaligned");
    if (mode == VR_EA && !v->tf_set) { set_error("emission-absorption render before vr_set_transfer_function"); return VR_ERR_NOT_READY; }
    const bool sort_last = (c->flags & VR_SORT_LAST) != 0;
    // progressive pass: only the pixels of one sub-lattice of the image, in place (VR_SUBSAMPLE)
    const int sub = std::max(1, (int)((c->flags >> 8) & 0xffu)), sub_x = (int)((c->flags >> 16) & 0xffu), sub_y = (int)((c->flags >> 24) & 0xffu);
    VR_REQUIRE(sub_x < sub && sub_y < sub, "VR_SUBSAMPLE: phase (%d, %d) must be below the stride %d", sub_x, sub_y, sub);
    const bool ert = mode == VR_EA && c->ert_alpha > 0.0f;
    const bool persp = zero3(c->ou) && zero3(c->ov), ortho = zero3(c->du) && zero3(c->dv);
    if (sort_last) {
        if (!v->desc.brick) { set_error("VR_SORT_LAST needs a bricked volume (brick > 0)"); return VR_ERR_UNSUPPORTED; }
        if (ert) { set_error("early ray termination is not defined for independent per-brick partials (S15)"); return VR_ERR_UNSUPPORTED; }
        if (v->out_of_core) { set_error("VR_SORT_LAST is not available for out-of-core volumes (they render as a chain)"); return VR_ERR_UNSUPPORTED; }
    }
    const bool need_plan = sort_last || v->out_of_core || v->desc.layout == VR_BRICKED_HALO1;
    if (sub > 1 && need_plan) { set_error("VR_SUBSAMPLE is available for single-march renders of resident VR_LINEAR volumes only"); return VR_ERR_UNSUPPORTED; }
    if (sub > 1 && im->location != VR_DEVICE) { set_error("VR_SUBSAMPLE renders in place: the image must be in device memory"); return VR_ERR_UNSUPPORTED; }
    if (need_plan && !persp && !ortho) { set_error("bricked rendering needs a pure perspective or pure orthographic camera"); return VR_ERR_UNSUPPORTED; }

    VR_CUDA(cudaSetDevice(v->device));
    cudaStream_t st = (cudaStream_t)stream;
    v->stats.kernel_launches = 0; v->stats.h2d_bytes = 0; v->stats.d2h_bytes = 0; v->stats.fragments = 0;
    v->stats.bricks_drawn = v->stats.bricks_culled = v->stats.bricks_empty = v->stats.quad_launches = 0;

    float *img = im->pixels;
    long long pitch_f = (long long)(pitch / 4);
    if (im->location == VR_HOST_PINNED) {
        vr_status rc = v->host_image.reserve((size_t)c->width * c->height * ch);
        if (rc != VR_OK) return rc;
        img = v->host_image.p; pitch_f = (long long)c->width * ch;
    }
    vr_status rc = ensure_mirror(v, st);
    if (rc != VR_OK) return rc;

    if (mode == VR_EA) { rc = upload_tf(v, st); if (rc != VR_OK) return rc; }
    CamK cam = to_camk(c);
    vr_camera lattice = *c;                  // the camera of the pixels this call renders (lane map, class probes)
    if (sub > 1) {
        cam.sub = sub; cam.sx = sub_x; cam.sy = sub_y;
        cam.width = ((int)c->width - sub_x + sub - 1) / sub; cam.height = ((int)c->height - sub_y + sub - 1) / sub;
        lattice.width = (uint32_t)std::max(cam.width, 0); lattice.height = (uint32_t)std::max(cam.height, 0);
        for (int a = 0; a < 3; ++a) {
            lattice.o0[a] += (float)sub_x * c->ou[a] + (float)sub_y * c->ov[a]; lattice.d0[a] += (float)sub_x * c->du[a] + (float)sub_y * c->dv[a];
            lattice.ou[a] *= (float)sub; lattice.ov[a] *= (float)sub; lattice.du[a] *= (float)sub; lattice.dv[a] *= (float)sub;
        }
        if (cam.width <= 0 || cam.height <= 0) return VR_OK;        // the sub-lattice has no pixel in this image
    }
    TfK tf; tf.table = v->d_tf; tf.scale = v->tf_scale; tf.bias = v->tf_bias;
    if (sort_last) rc = render_sort_last(v, c, cam, mode, tf, img, pitch_f, st);
    else if (v->out_of_core || v->desc.layout == VR_BRICKED_HALO1) rc = render_chain(v, c, cam, mode, ert, tf, img, pitch_f, st);
    else if (v->opt_path == 1 || !lanes_addressable(v)) rc = render_single(v, cam, mode, ert, tf, img, pitch_f, st);
    else rc = render_lanes(v, &lattice, cam, mode, ert, tf, nullptr, img, pitch_f, st);
    if (rc != VR_OK) return rc;
    VR_CUDA(cudaGetLastError());
    if (im->location == VR_HOST_PINNED) {
        if (pitch == row_bytes) VR_CUDA(cudaMemcpyAsync(im->pixels, img, row_bytes * c->height, cudaMemcpyDeviceToHost, st));
        else VR_CUDA(cudaMemcpy2DAsync(im->pixels, pitch, img, row_bytes, row_bytes, c->height, cudaMemcpyDeviceToHost, st));
        v->stats.d2h_bytes += row_bytes * c->height;
    }
    v->stats.total_kernel_launches += v->stats.kernel_launches;
    return VR_OK;
}

VR_API vr_status vr_minmax_histogram(vr_volume *v, uint32_t nbins, const float *range, vr_summary *out,
                                     uint32_t out_location, void *stream)
{
    g_err[0] = 0;
    VR_REQUIRE(v && out, "vr_minmax_histogram: NULL argument");
    VR_REQUIRE(nbins >= 1 && nbins <= 4096, "nbins must be in 1..4096 (got %u)", nbins);
    VR_REQUIRE(out_location == VR_DEVICE || out_location == VR_HOST_PINNED, "bad out_location %u", out_location);
    VR_REQUIRE(((uintptr_t)out & 7u) == 0, "out must be 8-byte aligned");
    float lo = 0.0f, hi = 0.0f;
    if (range) {
        lo = range[0]; hi = range[1];
        VR_REQUIRE(std::isfinite(lo) && std::isfinite(hi) && hi >= lo, "range must be finite with range[1] >= range[0]");
    }
    VR_CUDA(cudaSetDevice(v->device));
    cudaStream_t st = (cudaStream_t)stream;
    v->stats.kernel_launches = 0; v->stats.h2d_bytes = 0; v->stats.d2h_bytes = 0;
    vr_status rc = ensure_mirror(v, st);
    if (rc != VR_OK) return rc;
    const int grid = v->sm_count * 2;
    SummaryScratch *S = v->d_sum;
    launch_summary_reset(S, st);
    v->stats.kernel_launches += 1;
    const int n_pass = range ? 1 : 2;
    // brick-major volumes: the first summary call also gathers the value range of every brick slot (the data is
    // immutable while the handle exists), which later renders use to drop empty bricks before upload
    bool gather_ranges = false;
    if (v->desc.layout == VR_BRICKED_HALO1 && !v->brick_rng_issued) {
        if (!v->d_brick_rng) {
            VR_CUDA(cudaMalloc(&v->d_brick_rng, v->n_bricks * sizeof(BrickRangeK)));
            VR_CUDA(cudaMallocHost(&v->h_brick_rng, v->n_bricks * sizeof(BrickRangeK)));
            VR_CUDA(cudaEventCreateWithFlags(&v->brick_rng_ev, cudaEventDisableTiming));
        }
        launch_brick_range_init(v->d_brick_rng, v->n_bricks, st);
        v->stats.kernel_launches += 1;
        gather_ranges = true;
    }
    for (int pass = 0; pass < n_pass; ++pass) {
        // pass 0: min/max (+ histogram when the caller gave the range); pass 1: histogram over [min,max]
        if (range && pass == 0) { launch_summary_range(S, 1, lo, hi, nbins, st); v->stats.kernel_launches += 1; }
        if (pass == 1) { launch_summary_range(S, 0, 0.0f, 0.0f, nbins, st); v->stats.kernel_launches += 1; }
        rc = sweep_volume(v, st, grid,
            [&](const float *p, unsigned long long n, int g) {
                if (pass == 1) launch_hist_flat(p, n, nbins, S, g, st);
                else if (range) launch_minmax_hist_flat(p, n, nbins, S, g, st);
                else launch_minmax_flat(p, n, S, g, st);
            },
            [&](const BoxK &box, int g, uint64_t id) {
                if (pass == 1) launch_hist_box(box, nbins, S, g, st);
                else if (range) launch_minmax_hist_box(box, nbins, S, g, st);
                else launch_minmax_box(box, S, g, st);
                if (gather_ranges && pass == 0) {        // the whole slot, halo included: what the brick's samples read
                    launch_brick_range(box.base, v->brick_elems, v->d_brick_rng + id, std::max(1, std::min(g, 64)), st);
                    v->stats.kernel_launches += 1;
                }
            });
        if (rc != VR_OK) return rc;
        if (gather_ranges && pass == 0) {
            VR_CUDA(cudaMemcpyAsync(v->h_brick_rng, v->d_brick_rng, v->n_bricks * sizeof(BrickRangeK), cudaMemcpyDeviceToHost, st));
            VR_CUDA(cudaEventRecord(v->brick_rng_ev, st));
            v->brick_rng_issued = true;
            v->stats.d2h_bytes += v->n_bricks * sizeof(BrickRangeK);
        }
    }
    if (out_location == VR_DEVICE) launch_summary_finish(S, nbins, out, st);
    else {
        launch_summary_finish(S, nbins, v->d_sum_out, st);
        VR_CUDA(cudaMemcpyAsync(out, v->d_sum_out, VR_SUMMARY_BYTES(nbins), cudaMemcpyDeviceToHost, st));
        v->stats.d2h_bytes += VR_SUMMARY_BYTES(nbins);
    }
    v->stats.kernel_launches += 1;
    VR_CUDA(cudaGetLastError());
    v->stats.total_kernel_launches += v->stats.kernel_launches;
    return VR_OK;
}

VR_API vr_status vr_statistics(vr_volume *v, vr_statistics_result *out, uint32_t out_location, void *stream)
{
    g_err[0] = 0;
    VR_REQUIRE(v && out, "vr_statistics: NULL argument");
    VR_REQUIRE(out_location == VR_DEVICE || out_location == VR_HOST_PINNED, "bad out_location %u", out_location);
    VR_REQUIRE(((uintptr_t)out & 7u) == 0, "out must be 8-byte aligned");
    VR_CUDA(cudaSetDevice(v->device));
    cudaStream_t st = (cudaStream_t)stream;
    v->stats.kernel_launches = 0; v->stats.h2d_bytes = 0; v->stats.d2h_bytes = 0;
    vr_status rc = ensure_mirror(v, st);
    if (rc != VR_OK) return rc;
    if (!v->d_stat) {
        VR_CUDA(cudaMalloc(&v->d_stat, sizeof(StatScratch)));
        VR_CUDA(cudaMalloc(&v->d_stat_out, sizeof(vr_statistics_result)));
    }
    const int grid = std::min(v->sm_count * 2, kStatMaxGrid);
    StatScratch *S = v->d_stat;
    launch_stat_reset(S, st);
    v->stats.kernel_launches += 1;
    // pass 0: count, sum, key range; 1: squared deviations + first select pass; 2-4: select (return at once when
    // the median is already known).  Nothing is read back in between: the one-thread kernel steers the next pass.
    for (int pass = 0; pass < 5; ++pass) {
        rc = sweep_volume(v, st, grid,
            [&](const float *p, unsigned long long n, int g) { launch_stat_pass_flat(pass, p, n, S, g, st); },
            [&](const BoxK &box, int g, uint64_t) { launch_stat_pass_box(pass, box, S, g, st); });
        if (rc != VR_OK) return rc;
        launch_stat_step(S, pass, st);
        v->stats.kernel_launches += 1;
    }
    if (out_location == VR_DEVICE) launch_stat_finish(S, out, st);
    else {
        launch_stat_finish(S, v->d_stat_out, st);
        VR_CUDA(cudaMemcpyAsync(out, v->d_stat_out, sizeof(vr_statistics_result), cudaMemcpyDeviceToHost, st));
        v->stats.d2h_bytes += sizeof(vr_statistics_result);
    }
    v->stats.kernel_launches += 1;
    VR_CUDA(cudaGetLastError());
    v->stats.total_kernel_launches += v->stats.kernel_launches;
    return VR_OK;
}

VR_API vr_status vr_encode_rgba8(vr_volume *v, const vr_encode_desc *d, const vr_image *src, uint8_t *out,
                                 uint64_t out_pitch_bytes, uint32_t out_location, void *stream)
{
    g_err[0] = 0;
    VR_REQUIRE(v && d && src && out, "vr_encode_rgba8: NULL argument");
    VR_REQUIRE(d->struct_size == sizeof(vr_encode_desc), "vr_encode_desc.struct_size %u != %zu", d->struct_size, sizeof(vr_encode_desc));
    VR_REQUIRE(src->struct_size == sizeof(vr_image), "vr_image.struct_size %u != %zu", src->struct_size, sizeof(vr_image));
    VR_REQUIRE(d->mode == VR_EA || d->mode == VR_MIP, "bad mode %u", d->mode);
    VR_REQUIRE(d->width > 0 && d->height > 0 && d->width <= 65536 && d->height <= 65536, "bad image size %ux%u", d->width, d->height);
    const uint32_t ch = d->mode == VR_EA ? 4u : 1u;
    VR_REQUIRE(src->channels == ch && src->location == VR_DEVICE && src->pixels, "src must be a DEVICE image of %u channel(s)", ch);
    const uint64_t row_bytes = (uint64_t)d->width * ch * 4;
    const uint64_t pitch = src->row_pitch_bytes ? src->row_pitch_bytes : row_bytes;
    VR_REQUIRE(pitch >= row_bytes && pitch % (d->mode == VR_EA ? 16 : 4) == 0, "bad src row_pitch_bytes %llu", (unsigned long long)pitch);
    VR_REQUIRE(((uintptr_t)src->pixels & (d->mode == VR_EA ? 15u : 3u)) == 0, "src pixels are misaligned");
    const uint64_t out_row = (uint64_t)d->width * 4;
    const uint64_t opitch = out_pitch_bytes ? out_pitch_bytes : out_row;
    VR_REQUIRE(opitch >= out_row && opitch % 4 == 0 && ((uintptr_t)out & 3u) == 0, "bad out pitch / alignment");
    VR_REQUIRE(out_location == VR_DEVICE || out_location == VR_HOST_PINNED, "bad out_location %u", out_location);
    EncodeK P;
    P.scale = P.bias = 0.0f;
    for (int c = 0; c < 3; ++c) {
        P.bg[c] = d->background[c];
        VR_REQUIRE(d->mode != VR_EA || (std::isfinite(P.bg[c]) && P.bg[c] >= 0.0f && P.bg[c] <= 1.0f), "background must be in [0,1]");
    }
    if (d->mode == VR_MIP) {
        VR_REQUIRE(std::isfinite(d->vmin) && std::isfinite(d->vmax) && d->vmax > d->vmin, "need finite vmin < vmax (got %g, %g)", d->vmin, d->vmax);
        P.scale = 1.0f / (d->vmax - d->vmin);                       // C.4 / C.14, float32
        P.bias = -d->vmin * P.scale;
    }
    VR_CUDA(cudaSetDevice(v->device));
    cudaStream_t st = (cudaStream_t)stream;
    v->stats.kernel_launches = 0; v->stats.h2d_bytes = 0; v->stats.d2h_bytes = 0;
    unsigned int *dst = reinterpret_cast<unsigned int *>(out);
    long long dst_pitch_w = (long long)(opitch / 4);
    if (out_location == VR_HOST_PINNED) {
        vr_status rc = v->host_frame.reserve((size_t)d->width * d->height);
        if (rc != VR_OK) return rc;
        dst = v->host_frame.p; dst_pitch_w = d->width;
    }
    launch_encode_rgba8((int)d->mode, src->pixels, (long long)(pitch / 4), (int)d->width, (int)d->height, P, dst, dst_pitch_w, st);
    v->stats.kernel_launches = 1;
    VR_CUDA(cudaGetLastError());
    if (out_location == VR_HOST_PINNED) {
        if (opitch == out_row) VR_CUDA(cudaMemcpyAsync(out, dst, out_row * d->height, cudaMemcpyDeviceToHost, st));
        else VR_CUDA(cudaMemcpy2DAsync(out, opitch, dst, out_row, out_row, d->height, cudaMemcpyDeviceToHost, st));
        v->stats.d2h_bytes = out_row * d->height;
    }
    v->stats.total_kernel_launches += 1;
    return VR_OK;
}

VR_API vr_status vr_set_option(vr_volume *v, uint32_t option, int64_t value)
{
    g_err[0] = 0;
    VR_REQUIRE(v, "vr_set_option: NULL handle");
    switch (option) {
    case VR_OPT_RENDER_PATH:
        VR_REQUIRE(value == 0 || value == 1, "VR_OPT_RENDER_PATH: 0 auto (lane-mapped), 1 ray-major tiles (got %lld)", (long long)value);
        v->opt_path = (int)value; return VR_OK;
    case VR_OPT_ZFAST_COPY:
        VR_REQUIRE(value == 0 || value == 1, "VR_OPT_ZFAST_COPY: 0 never, 1 when needed and it fits (got %lld)", (long long)value);
        v->opt_zcopy = (int)value; return VR_OK;
    case VR_OPT_LANE_LAG:
        VR_REQUIRE(value >= 0 && value <= 1024, "VR_OPT_LANE_LAG: 0..1024 base planes (got %lld)", (long long)value);
        v->opt_lag = (int)value; return VR_OK;
    case VR_OPT_ROW_LOADS:
        VR_REQUIRE(value >= 0 && value <= 2, "VR_OPT_ROW_LOADS: 0 scalar, 1 one 16-byte load per row, 2 auto (got %lld)", (long long)value);
        v->opt_quad = (int)value; return VR_OK;
    case VR_OPT_TILE_SHEAR:
        VR_REQUIRE(value == 0 || value == 1, "VR_OPT_TILE_SHEAR: 0 one shear per frame, 1 one per tile (got %lld)", (long long)value);
        v->opt_tile_shear = (int)value; return VR_OK;
    case VR_OPT_FORCE_WIDE:
        VR_REQUIRE(value == 0 || value == 1, "VR_OPT_FORCE_WIDE: 0 or 1 (got %lld)", (long long)value);
        v->opt_wide = (int)value; return VR_OK;
    case VR_OPT_EMPTY_SKIP:
        VR_REQUIRE(value == 0 || value == 1, "VR_OPT_EMPTY_SKIP: 0 never, 1 when the transfer function has empty intervals (got %lld)", (long long)value);
        v->opt_skip = (int)value; return VR_OK;
    default:
        set_error("unknown option %u", option); return VR_ERR_INVALID_ARG;
    }
}

VR_API vr_status vr_get_stats(vr_volume *v, vr_stats *s)
{
    g_err[0] = 0;
    VR_REQUIRE(v && s, "vr_get_stats: NULL argument");
    VR_REQUIRE(s->struct_size == sizeof(vr_stats), "vr_stats.struct_size %u != %zu", s->struct_size, sizeof(vr_stats));
    *s = v->stats;
    s->empty_cells = v->h_nskip ? (uint64_t)*v->h_nskip : 0;          // as of the last completed flag pass
    return VR_OK;
}

}  // extern "C"
