// vr_reduce.cu — global min/max (+ non-finite count) and the 256-bin (<= 4096-bin) histogram.
// SURVEY.md §8(a) rows A1, A2; arithmetic = reading C.8: PAPER.md:L14, L66.
//
// Both passes are HBM-bound streams of the cube (4 B/voxel each).  Design:
//   * persistent grid (SMs x 2 CTAs of 512 threads), grid-stride 16-byte loads that bypass L1
//     (ld.global.nc.L1::no_allocate), four loads in flight per thread;
//   * min/max: per-thread registers -> warp shuffles -> one pair of atomics per CTA on an
//     order-preserving uint encoding, so the result is exact and order-independent;
//   * histogram: privatised shared-memory counters laid out [bin][replica] with replica =
//     lane % R, so that the lanes of a warp that hit the same (popular, central-noise) bin land
//     in different banks and different addresses — the same-address serialisation the paper
//     warns about (footnote 3) never happens inside a warp instruction.
//     Counters are uint32 per CTA (a CTA sees < 2^32 voxels) and are merged into the global
//     uint64 counts with one atomic per non-empty bin per CTA.
#include <float.h>

#include "vr_internal.h"
#include "vr_sweep.cuh"

namespace vr {

namespace {

constexpr int kThreads = kSweepThreads;
constexpr int kHistSmemWords = 8192;          // 32 KB of uint32 counters

struct Acc {                                   // per-thread running state
    float mn, mx;
    unsigned int nonfinite, below, above;
};

struct HistCtx {
    unsigned int *h;                           // shared counters [bin * R + replica]
    float lo, hi, scale;
    int nbins, R, rep;
};

template <bool MINMAX, bool HIST>
__device__ __forceinline__ void visit(float v, Acc &a, const HistCtx &hc)
{
    const bool fin = fabsf(v) <= FLT_MAX;      // false for NaN and +-Inf (C.8: isfinite)
    if (MINMAX) {
        if (fin) { a.mn = fminf(a.mn, v); a.mx = fmaxf(a.mx, v); }
        else a.nonfinite++;
    }
    if (HIST) {
        if (fin) {
            if (v < hc.lo) a.below++;
            else if (v > hc.hi) a.above++;
            else {
                const float t = __fmul_rn(__fsub_rn(v, hc.lo), hc.scale);    // sub then mul, no FMA (S23)
                const int b = min(__float2int_rz(t), hc.nbins - 1);
                atomicAdd(&hc.h[b * hc.R + hc.rep], 1u);
            }
        }
    }
}

template <bool MINMAX, bool HIST>
__device__ __forceinline__ void finish_block(Acc a, const HistCtx &hc, SummaryScratch *s)
{
    __shared__ float s_mn[kThreads / 32], s_mx[kThreads / 32];
    __shared__ unsigned int s_cnt[3][kThreads / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        if (MINMAX) {
            a.mn = fminf(a.mn, __shfl_xor_sync(0xffffffffu, a.mn, o));
            a.mx = fmaxf(a.mx, __shfl_xor_sync(0xffffffffu, a.mx, o));
            a.nonfinite += __shfl_xor_sync(0xffffffffu, a.nonfinite, o);
        }
        if (HIST) {
            a.below += __shfl_xor_sync(0xffffffffu, a.below, o);
            a.above += __shfl_xor_sync(0xffffffffu, a.above, o);
        }
    }
    if (lane == 0) {
        s_mn[warp] = a.mn; s_mx[warp] = a.mx;
        s_cnt[0][warp] = a.nonfinite; s_cnt[1][warp] = a.below; s_cnt[2][warp] = a.above;
    }
    __syncthreads();                           // also orders the shared histogram atomics
    if (threadIdx.x == 0) {
        float mn = CUDART_INF_F, mx = -CUDART_INF_F;
        unsigned long long c0 = 0, c1 = 0, c2 = 0;
        for (int w = 0; w < kThreads / 32; ++w) {
            mn = fminf(mn, s_mn[w]); mx = fmaxf(mx, s_mx[w]);
            c0 += s_cnt[0][w]; c1 += s_cnt[1][w]; c2 += s_cnt[2][w];
        }
        if (MINMAX) {
            atomicMin(&s->enc_min, enc_f(mn));
            atomicMax(&s->enc_max, enc_f(mx));
            if (c0) atomicAdd(&s->n_nonfinite, c0);
        }
        if (HIST) {
            if (c1) atomicAdd(&s->n_below, c1);
            if (c2) atomicAdd(&s->n_above, c2);
        }
    }
    if (HIST) {
        for (int b = threadIdx.x; b < hc.nbins; b += kThreads) {
            unsigned int sum = 0;
            for (int r = 0; r < hc.R; ++r) sum += hc.h[b * hc.R + ((r + b) & (hc.R - 1))];
            if (sum) atomicAdd(&s->counts[b], (unsigned long long)sum);
        }
    }
}

template <bool HIST>
__device__ __forceinline__ HistCtx hist_begin(const SummaryScratch *s, uint32_t nbins, unsigned int *smem)
{
    HistCtx hc;
    hc.h = smem; hc.nbins = (int)nbins; hc.lo = hc.hi = hc.scale = 0.0f;
    int R = 32;
    while ((int)nbins * R > kHistSmemWords) R >>= 1;
    hc.R = R; hc.rep = threadIdx.x & (R - 1);
    if (HIST) {
        hc.lo = s->lo; hc.hi = s->hi; hc.scale = s->scale_h;
        for (int i = threadIdx.x; i < (int)nbins * R; i += kThreads) smem[i] = 0u;
        __syncthreads();
    }
    return hc;
}

// flat array of n voxels, 16-byte aligned base
template <bool MINMAX, bool HIST>
__global__ void __launch_bounds__(kThreads, 2)
k_reduce_flat(const float *__restrict__ v, unsigned long long n, uint32_t nbins, SummaryScratch *s)
{
    VR_DYN_SHARED(unsigned int, smem);
    const HistCtx hc = hist_begin<HIST>(s, nbins, smem);
    Acc a = { CUDART_INF_F, -CUDART_INF_F, 0u, 0u, 0u };
    sweep_flat(v, n, [&](float x) { visit<MINMAX, HIST>(x, a, hc); });
    finish_block<MINMAX, HIST>(a, hc, s);
}

// a box of ex*ey*ez voxels inside a strided array (bricked layouts: the halo is outside the box)
template <bool MINMAX, bool HIST>
__global__ void __launch_bounds__(kThreads, 2)
k_reduce_box(BoxK b, uint32_t nbins, SummaryScratch *s)
{
    VR_DYN_SHARED(unsigned int, smem);
    const HistCtx hc = hist_begin<HIST>(s, nbins, smem);
    Acc a = { CUDART_INF_F, -CUDART_INF_F, 0u, 0u, 0u };
    sweep_box(b, [&](float x) { visit<MINMAX, HIST>(x, a, hc); });
    finish_block<MINMAX, HIST>(a, hc, s);
}

__global__ void k_summary_reset(SummaryScratch *s)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < 4096) s->counts[i] = 0ull;
    if (i == 0) {
        s->enc_min = enc_f(CUDART_INF_F); s->enc_max = enc_f(-CUDART_INF_F);
        s->lo = s->hi = s->scale_h = 0.0f;
        s->n_nonfinite = s->n_below = s->n_above = 0ull;
    }
}

__global__ void k_summary_range(SummaryScratch *s, int range_mode, float lo, float hi, uint32_t nbins)
{
    if (range_mode == 0) { lo = dec_f(s->enc_min); hi = dec_f(s->enc_max); }
    s->lo = lo; s->hi = hi;
    s->scale_h = (hi == lo) ? 0.0f : __fdiv_rn((float)nbins, __fsub_rn(hi, lo));    // C.8
}

__global__ void k_summary_finish(const SummaryScratch *s, uint32_t nbins, vr_summary *out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < (int)nbins) out->counts[i] = s->counts[i];
    if (i == 0) {
        out->vmin = dec_f(s->enc_min); out->vmax = dec_f(s->enc_max);
        out->n_nonfinite = s->n_nonfinite; out->n_below = s->n_below; out->n_above = s->n_above;
    }
}

constexpr size_t kHistSmemBytes = kHistSmemWords * sizeof(unsigned int);

}  // namespace

void launch_summary_reset(SummaryScratch *s, cudaStream_t st) { vr_launch(k_summary_reset, 16, 256, 0, st, s); }

void launch_minmax_flat(const float *v, unsigned long long n, SummaryScratch *s, int grid, cudaStream_t st)
{
    vr_launch(k_reduce_flat<true, false>, grid, kThreads, 0, st, v, n, 0u, s);
}
void launch_minmax_box(BoxK b, SummaryScratch *s, int grid, cudaStream_t st)
{
    vr_launch(k_reduce_box<true, false>, grid, kThreads, 0, st, b, 0u, s);
}
void launch_summary_range(SummaryScratch *s, int range_mode, float lo, float hi, uint32_t nbins, cudaStream_t st)
{
    vr_launch(k_summary_range, 1, 1, 0, st, s, range_mode, lo, hi, nbins);
}
void launch_hist_flat(const float *v, unsigned long long n, uint32_t nbins, SummaryScratch *s, int grid, cudaStream_t st)
{
    vr_launch(k_reduce_flat<false, true>, grid, kThreads, kHistSmemBytes, st, v, n, nbins, s);
}
void launch_hist_box(BoxK b, uint32_t nbins, SummaryScratch *s, int grid, cudaStream_t st)
{
    vr_launch(k_reduce_box<false, true>, grid, kThreads, kHistSmemBytes, st, b, nbins, s);
}
void launch_minmax_hist_flat(const float *v, unsigned long long n, uint32_t nbins, SummaryScratch *s, int grid,
                             cudaStream_t st)
{
    vr_launch(k_reduce_flat<true, true>, grid, kThreads, kHistSmemBytes, st, v, n, nbins, s);
}
void launch_minmax_hist_box(BoxK b, uint32_t nbins, SummaryScratch *s, int grid, cudaStream_t st)
{
    vr_launch(k_reduce_box<true, true>, grid, kThreads, kHistSmemBytes, st, b, nbins, s);
}
void launch_summary_finish(const SummaryScratch *s, uint32_t nbins, vr_summary *out, cudaStream_t st)
{
    vr_launch(k_summary_finish, (nbins + 255) / 256, 256, 0, st, s, nbins, out);
}

}  // namespace vr
