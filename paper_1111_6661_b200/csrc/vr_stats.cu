// vr_stats.cu — the multi-pass "global view" statistics the paper names next to min/max: mean, standard
// deviation and median of the whole cube ("global view data analysis tasks ... median and
// standard deviation", which "require the whole cube" and several passes; readings
// S35-S37 of DESIGN.md §3).
//
//   pass 0   n = #finite, sum(v) in double, min / max as order-preserving keys           -> mean = sum / n
//   pass 1   sum((v - mean)^2) in double                                                 -> stddev = sqrt(. / n)
//            + first radix-select pass
//   pass 2-4 radix select of the LOWER median: the element of rank floor((n-1)/2) of the finite voxels in
//            IEEE totalOrder.  State = a key interval [klo, khi] that contains the answer and the rank of
//            the answer inside it; a pass counts the candidates into 256 bins of width 2^shift keys and the
//            one-thread kernel between passes narrows the interval to the bin that holds the rank.  The key
//            space has 32 bits and every pass resolves 8 of them, so 4 passes always suffice; once the
//            interval is a single key the remaining passes return at once.  Exact: the result is a data value.
// Every pass is the HBM-bound stream of vr_sweep.cuh (4 B/voxel); nothing is read back between passes.
// Double sums are deterministic for a given grid: Kahan-compensated per thread, a fixed shuffle tree per
// warp, warps in order per CTA, one slot per CTA, CTAs in order (Neumaier) in the one-thread kernel.
// Shared counters of the select passes: [bin][lane] uint32 (32 KB): no two lanes of a warp ever share an
// address or a bank (the same-address serialisation PAPER.md:L40 warns about cannot happen inside a warp).
#include <float.h>

#include "vr_internal.h"
#include "vr_sweep.cuh"

namespace vr {

namespace {

constexpr int kThreads = kSweepThreads;
constexpr int kWarps = kThreads / 32;
constexpr size_t kSelSmemBytes = 256 * 32 * sizeof(unsigned int);

__device__ __forceinline__ bool finite_f(float v) { return fabsf(v) <= FLT_MAX; }

struct Kahan {
    double s = 0.0, c = 0.0;
    __device__ __forceinline__ void add(double x)
    {
        const double y = x - c, t = s + y;
        c = (t - s) - y;
        s = t;
    }
    __device__ __forceinline__ double value() const { return s - c; }
};

// sum of one double per thread over the CTA in a fixed order; valid in thread 0
__device__ __forceinline__ double cta_sum(double x)
{
    __shared__ double s_part[kWarps];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    if ((threadIdx.x & 31) == 0) s_part[threadIdx.x >> 5] = x;
    __syncthreads();
    double r = 0.0;
    if (threadIdx.x == 0)
        for (int w = 0; w < kWarps; ++w) r += s_part[w];
    __syncthreads();
    return r;
}

__device__ __forceinline__ unsigned long long cta_count(unsigned int x)
{
    __shared__ unsigned int s_cnt[kWarps];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    if ((threadIdx.x & 31) == 0) s_cnt[threadIdx.x >> 5] = x;
    __syncthreads();
    unsigned long long r = 0;
    if (threadIdx.x == 0)
        for (int w = 0; w < kWarps; ++w) r += s_cnt[w];
    __syncthreads();
    return r;
}

// adds x to this CTA's slot (Kahan across the launches of one call, which are stream-ordered: only CTA
// blockIdx.x of each launch touches slot blockIdx.x)
__device__ __forceinline__ void slot_add(StatScratch *s, double x)
{
    const double y = x - s->part_c[blockIdx.x], t = s->part[blockIdx.x] + y;
    s->part_c[blockIdx.x] = (t - s->part[blockIdx.x]) - y;
    s->part[blockIdx.x] = t;
}

// ---------------------------------------------------------------- pass 0: count, sum, key range
struct Pass0 {
    Kahan sum;
    unsigned int n = 0, bad = 0, kmin = 0xffffffffu, kmax = 0u;
    __device__ __forceinline__ void operator()(float v)
    {
        if (finite_f(v)) {
            ++n;
            sum.add((double)v);
            const unsigned int k = enc_f(v);
            kmin = min(kmin, k); kmax = max(kmax, k);
        } else ++bad;
    }
};

__device__ __forceinline__ void finish_pass0(Pass0 &p, StatScratch *s)
{
    const double sum = cta_sum(p.sum.value());
    const unsigned long long n = cta_count(p.n), bad = cta_count(p.bad);
    const unsigned int kmin = __reduce_min_sync(0xffffffffu, p.kmin), kmax = __reduce_max_sync(0xffffffffu, p.kmax);
    if ((threadIdx.x & 31) == 0) { atomicMin(&s->klo, kmin); atomicMax(&s->khi, kmax); }
    if (threadIdx.x == 0) {
        slot_add(s, sum);
        s->part_n[blockIdx.x] += n;
        if (bad) atomicAdd(&s->n_nonfinite, bad);
    }
}

__global__ void __launch_bounds__(kThreads, 2) k_stat0_flat(const float *__restrict__ v, unsigned long long n, StatScratch *s)
{
    Pass0 p;
    sweep_flat(v, n, p);
    finish_pass0(p, s);
}
__global__ void __launch_bounds__(kThreads, 2) k_stat0_box(BoxK b, StatScratch *s)
{
    Pass0 p;
    sweep_box(b, p);
    finish_pass0(p, s);
}

// ---------------------------------------------------------------- passes 1-4: squared deviations and/or select
template <bool DEV>
struct PassSel {
    Kahan m2;
    double mean;
    unsigned int klo, span, shift;
    bool select;                                   // false: the median is already known (moments only)
    unsigned int *h;                               // shared counters [bin * 32 + lane]
    __device__ __forceinline__ void operator()(float v)
    {
        if (!finite_f(v)) return;
        if (DEV) { const double d = (double)v - mean; m2.add(d * d); }
        const unsigned int r = enc_f(v) - klo;     // unsigned: keys below klo wrap to huge values
        if (select && r <= span) atomicAdd(&h[(r >> shift) * 32u + (threadIdx.x & 31u)], 1u);
    }
};

template <bool DEV>
__device__ __forceinline__ bool begin_sel(PassSel<DEV> &p, const StatScratch *s, unsigned int *smem)
{
    if (s->done && !DEV) return false;
    p.mean = s->mean; p.klo = s->klo; p.span = s->khi - s->klo; p.shift = s->shift; p.h = smem;
    p.select = !s->done;
    for (int i = threadIdx.x; i < 256 * 32; i += kThreads) smem[i] = 0u;
    __syncthreads();
    return true;
}

template <bool DEV>
__device__ __forceinline__ void finish_sel(PassSel<DEV> &p, StatScratch *s)
{
    if (DEV) {
        const double m2 = cta_sum(p.m2.value());
        if (threadIdx.x == 0) slot_add(s, m2);
    }
    __syncthreads();                               // orders the shared atomics before the merge
    if (s->done) return;
    for (int b = threadIdx.x; b < 256; b += kThreads) {
        unsigned int sum = 0;
        for (int r = 0; r < 32; ++r) sum += p.h[b * 32 + ((r + b) & 31)];
        if (sum) atomicAdd(&s->hist[b], (unsigned long long)sum);
    }
}

template <bool DEV>
__global__ void __launch_bounds__(kThreads, 2) k_stat_sel_flat(const float *__restrict__ v, unsigned long long n, StatScratch *s)
{
    VR_DYN_SHARED(unsigned int, smem);
    PassSel<DEV> p;
    if (!begin_sel(p, s, smem)) return;
    sweep_flat(v, n, p);
    finish_sel(p, s);
}
template <bool DEV>
__global__ void __launch_bounds__(kThreads, 2) k_stat_sel_box(BoxK b, StatScratch *s)
{
    VR_DYN_SHARED(unsigned int, smem);
    PassSel<DEV> p;
    if (!begin_sel(p, s, smem)) return;
    sweep_box(b, p);
    finish_sel(p, s);
}

// ---------------------------------------------------------------- one-thread kernels between the passes
__device__ __forceinline__ unsigned int bits_of(unsigned int x) { return x ? 32u - (unsigned int)__clz((int)x) : 0u; }

__device__ __forceinline__ double ordered_sum(const double *part, const double *part_c, int n)     // Neumaier, slots in order
{
    double s = 0.0, c = 0.0;
    for (int i = 0; i < n; ++i) {
        const double x = part[i] - part_c[i], t = s + x;
        c += fabs(s) >= fabs(x) ? (s - t) + x : (x - t) + s;
        s = t;
    }
    return s + c;
}

__global__ void k_stat_reset(StatScratch *s)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < kStatMaxGrid) { s->part[i] = s->part_c[i] = 0.0; s->part_n[i] = 0ull; }
    if (i < 256) s->hist[i] = 0ull;
    if (i == 0) {
        s->klo = 0xffffffffu; s->khi = 0u; s->shift = 0u; s->done = 0u;
        s->n_finite = s->n_nonfinite = s->rank = 0ull;
        s->mean = s->m2 = s->stddev = 0.0;
    }
}

// after pass `pass` (0..4)
__global__ void k_stat_step(StatScratch *s, int pass)
{
    if (pass == 0) {
        unsigned long long n = 0;
        for (int i = 0; i < kStatMaxGrid; ++i) n += s->part_n[i];
        s->n_finite = n;
        if (n == 0) { s->mean = s->stddev = (double)CUDART_NAN_F; s->done = 1u; }
        else {
            s->mean = ordered_sum(s->part, s->part_c, kStatMaxGrid) / (double)n;
            s->rank = (n - 1) / 2;
            s->done = s->klo == s->khi ? 1u : 0u;
        }
        for (int i = 0; i < kStatMaxGrid; ++i) s->part[i] = s->part_c[i] = 0.0;
    } else {
        if (pass == 1 && s->n_finite) s->stddev = sqrt(ordered_sum(s->part, s->part_c, kStatMaxGrid) / (double)s->n_finite);
        if (!s->done) {
            unsigned long long cum = 0;
            unsigned int b = 0;
            for (; b < 255; ++b) {
                if (cum + s->hist[b] > s->rank) break;
                cum += s->hist[b];
            }
            s->rank -= cum;
            const unsigned long long lo = (unsigned long long)s->klo + ((unsigned long long)b << s->shift);
            const unsigned long long hi = lo + ((1ull << s->shift) - 1ull);
            s->klo = (unsigned int)lo;
            s->khi = hi < (unsigned long long)s->khi ? (unsigned int)hi : s->khi;
            if (s->klo == s->khi || s->shift == 0u) { s->khi = s->klo; s->done = 1u; }
        }
    }
    if (!s->done) {                                 // bin width of the next pass: 256 bins cover [klo, khi]
        const unsigned int nb = bits_of(s->khi - s->klo);
        s->shift = nb > 8u ? nb - 8u : 0u;
    }
    for (int i = 0; i < 256; ++i) s->hist[i] = 0ull;
}

__global__ void k_stat_finish(const StatScratch *s, vr_statistics_result *out)
{
    out->n_finite = s->n_finite; out->n_nonfinite = s->n_nonfinite;
    out->mean = s->mean; out->stddev = s->stddev;
    out->median = s->n_finite ? dec_f(s->klo) : CUDART_NAN_F;
    out->reserved = 0u;
}

}  // namespace

void launch_stat_reset(StatScratch *s, cudaStream_t st) { vr_launch(k_stat_reset, (kStatMaxGrid + 255) / 256, 256, 0, st, s); }
void launch_stat_step(StatScratch *s, int pass, cudaStream_t st) { vr_launch(k_stat_step, 1, 1, 0, st, s, pass); }
void launch_stat_finish(const StatScratch *s, vr_statistics_result *out, cudaStream_t st) { vr_launch(k_stat_finish, 1, 1, 0, st, s, out); }

void launch_stat_pass_flat(int pass, const float *v, unsigned long long n, StatScratch *s, int grid, cudaStream_t st)
{
    if (pass == 0) vr_launch(k_stat0_flat, grid, kThreads, 0, st, v, n, s);
    else if (pass == 1) vr_launch(k_stat_sel_flat<true>, grid, kThreads, kSelSmemBytes, st, v, n, s);
    else vr_launch(k_stat_sel_flat<false>, grid, kThreads, kSelSmemBytes, st, v, n, s);
}

void launch_stat_pass_box(int pass, BoxK b, StatScratch *s, int grid, cudaStream_t st)
{
    if (pass == 0) vr_launch(k_stat0_box, grid, kThreads, 0, st, b, s);
    else if (pass == 1) vr_launch(k_stat_sel_box<true>, grid, kThreads, kSelSmemBytes, st, b, s);
    else vr_launch(k_stat_sel_box<false>, grid, kThreads, kSelSmemBytes, st, b, s);
}

}  // namespace vr
