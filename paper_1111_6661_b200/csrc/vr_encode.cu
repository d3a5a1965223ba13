// vr_encode.cu — 8-bit RGBA frame for delivery to a thin client: the headless end of the paper's "server-side
// rendering back-end" whose viewer only displays results (reading S40 / C.14 of
// DESIGN.md §3).  No graphics API: the frame is a byte buffer in device or pinned host memory.
//   EA  : x_c = fmaf(1 - A, bg_c, C_c) (the premultiplied image over an opaque background), clamped to [0,1]
//         (NaN -> 0), byte = round-half-even(x_c * 255); alpha byte 255.
//   MIP : u = sat(fmaf(m, scale, bias)), scale = 1/(vmax - vmin), bias = -vmin * scale; byte = round-half-even(u * 255)
//         in r, g, b; a miss (-inf) gives 0; alpha byte 255.
// HBM-bound: 16 (EA) or 4 (MIP) bytes read and 4 written per pixel; one thread per pixel, one 4-byte store.
#include "vr_internal.h"

namespace vr {

namespace {

__device__ __forceinline__ unsigned int byte_of_unit(float x)
{
    return (unsigned int)__float2int_rn(__fmul_rn(__saturatef(x), 255.0f));     // __saturatef: NaN -> 0
}

template <int MODE>
__global__ void __launch_bounds__(256) k_encode_rgba8(const float *__restrict__ img, long long pitch_f, int W, int H,
                                                      EncodeK P, unsigned int *__restrict__ out, long long out_pitch_w)
{
    const int i = blockIdx.x * 32 + (threadIdx.x & 31), j = blockIdx.y * 8 + (threadIdx.x >> 5);
    if (i >= W || j >= H) return;
    unsigned int r, g, b;
    if (MODE == VR_EA) {
        const float4 p = __ldg(reinterpret_cast<const float4 *>(img + (long long)j * pitch_f) + i);
        const float w = __fsub_rn(1.0f, p.w);
        r = byte_of_unit(__fmaf_rn(w, P.bg[0], p.x));
        g = byte_of_unit(__fmaf_rn(w, P.bg[1], p.y));
        b = byte_of_unit(__fmaf_rn(w, P.bg[2], p.z));
    } else
        r = g = b = byte_of_unit(__fmaf_rn(__ldg(img + (long long)j * pitch_f + i), P.scale, P.bias));
    out[(long long)j * out_pitch_w + i] = r | (g << 8) | (b << 16) | 0xff000000u;
}

}  // namespace

void launch_encode_rgba8(int mode, const float *img, long long pitch_f, int W, int H, const EncodeK &P, unsigned int *out,
                         long long out_pitch_w, cudaStream_t st)
{
    const dim3 g((W + 31) / 32, (H + 7) / 8);
    if (mode == VR_MIP) vr_launch(k_encode_rgba8<VR_MIP>, g, 256, 0, st, img, pitch_f, W, H, P, out, out_pitch_w);
    else vr_launch(k_encode_rgba8<VR_EA>, g, 256, 0, st, img, pitch_f, W, H, P, out, out_pitch_w);
}

}  // namespace vr
