// blur.cu -- the Gaussian pre-filter F0 / A6 (config 3) as a separable spatial stencil.
//
// Definition (F0; the form of the MTF model PAPER.md:184, standing in for G{l} of Eq. 5):
//   h_f = Re F^-1{ F{h} Ghat },  Ghat(kx, ky) = exp(-2 pi^2 sigma^2 ((kx/Nx)^2 + (ky/Ny)^2)),
// i.e. the circular convolution of h with g_y (x) g_x, g[n] = (1/N) sum_k Ghat(k) cos(2 pi k n / N).  For the small
// sigma of a lithography kernel g is negligible beyond |n| = R = ceil(6 sigma) (a relative tail of 2e-9), so two
// streaming passes over the fp32 plane (rows, then columns; 4 bytes in + 4 bytes out per point each) replace the
// ten complex FFT passes of the spectral form (104 bytes per point).  The taps are the definition's own inverse DFT,
// summed in fp64 on the host (plan.cu), so the only difference from the spectral result is the dropped tail.
// Self-adjoint (g even), so A6 runs the same two kernels on dL/dh.
#include "dop_internal.h"

namespace dop {

struct BlurTaps { float w[2 * 24 + 1]; }; // w[RT + d], d = -RT .. RT (zeros beyond the true radius)

// rows: thread = 8 adjacent outputs of one row; its window (8 + 2 RT floats) comes in as aligned float4 chunks with
// circular wrap (nx % 8 == 0, RT % 4 == 0), the taps are constant-bank operands of the FMAs.
template <int RT>
__global__ void __launch_bounds__(256) blur_x_kernel(const float* __restrict__ src, float* __restrict__ dst, long long ny,
                                                     long long nx, const __grid_constant__ BlurTaps taps)
{
    const long long chunks = nx / 8;
    const long long t = (long long)blockIdx.x * 256 + threadIdx.x;
    if (t >= ny * chunks) return;
    const long long row = t / chunks, x0 = (t - row * chunks) * 8;
    const float* __restrict__ r = src + row * nx;
    constexpr int NW = 8 + 2 * RT;
    float win[NW];
#pragma unroll
    for (int q = 0; q < NW / 4; ++q) {
        long long x = x0 - RT + 4 * q;
        x = x < 0 ? x + nx : (x >= nx ? x - nx : x);
        const float4 v = *reinterpret_cast<const float4*>(r + x);
        win[4 * q] = v.x; win[4 * q + 1] = v.y; win[4 * q + 2] = v.z; win[4 * q + 3] = v.w;
    }
    float acc[8];
#pragma unroll
    for (int o = 0; o < 8; ++o) {
        float a = 0.0f;
#pragma unroll
        for (int d = 0; d <= 2 * RT; ++d) a = fmaf(taps.w[d], win[o + d], a);
        acc[o] = a;
    }
    float4* out = reinterpret_cast<float4*>(dst + row * nx + x0);
    out[0] = make_float4(acc[0], acc[1], acc[2], acc[3]);
    out[1] = make_float4(acc[4], acc[5], acc[6], acc[7]);
}

// columns: thread = 32 output rows of one column (lanes over adjacent columns: coalesced rows), sliding over the
// 32 + 2 RT input rows with circular wrap (ny % 32 == 0).
template <int RT>
__global__ void __launch_bounds__(128) blur_y_kernel(const float* __restrict__ src, float* __restrict__ dst, long long ny,
                                                     long long nx, const __grid_constant__ BlurTaps taps)
{
    const long long x = (long long)blockIdx.x * 128 + threadIdx.x;
    if (x >= nx) return;
    const long long y0 = (long long)blockIdx.y * 32;
    float acc[32];
#pragma unroll
    for (int o = 0; o < 32; ++o) acc[o] = 0.0f;
#pragma unroll
    for (int d = 0; d < 32 + 2 * RT; ++d) {
        long long y = y0 - RT + d;
        y = y < 0 ? y + ny : (y >= ny ? y - ny : y);
        const float v = __ldg(src + y * nx + x);
#pragma unroll
        for (int o = 0; o < 32; ++o)
            if (d - o >= 0 && d - o <= 2 * RT) acc[o] = fmaf(taps.w[d - o], v, acc[o]);
    }
#pragma unroll
    for (int o = 0; o < 32; ++o) dst[(y0 + o) * nx + x] = acc[o];
}

template <int RT>
static cudaError_t launch_blur_rt(const float* src, float* tmp, float* dst, long long ny, long long nx, const BlurTaps& tx,
                                  const BlurTaps& ty, cudaStream_t st, cudaEvent_t mid_stop, cudaEvent_t mid_start)
{
    const long long threads = ny * (nx / 8);
    blur_x_kernel<RT><<<(unsigned)((threads + 255) / 256), 256, 0, st>>>(src, tmp, ny, nx, tx);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (mid_stop != nullptr) cudaEventRecord(mid_stop, st);
    if (mid_start != nullptr) cudaEventRecord(mid_start, st);
    dim3 grid((unsigned)((nx + 127) / 128), (unsigned)(ny / 32));
    blur_y_kernel<RT><<<grid, 128, 0, st>>>(tmp, dst, ny, nx, ty);
    return cudaGetLastError();
}

// src -> (rows) tmp -> (columns) dst; tmp may not alias src or dst, dst may alias src.  radius <= 24 taps per side.
cudaError_t launch_blur(const float* src, float* tmp, float* dst, long long ny, long long nx, int radius, const float* wx,
                        const float* wy, cudaStream_t st, cudaEvent_t mid_stop, cudaEvent_t mid_start)
{
    if (radius < 1 || radius > 24 || nx % 8 != 0 || ny % 32 != 0) return cudaErrorInvalidValue;
    const int rt = (radius + 3) / 4 * 4;
    BlurTaps tx, ty;
    for (int i = 0; i < 49; ++i) tx.w[i] = ty.w[i] = 0.0f;
    for (int d = -radius; d <= radius; ++d) { // wx / wy: [0 .. radius], even
        tx.w[rt + d] = wx[d < 0 ? -d : d];
        ty.w[rt + d] = wy[d < 0 ? -d : d];
    }
    switch (rt) {
    case 4: return launch_blur_rt<4>(src, tmp, dst, ny, nx, tx, ty, st, mid_stop, mid_start);
    case 8: return launch_blur_rt<8>(src, tmp, dst, ny, nx, tx, ty, st, mid_stop, mid_start);
    case 12: return launch_blur_rt<12>(src, tmp, dst, ny, nx, tx, ty, st, mid_stop, mid_start);
    case 16: return launch_blur_rt<16>(src, tmp, dst, ny, nx, tx, ty, st, mid_stop, mid_start);
    case 20: return launch_blur_rt<20>(src, tmp, dst, ny, nx, tx, ty, st, mid_stop, mid_start);
    case 24: return launch_blur_rt<24>(src, tmp, dst, ny, nx, tx, ty, st, mid_stop, mid_start);
    }
    return cudaErrorInvalidValue;
}

} // namespace dop
