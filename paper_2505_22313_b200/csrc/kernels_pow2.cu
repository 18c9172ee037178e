// kernels_pow2.cu -- register-blocked tile-pass kernels for power-of-two digits (the fast path).
//
// Same pass semantics as kernels_generic.cu (one CTA = one tile, one read + one write of the
// field, fused pointwise ops; Eq. 1-4, PAPER.md:200 row-column 2-D FFT), same
// slot order, so a plan may mix the two kernels pass by pass.  Here every thread keeps 16 points
// in registers (fft_regs.cuh); global loads / stores go straight from / to registers:
//   column-type tile: 16 adjacent lines x L slots, lanes run over the 16 lines (128-byte segments);
//   row-type tile   : LINES contiguous lines of L points, lanes run over consecutive points.
#include "dop_internal.h"
#include "fft_regs.cuh"

namespace dop {

using fx::P;

// ---- fused pointwise ops on the element at plane offset `off` ---------------------------------
__device__ __forceinline__ float2 load_point(const PassDesc& p, long long off)
{
    if (p.load_op == LD_C64) return p.field[off];
    if (p.load_op == LD_HEIGHT) {
        float2 v;
        float tt = __ldg(p.height + off) * p.phase_coef; // Eq. (1) in turns
        sincospif(2.0f * tt, &v.y, &v.x);                // Eq. (2), E_in = 1
        return v;
    }
    if (p.load_op == LD_SEED) {
        float2 u = p.field[off];
        float g = 2.0f * __ldg(p.plane_in + off);
        return make_float2(g * u.x, g * u.y);
    }
    return make_float2(__ldg(p.plane_in + off), 0.0f);
}

__device__ __forceinline__ void store_point(const PassDesc& p, long long off, float2 v)
{
    if (p.store_op == ST_C64) {
        p.field[off] = v;
    } else if (p.store_op == ST_GRAD || p.store_op == ST_GRAD_ACC) {
        float tt = __ldg(p.height + off) * p.phase_coef;
        float sn, cs;
        sincospif(2.0f * tt, &sn, &cs); // u0 recomputed, not stored
        float g = p.grad_coef * (cs * v.y - sn * v.x); // A5: c Im(conj(u0) g)
        if (p.store_op == ST_GRAD_ACC) g += p.plane_out[off];
        p.plane_out[off] = g;
    } else if (p.store_op == ST_C64_INTENSITY) {
        p.field[off] = v;
        p.plane_out[off] = v.x * v.x + v.y * v.y;
    } else {
        p.plane_out[off] = v.x;
    }
}

// F4 / A3: v *= H (or conj H) / N at (x slot col, y slot row); evanescent bins zeroed.
// a and the phase z sqrt(a) are fp64; sqrt = fp32 rsqrt seed + two
// fp64 Newton steps (full double accuracy, no slow-path DSQRT).
__device__ __forceinline__ float2 apply_h(const PassDesc& p, float2 v, double c_minus_fx2, double fy2)
{
    const double a = c_minus_fx2 - fy2; // (1/lambda^2 - fx^2) - fy^2, the definition's own order
    if (a >= 0.0) {
        double s = 0.0;
        if (a > 0.0) {
            const double y = (double)rsqrtf((float)a);
            const double hy = 0.5 * y;
            s = a * y;
            s = fma(fma(-s, s, a), hy, s);
            s = fma(fma(-s, s, a), hy, s);
        }
        const double turns = p.z * s;
        const float f = (float)(turns - rint(turns)); // fractional turn, |f| <= 0.5
        float sn, cs;
        sincospif(2.0f * f, &sn, &cs);
        const float hr = cs * p.scale, hi = (p.mid_op == MID_H ? sn : -sn) * p.scale;
        return make_float2(fmaf(-v.y, hi, v.x * hr), fmaf(v.x, hi, v.y * hr));
    }
    return make_float2(0.0f, 0.0f);
}

// deterministic CTA reduction of the loss partial (warp shuffle tree, then thread 0 in warp order)
__device__ __forceinline__ void block_loss(const PassDesc& p, double acc, double* red)
{
    for (int d = 16; d > 0; d >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, d);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        const int nw = (blockDim.x + 31) >> 5;
        for (int w = 0; w < nw; ++w) t += red[w];
        p.loss_scratch[blockIdx.x] = t;
    }
}

// ---- the tile-pass kernel -------------------------------------------------------------------
template <int L, bool COL, int LINES>
__global__ void __launch_bounds__(COL ? L : LINES * (L / P)) pow2_kernel(const __grid_constant__ PassDesc p)
{
    using TL = fx::Tile<L, COL>;
    using S = fx::Sched<L>;
    constexpr int T = L / P;
    constexpr int GL = S::NG - 1; // last group
    extern __shared__ float2 s[];
    __shared__ float2 twb_s[COL ? L : 1];
    __shared__ double red[32];

    // ---- which tile (same enumeration as the generic kernel)
    long long t = blockIdx.x;
    const long long cg = t % p.n_cgroups;
    t /= p.n_cgroups;
    const long long m = t % p.n_m;
    const long long o = t / p.n_m;
    const long long c0 = cg * p.nl;
    const int tid = threadIdx.x;
    const int sub = COL ? (tid & 15) : (tid / T); // column in the bundle / line in the tile
    const int tt = COL ? (tid >> 4) : (tid % T);
    const long long es = COL ? p.es : 1;
    const long long tbase = o * p.SO + m * p.SM + (c0 + sub) * p.SCc;
    const int soff = COL ? sub : sub * TL::LINE_ELEMS;
    const float2* __restrict__ tw = p.tw_g;
    const bool twb_tile = COL && p.tw_b != nullptr && p.r_from == 1; // r constant over the tile
    const long long r_lane = c0 + sub;                                // r of this lane otherwise

    if (twb_tile) { // W_{N_j}^{m k(slot)}, the exact fraction reduced in integers
        const long long e = (m * (long long)__ldg(p.pi + tid)) % p.twb_n;
        float sn, cs;
        sincospif(2.0f * (float)e / (float)p.twb_n, &sn, &cs);
        twb_s[tid] = make_float2(cs, -sn);
        __syncthreads();
    }
    auto twb = [&](int slot) -> float2 {
        if (twb_tile) return twb_s[slot];
        return __ldg(p.tw_b + r_lane * (long long)__ldg(p.pi + slot));
    };

    float2 v[P];
    // ---- load (+ prologue op, + conj boundary twiddle before an inverse DFT)
    if (p.fft1_dir > 0) {
#pragma unroll
        for (int i = 0; i < P; ++i) v[i] = load_point(p, tbase + (long long)TL::template slot<0>(tt, i) * es);
    } else {
        if (!COL && p.load_op == LD_C64) {
#pragma unroll
            for (int i = 0; i < P; i += 2) {
                const float4 q = *reinterpret_cast<const float4*>(p.field + tbase + TL::template slot<GL>(tt, i));
                v[i] = make_float2(q.x, q.y);
                v[i + 1] = make_float2(q.z, q.w);
            }
        } else {
#pragma unroll
            for (int i = 0; i < P; ++i) v[i] = load_point(p, tbase + (long long)TL::template slot<GL>(tt, i) * es);
        }
        if (p.tw_b != nullptr) {
#pragma unroll
            for (int i = 0; i < P; ++i) v[i] = fx::cmulc(v[i], twb(TL::template slot<GL>(tt, i)));
        }
    }

    if (p.fft1_dir > 0) TL::template forward<0>(v, s, tt, soff, tw);
    else TL::template inverse<GL>(v, s, tt, soff, tw);

    // ---- middle op
    if (COL && (p.mid_op == MID_H || p.mid_op == MID_HCONJ)) {
        const long long row0 = o * p.row_o + m * p.row_m;
        const double cfx = p.inv_lam2 - __ldg(p.fx2 + c0 + sub);
#pragma unroll
        for (int i = 0; i < P; ++i) {
            const long long row = row0 + (long long)TL::template slot<GL>(tt, i) * p.row_i;
            v[i] = apply_h(p, v[i], cfx, __ldg(p.fy2 + row));
        }
    } else if (COL && p.mid_op == MID_GAUSS) {
        const long long row0 = o * p.row_o + m * p.row_m;
        const float gxs = __ldg(p.gx + c0 + sub) * p.scale;
#pragma unroll
        for (int i = 0; i < P; ++i) {
            const float g = gxs * __ldg(p.gy + row0 + (long long)TL::template slot<GL>(tt, i) * p.row_i);
            v[i] = make_float2(v[i].x * g, v[i].y * g);
        }
    } else if (p.mid_op == MID_LOSS) { // registers hold spatial points in the layout of group 0
        double acc = 0.0;
#pragma unroll
        for (int i = 0; i < P; ++i) {
            const long long off = tbase + (long long)TL::template slot<0>(tt, i) * es;
            const float I = v[i].x * v[i].x + v[i].y * v[i].y; // F6
            const float d = I - __ldg(p.plane_in + off);       // F7
            acc += (double)d * (double)d;
            const float g = p.seed_coef * d;                    // A1: 2 gI = 4 (I - T)/N
            v[i] = make_float2(g * v[i].x, g * v[i].y);
            if (p.write_intensity) p.plane_out[off] = I;
        }
        block_loss(p, acc, red);
    }

    int last_dir = p.fft1_dir;
    if (p.fft2_dir != 0) {
        if (p.fft2_dir > 0) TL::template forward<0>(v, s, tt, soff, tw);
        else TL::template inverse<GL>(v, s, tt, soff, tw);
        last_dir = p.fft2_dir;
    }

    // ---- store (+ boundary twiddle after a forward DFT, + epilogue op)
    if (last_dir > 0) {
        if (p.tw_b != nullptr) {
#pragma unroll
            for (int i = 0; i < P; ++i) v[i] = fx::cmul(v[i], twb(TL::template slot<GL>(tt, i)));
        }
        if (!COL && p.store_op == ST_C64) {
#pragma unroll
            for (int i = 0; i < P; i += 2)
                *reinterpret_cast<float4*>(p.field + tbase + TL::template slot<GL>(tt, i)) =
                    make_float4(v[i].x, v[i].y, v[i + 1].x, v[i + 1].y);
        } else {
#pragma unroll
            for (int i = 0; i < P; ++i) store_point(p, tbase + (long long)TL::template slot<GL>(tt, i) * es, v[i]);
        }
    } else {
#pragma unroll
        for (int i = 0; i < P; ++i) store_point(p, tbase + (long long)TL::template slot<0>(tt, i) * es, v[i]);
    }
}

// ---- host side -------------------------------------------------------------------------------
template <int L, bool COL, int LINES>
static cudaError_t launch_one(const PassDesc& p, cudaStream_t stream)
{
    using TL = fx::Tile<L, COL>;
    constexpr int threads = COL ? L : LINES * (L / P);
    constexpr int smem = (COL ? 1 : LINES) * TL::LINE_ELEMS * (int)sizeof(float2);
    static bool attr_done = false; // per instantiation; the attribute is per device function
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(pow2_kernel<L, COL, LINES>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    const long long ntiles = p.n_cgroups * p.n_m * p.n_o;
    if (ntiles <= 0 || ntiles > 2147483647LL) return cudaErrorInvalidConfiguration;
    pow2_kernel<L, COL, LINES><<<(unsigned)ntiles, threads, smem, stream>>>(p);
    return cudaGetLastError();
}

bool pow2_supported(long long L, bool col_type)
{
    if (L < 16 || (L & (L - 1)) != 0) return false;
    return col_type ? L <= 512 : (L >= 64 && L <= 16384);
}

int pow2_lines(long long L, bool col_type)
{
    if (col_type) return 16;
    return L >= 4096 ? 1 : (int)(4096 / L);
}

cudaError_t launch_tile_pass_pow2(const PassDesc& p, cudaStream_t stream, bool* handled)
{
    *handled = false;
    if (p.tw_g == nullptr || !pow2_supported(p.L, p.col_type != 0)) return cudaSuccess;
    if (p.nl != pow2_lines(p.L, p.col_type != 0) || p.NC % p.nl != 0) return cudaSuccess;
    if (!p.col_type && (p.mid_op == MID_H || p.mid_op == MID_HCONJ || p.mid_op == MID_GAUSS)) return cudaSuccess;
    *handled = true;
    if (p.col_type) {
        switch (p.L) {
        case 16: return launch_one<16, true, 16>(p, stream);
        case 32: return launch_one<32, true, 16>(p, stream);
        case 64: return launch_one<64, true, 16>(p, stream);
        case 128: return launch_one<128, true, 16>(p, stream);
        case 256: return launch_one<256, true, 16>(p, stream);
        case 512: return launch_one<512, true, 16>(p, stream);
        }
    } else {
        switch (p.L) {
        case 64: return launch_one<64, false, 64>(p, stream);
        case 128: return launch_one<128, false, 32>(p, stream);
        case 256: return launch_one<256, false, 16>(p, stream);
        case 512: return launch_one<512, false, 8>(p, stream);
        case 1024: return launch_one<1024, false, 4>(p, stream);
        case 2048: return launch_one<2048, false, 2>(p, stream);
        case 4096: return launch_one<4096, false, 1>(p, stream);
        case 8192: return launch_one<8192, false, 1>(p, stream);
        case 16384: return launch_one<16384, false, 1>(p, stream);
        }
    }
    *handled = false;
    return cudaSuccess;
}

// Twiddle tables of the register-blocked schedule of a digit of length L (layout of fft_regs.cuh:
// group g at twoff(g), entry (k-1) m_g + j = W_{n_g}^{j k}), computed in long double.
std::vector<float2> pow2_group_twiddles(long long L)
{
    std::vector<float2> out;
    int lg = 0;
    while ((1LL << lg) < L) ++lg;
    const int n4 = lg / 2, n2 = lg & 1, nfull = n4 / 2, rlast = ((n4 & 1) ? 4 : 1) * (n2 ? 2 : 1);
    const int ng = nfull + (rlast > 1 ? 1 : 0);
    long long n = L;
    const long double pi = 3.141592653589793238462643383279502884L;
    for (int g = 0; g < ng; ++g) {
        const int R = g < nfull ? 16 : rlast;
        const int RA = R == 2 ? 2 : 4, RB = R / RA;
        (void)RA; (void)RB;
        const long long m = n / R;
        for (int k = 1; k < R; ++k)
            for (long long j = 0; j < m; ++j) {
                long double a = 2.0L * pi * (long double)((j * k) % n) / (long double)n;
                out.push_back(make_float2((float)cosl(a), (float)(-sinl(a))));
            }
        n = m;
    }
    return out;
}

} // namespace dop
