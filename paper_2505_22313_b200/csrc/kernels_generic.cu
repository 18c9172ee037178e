// kernels_generic.cu -- the generic tile-pass kernel: any digit length whose prime factors are <= 127, any
// tile shape, every fused pointwise op.  One CTA = one tile held in shared memory; in-place mixed-radix
// (2/3/4, and direct odd-prime butterflies) decimation-in-frequency forward, mirrored decimation-in-time inverse.
// It is the correctness backbone and the fallback for shapes the specialised kernels
// (kernels_pow2.cu) do not cover.
//
// Math (Eq. 1-4; PAPER.md:200 row-column 2-D FFT):
//   forward digit pass : v <- DFT_L(v) along the line, then v *= T_j      (T_j boundary twiddle)
//   inverse digit pass : v *= conj(T_j), then v <- L * IDFT_L(v)          (1/N folded into H)
#include <atomic>

#include "dop_internal.h"
#include "bfly.cuh"

namespace dop {

// a / d for the small non-negative index arithmetic of this file (a < 2^20, d < 2^14): one multiply by the
// precomputed reciprocal instead of a ~25-instruction integer division.  (a + 1/2) inv is off by less than
// a 2^-22 / d < 1/(2 d), and the fractional part of (a + 1/2)/d is at least 1/(2 d), so the floor is exact.
struct FastDiv {
    int d;
    float inv;
    __device__ __forceinline__ explicit FastDiv(int dd) : d(dd), inv(1.0f / (float)dd) {}
    __device__ __forceinline__ int div(int a) const { return __float2int_rz(((float)a + 0.5f) * inv); }
    __device__ __forceinline__ void divmod(int a, int* q, int* r) const { *q = div(a); *r = a - *q * d; }
};

// One radix-r step for an odd prime r > 3 (the paper's own grids carry 5^2, 5^4 and 67: Table 2):
// the r-point DFT of every butterfly written out directly, with the conjugate symmetry of its kernel halving the
// multiplies.  With a_c = x_c + x_{r-c}, b_c = x_c - x_{r-c} (c = 1 .. (r-1)/2):
//   A_k = sum_c a_c cos(2 pi c k / r),  B_k = sum_c b_c sin(2 pi c k / r),
//   forward:  y_k = x_0 + A_k - i B_k,  y_{r-k} = x_0 + A_k + i B_k      (inverse: the two swapped).
// One work item = one output pair (k, r - k) of one butterfly (k = 0: the plain sum); the step runs out of place
// into the second half of the tile's shared memory (s2) and is copied back, the twiddles W_{n_q}^{j k} ride on
// the outputs (forward) or are applied to the inputs in a pass of their own (inverse), as in the radix-2/3/4 steps.
template <int DIR, bool COL>
__device__ void prime_step(float2* s, float2* s2, const PassDesc& p, int nl_eff, int sl, int se, int r, int nq)
{
    const int L = p.L;
    const float2* __restrict__ wL = p.wL;
    const int m = nq / r, tws = L / nq, twr = L / r, per_line = L / r, h = (r - 1) / 2;
    const int total = nl_eff * L;
    const FastDiv d_nl(nl_eff), d_L(L), d_nq(nq), d_m(m), d_pl(per_line);
    if (DIR < 0 && m > 1) {
        for (int idx = threadIdx.x; idx < total; idx += blockDim.x) {
            int l, i;
            if (COL) d_nl.divmod(idx, &i, &l);
            else d_L.divmod(idx, &l, &i);
            int blk, pos, c, j;
            d_nq.divmod(i, &blk, &pos);
            d_m.divmod(pos, &c, &j);
            if (c > 0 && j > 0) s[l * sl + i * se] = cmulc(s[l * sl + i * se], __ldg(wL + j * c * tws));
        }
        __syncthreads();
    }
    const int items = nl_eff * per_line * (h + 1);
    for (int it = threadIdx.x; it < items; it += blockDim.x) {
        int l, jj, kk;
        int rest, b, j;
        if (COL) { d_nl.divmod(it, &rest, &l); d_pl.divmod(rest, &kk, &jj); }
        else { d_pl.divmod(it, &rest, &jj); d_nl.divmod(rest, &kk, &l); }
        d_m.divmod(jj, &b, &j);
        const int base = l * sl + (b * nq + j) * se, step = m * se;
        const float2 x0 = s[base];
        if (kk == 0) {
            float2 acc = x0;
            for (int c = 1; c < r; ++c) acc = cadd(acc, s[base + c * step]);
            s2[base] = acc;
        } else {
            float2 A = make_float2(0.0f, 0.0f), B = make_float2(0.0f, 0.0f);
            int q = 0;
            for (int c = 1; c <= h; ++c) {
                q += kk;
                if (q >= r) q -= r;
                const float2 w = __ldg(wL + q * twr); // (cos, -sin) of 2 pi c k / r
                const float2 xa = s[base + c * step], xb = s[base + (r - c) * step];
                const float2 sum = cadd(xa, xb), dif = csub(xa, xb);
                A.x = fmaf(sum.x, w.x, A.x);
                A.y = fmaf(sum.y, w.x, A.y);
                B.x = fmaf(dif.x, -w.y, B.x);
                B.y = fmaf(dif.y, -w.y, B.y);
            }
            const float2 t = cadd(x0, A);
            const float2 iB = make_float2(-B.y, B.x);
            float2 yk = DIR > 0 ? csub(t, iB) : cadd(t, iB);
            float2 yr = DIR > 0 ? cadd(t, iB) : csub(t, iB);
            if (DIR > 0 && j > 0) {
                yk = cmul(yk, __ldg(wL + j * kk * tws));
                yr = cmul(yr, __ldg(wL + j * (r - kk) * tws));
            }
            s2[base + kk * step] = yk;
            s2[base + (r - kk) * step] = yr;
        }
    }
    __syncthreads();
    for (int idx = threadIdx.x; idx < total; idx += blockDim.x) s[idx] = s2[idx];
    __syncthreads();
}

// In-place L-point DFT on every line of the tile in shared memory.
// Element (line l, slot i) lives at s[l*sl + i*se].
template <int DIR, bool COL>
__device__ void tile_fft(float2* s, float2* s2, const PassDesc& p, int nl_eff, int sl, int se)
{
    const int L = p.L;
    const float2* __restrict__ wL = p.wL;
    int nq = (DIR > 0) ? L : 1; // current sub-length n_q
    for (int qq = 0; qq < p.n_radix; ++qq) {
        const int q = (DIR > 0) ? qq : (p.n_radix - 1 - qq);
        const int r = p.radix[q];
        if (DIR < 0) nq *= r;       // inverse walks the steps backwards: n_q grows
        if (r > 7) { // larger odd prime factor: direct r-point butterflies, out of place
            prime_step<DIR, COL>(s, s2, p, nl_eff, sl, se, r, nq);
            if (DIR > 0) nq /= r;
            continue;
        }
        const int m = nq / r;       // butterfly stride (slots)
        const int tws = L / nq;     // W_{n_q}^x = wL[x * tws]
        const int per_line = L / r;
        const int nbf = nl_eff * per_line;
        const FastDiv d_nl(nl_eff), d_pl(per_line), d_m(m);
        for (int bf = threadIdx.x; bf < nbf; bf += blockDim.x) {
            int l, jj, b, j;
            if (COL) d_nl.divmod(bf, &jj, &l);
            else d_pl.divmod(bf, &l, &jj);
            d_m.divmod(jj, &b, &j);
            float2* e = s + l * sl + (b * nq + j) * se;
            const int step = m * se;
            float2 v[7];
#pragma unroll
            for (int c = 0; c < 7; ++c)
                if (c < r) v[c] = e[c * step];
            if (DIR < 0) { // DIT mirror: conj twiddle first
#pragma unroll
                for (int c = 1; c < 7; ++c)
                    if (c < r) v[c] = cmulc(v[c], __ldg(wL + j * c * tws));
            }
            if (r == 4) bfly4<DIR>(v);
            else if (r == 2) bfly2<DIR>(v);
            else if (r == 3) bfly3<DIR>(v);
            else if (r == 5) bfly5<DIR>(v);
            else bfly7<DIR>(v);
            if (DIR > 0) {
#pragma unroll
                for (int c = 1; c < 7; ++c)
                    if (c < r) v[c] = cmul(v[c], __ldg(wL + j * c * tws));
            }
#pragma unroll
            for (int c = 0; c < 7; ++c)
                if (c < r) e[c * step] = v[c];
        }
        __syncthreads();
        if (DIR > 0) nq = m;
    }
}

// height of the fine-grid point at linear offset `off` from the design layout (nearest up-sampling, gray levels)
__device__ __forceinline__ float layout_height(const PassDesc& p, const void* base, long long off)
{
    if ((p.up_lg | p.h_dtype) == 0) return ((const float*)base)[off];
    const long long nx = p.cnx << p.up_lg;
    const long long row = off / nx, x = off - row * nx;
    const long long ci = (row >> p.up_lg) * p.cnx + (x >> p.up_lg);
    if (p.h_dtype == DOP_LAYOUT_F32) return ((const float*)base)[ci];
    if (p.h_dtype == DOP_LAYOUT_U8) return p.h_step * (float)((const unsigned char*)base)[ci];
    return p.h_step * (float)((const unsigned short*)base)[ci];
}

// pad = 2 (dop_plan_desc.pad): the field offset `off` of a point of the [.][grid_nx] window -> the offset of the same
// point in the caller's [ap_ny][ap_nx] planes, or -1 outside the aperture (zero amplitude on the way in, nothing to
// compare or to store on the way out).  ap_nx = 0: no padding, planes and field share their offsets.
__device__ __forceinline__ long long plane_offset(const PassDesc& p, long long off)
{
    if (p.ap_nx == 0) return off;
    const long long row = off / p.grid_nx, x = off - row * p.grid_nx;
    return (x < p.ap_nx && row < p.ap_ny) ? row * p.ap_nx + x : -1;
}

template <bool COL>
__global__ void __launch_bounds__(256, 4) tile_pass_kernel(const PassDesc p)
{
    extern __shared__ float2 s[];
    __shared__ double red[8];
    __shared__ double sred[4][8];
    double st0 = 0.0, st1 = 0.0, st2 = 0.0, st3 = 0.0; // ST_C64_STATS: <I,T>, <I,I>, sum I, <T,T>

    // ---- which tile
    long long t = blockIdx.x;
    const long long cg = t % p.n_cgroups + p.cg0;
    t /= p.n_cgroups;
    const long long m = t % p.n_m;
    const long long o = t / p.n_m + p.o0;
    const long long c0 = cg * p.nl;
    const int nl_eff = (int)((p.NC - c0) < (long long)p.nl ? (p.NC - c0) : (long long)p.nl);
    const long long base = o * p.SO + m * p.SM + c0 * p.SCc;
    const int L = p.L;
    const int sl = COL ? 1 : L;
    const int se = COL ? nl_eff : 1;
    const long long ls = p.SCc, es = p.es;
    const int total = nl_eff * L;
    const FastDiv d_nl(nl_eff), d_L(L);
    float2* s2 = s + p.nl * L; // scratch of the prime-radix steps (the plan doubles smem_bytes for such digits)
    const long long r0 = p.r_from ? m : c0; // boundary-twiddle r of line 0 (x digit: r = c)
    const int r_per_line = p.r_from ? 0 : 1;

    // ---- load (+ prologue op, + conj boundary twiddle before an inverse DFT)
    for (int idx = threadIdx.x; idx < total; idx += blockDim.x) {
        int l, i;
        if (COL) d_nl.divmod(idx, &i, &l);
        else d_L.divmod(idx, &l, &i);
        const long long off = base + l * ls + i * es;
        float2 v;
        const long long poff = (p.load_op == LD_HEIGHT || p.load_op == LD_SEED) ? plane_offset(p, off) : off;
        if (p.load_op == LD_C64) {
            v = p.field[off];
        } else if (poff < 0) {                       // outside the aperture: zero amplitude / zero seed
            v = make_float2(0.0f, 0.0f);
        } else if (p.load_op == LD_HEIGHT) {
            float tt = layout_height(p, p.height, poff) * p.phase_coef; // Eq. (1) in turns
            sincospif(2.0f * tt, &v.y, &v.x);        // Eq. (2), E_in = 1
        } else if (p.load_op == LD_SEED) {
            float2 u = p.field[off];
            float g = 2.0f * p.plane_in[poff];
            v = make_float2(g * u.x, g * u.y);
        } else if (p.load_op == LD_SEED_SIMSE) {     // Eq. (6): 2 dL/dI = c0 + cI I + cT T
            float2 u = p.field[off];
            float g = p.coef[0] + p.coef[1] * (u.x * u.x + u.y * u.y) + p.coef[2] * p.plane_in[off];
            v = make_float2(g * u.x, g * u.y);
        } else {
            v = make_float2(p.coarse_in ? layout_height(p, p.plane_in, off) : p.plane_in[off], 0.0f);
        }
        if (p.tw_b != nullptr && p.fft1_dir < 0) {
            long long r = r0 + (long long)l * r_per_line;
            v = cmulc(v, __ldg(p.tw_b + r * p.pi[i]));
        }
        s[l * sl + i * se] = v;
    }
    __syncthreads();

    if (p.fft1_dir > 0) tile_fft<1, COL>(s, s2, p, nl_eff, sl, se);
    else tile_fft<-1, COL>(s, s2, p, nl_eff, sl, se);

    // ---- middle op
    if (p.mid_op == MID_H || p.mid_op == MID_HCONJ || p.mid_op == MID_GAUSS) {
        const long long row0 = o * p.row_o + m * p.row_m;
        for (int idx = threadIdx.x; idx < total; idx += blockDim.x) {
            int l, i;
            if (COL) d_nl.divmod(idx, &i, &l);
        else d_L.divmod(idx, &l, &i);
            const long long row = row0 + i * p.row_i;
            const long long col = c0 + l;
            float2 v = s[l * sl + i * se];
            if (p.mid_op == MID_GAUSS) {
                float g = p.gx[col] * p.gy[row] * p.scale;
                v = make_float2(v.x * g, v.y * g);
            } else {
                // F4: a = (1/lambda^2 - fx^2) - fy^2 in fp64, the definition's own expression
                double a = (p.inv_lam2 - p.fx2[col]) - p.fy2[row];
                if (a >= 0.0) {
                    double turns = p.z * sqrt(a);
                    float f = (float)(turns - rint(turns)); // fractional turn, |f| <= 0.5
                    float sn, cs;
                    sincospif(2.0f * f, &sn, &cs);
                    float2 H = make_float2(cs * p.scale, (p.mid_op == MID_H ? sn : -sn) * p.scale);
                    v = cmul(v, H);
                } else {
                    v = make_float2(0.0f, 0.0f); // evanescent: zeroed
                }
            }
            s[l * sl + i * se] = v;
        }
        __syncthreads();
    } else if (p.mid_op == MID_LOSS) {
        double acc = 0.0;
        for (int idx = threadIdx.x; idx < total; idx += blockDim.x) {
            int l, i;
            if (COL) d_nl.divmod(idx, &i, &l);
        else d_L.divmod(idx, &l, &i);
            const long long off = base + l * ls + i * es;
            float2 v = s[l * sl + i * se];
            const long long poff = plane_offset(p, off);
            if (poff < 0) {                        // outside the aperture: no loss term, zero seed
                s[l * sl + i * se] = make_float2(0.0f, 0.0f);
                continue;
            }
            float I = v.x * v.x + v.y * v.y;      // F6
            float d = I - p.plane_in[poff];        // F7
            acc += (double)d * (double)d;
            float g = p.seed_coef * d;             // A1: 2 gI = 4 (I - T)/N
            s[l * sl + i * se] = make_float2(g * v.x, g * v.y);
            if (p.write_intensity) p.plane_out[poff] = I;
        }
        // deterministic block reduction: warp shuffle tree, then warp 0 over the 8 partials
        for (int d = 16; d > 0; d >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, d);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
        __syncthreads();
        if (threadIdx.x == 0) {
            double tsum = 0.0;
            for (int w = 0; w < (int)(blockDim.x >> 5); ++w) tsum += red[w];
            p.loss_scratch[p.tile0 + blockIdx.x] = tsum;
        }
        __syncthreads();
    }

    int last_dir = p.fft1_dir;
    if (p.fft2_dir != 0) {
        if (p.fft2_dir > 0) tile_fft<1, COL>(s, s2, p, nl_eff, sl, se);
        else tile_fft<-1, COL>(s, s2, p, nl_eff, sl, se);
        last_dir = p.fft2_dir;
    }

    // ---- store (+ boundary twiddle after a forward DFT, + epilogue op)
    for (int idx = threadIdx.x; idx < total; idx += blockDim.x) {
        int l, i;
        if (COL) d_nl.divmod(idx, &i, &l);
        else d_L.divmod(idx, &l, &i);
        const long long off = base + l * ls + i * es;
        float2 v = s[l * sl + i * se];
        if (p.tw_b != nullptr && last_dir > 0) {
            long long r = r0 + (long long)l * r_per_line;
            v = cmul(v, __ldg(p.tw_b + r * p.pi[i]));
        }
        const long long poff = p.store_op == ST_C64 ? off : plane_offset(p, off);
        if (p.store_op == ST_C64) {
            p.field[off] = v;
        } else if (poff < 0) {                       // outside the aperture: the field is kept, no plane to write
            if (p.store_op == ST_C64_INTENSITY) p.field[off] = v;
        } else if (p.ap_nx != 0 && (p.store_op == ST_GRAD || p.store_op == ST_GRAD_ACC)) {
            float sn, cs;
            sincospif(2.0f * (p.height[poff] * p.phase_coef), &sn, &cs);
            float g = p.grad_coef * (cs * v.y - sn * v.x); // A5 on the aperture
            if (p.store_op == ST_GRAD_ACC) g += p.plane_out[poff];
            p.plane_out[poff] = g;
        } else if (p.ap_nx != 0 && p.store_op == ST_C64_INTENSITY) {
            p.field[off] = v;
            p.plane_out[poff] = v.x * v.x + v.y * v.y;
        } else if (p.store_op == ST_GRAD || p.store_op == ST_GRAD_ACC) {
            const float hv = layout_height(p, p.height, off);
            float tt = hv * p.phase_coef;
            float sn, cs;
            sincospif(2.0f * tt, &sn, &cs); // u0 recomputed, not stored
            float g = p.grad_coef * (cs * v.y - sn * v.x); // A5: c Im(conj(u0) g)
            if (p.store_op == ST_GRAD_ACC) g += p.plane_out[off];
            p.plane_out[off] = g;
            if (p.adam_m != nullptr) { // Adam (Kingma & Ba 2014, Alg. 1) on the last wavelength's store
                const float mn = p.adam_b1 * p.adam_m[off] + p.adam_c1 * g;
                const float vn = p.adam_b2 * p.adam_v[off] + p.adam_c2 * g * g;
                p.adam_m[off] = mn;
                p.adam_v[off] = vn;
                p.adam_h[off] = hv - p.adam_a1 * mn / (sqrtf(vn * p.adam_rb2) + p.adam_eps);
            }
        } else if (p.store_op == ST_C64_INTENSITY) {
            p.field[off] = v;
            p.plane_out[off] = v.x * v.x + v.y * v.y;
        } else if (p.store_op == ST_C64_STATS) {
            p.field[off] = v;
            const float I = v.x * v.x + v.y * v.y, Tv = p.plane_in[off];
            st0 += (double)I * (double)Tv;
            st1 += (double)I * (double)I;
            st2 += (double)I;
            st3 += (double)Tv * (double)Tv;
            if (p.write_intensity) p.plane_out[off] = I;
        } else {
            p.plane_out[off] = v.x;
        }
    }
    if (p.store_op == ST_C64_STATS) {
        for (int d = 16; d > 0; d >>= 1) {
            st0 += __shfl_down_sync(0xffffffffu, st0, d);
            st1 += __shfl_down_sync(0xffffffffu, st1, d);
            st2 += __shfl_down_sync(0xffffffffu, st2, d);
            st3 += __shfl_down_sync(0xffffffffu, st3, d);
        }
        if ((threadIdx.x & 31) == 0) {
            const int w = threadIdx.x >> 5;
            sred[0][w] = st0; sred[1][w] = st1; sred[2][w] = st2; sred[3][w] = st3;
        }
        __syncthreads();
        if (threadIdx.x < 4) {
            double r = 0.0;
            for (int w = 0; w < (int)(blockDim.x >> 5); ++w) r += sred[threadIdx.x][w];
            p.loss_scratch[4 * (p.tile0 + blockIdx.x) + threadIdx.x] = r;
        }
    }
}

cudaError_t launch_tile_pass_generic(const PassDesc& p, cudaStream_t stream)
{
    const long long ntiles = p.n_cgroups * p.n_m * p.n_o;
    if (ntiles <= 0 || ntiles > 2147483647LL) return cudaErrorInvalidConfiguration;
    // the > 48 KiB dynamic shared-memory opt-in is per device function AND per device: once each
    static std::atomic<unsigned long long> attr_mask{0};
    const unsigned long long bit = (p.device >= 0 && p.device < 64) ? 1ull << p.device : 0ull;
    if (bit == 0 || !(attr_mask.load(std::memory_order_acquire) & bit)) {
        const int max_smem = 200 * 1024;
        cudaError_t e = cudaFuncSetAttribute(tile_pass_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(tile_pass_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
        if (e != cudaSuccess) return e;
        if (bit != 0) attr_mask.fetch_or(bit, std::memory_order_release);
    }
    if (p.smem_bytes > 200 * 1024) return cudaErrorInvalidConfiguration;
    if (p.col_type) tile_pass_kernel<true><<<(unsigned)ntiles, p.threads, p.smem_bytes, stream>>>(p);
    else tile_pass_kernel<false><<<(unsigned)ntiles, p.threads, p.smem_bytes, stream>>>(p);
    return cudaGetLastError();
}

// Fixed-order final reduction of the per-CTA loss partials: L = inv_n * sum scratch[0..n)
__global__ void __launch_bounds__(1024) loss_reduce_kernel(const double* __restrict__ scratch, long long n,
                                                           double inv_n, double* __restrict__ out)
{
    __shared__ double sh[1024];
    double acc = 0.0;
    for (long long i = threadIdx.x; i < n; i += 1024) acc += scratch[i];
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int d = 512; d > 0; d >>= 1) {
        if ((int)threadIdx.x < d) sh[threadIdx.x] += sh[threadIdx.x + d];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = sh[0] * inv_n;
}

cudaError_t launch_loss_reduce(const double* scratch, long long n, double inv_n, double* d_loss,
                               cudaStream_t stream)
{
    loss_reduce_kernel<<<1, 1024, 0, stream>>>(scratch, n, inv_n, d_loss);
    return cudaGetLastError();
}

// Eq. (6) (reading in dop.h): fixed-order reduction of the four plane sums of every wavelength,
// then s = <I,T>/<I,I>, L = sum_lambda [ (<T,T> - <I,T>^2/<I,I>)/N + beta (1 - sum I / N) ] and the coefficients of
// the seed 2 dL/dI = c0 + cI I + cT T with dL/dI = (2 s/N)(s I - T) - beta/N.
__global__ void __launch_bounds__(1024) simse_reduce_kernel(const double* __restrict__ scratch, long long tiles, int n_lambda,
                                                            double npts, double beta, float* __restrict__ coef,
                                                            double* __restrict__ out)
{
    __shared__ double sh[4][1024];
    double total = 0.0;
    for (int lam = 0; lam < n_lambda; ++lam) {
        double a[4] = {0.0, 0.0, 0.0, 0.0};
        const double* sc = scratch + 4 * tiles * lam;
        for (long long i = threadIdx.x; i < tiles; i += 1024)
            for (int k = 0; k < 4; ++k) a[k] += sc[4 * i + k];
        for (int k = 0; k < 4; ++k) sh[k][threadIdx.x] = a[k];
        __syncthreads();
        for (int d = 512; d > 0; d >>= 1) {
            if ((int)threadIdx.x < d)
                for (int k = 0; k < 4; ++k) sh[k][threadIdx.x] += sh[k][threadIdx.x + d];
            __syncthreads();
        }
        if (threadIdx.x == 0) {
            const double it = sh[0][0], ii = sh[1][0], si = sh[2][0], tt = sh[3][0];
            const double s = ii > 0.0 ? it / ii : 0.0;
            total += (tt - s * it) / npts + beta * (1.0 - si / npts);
            coef[4 * lam + 0] = (float)(-2.0 * beta / npts);
            coef[4 * lam + 1] = (float)(4.0 * s * s / npts);
            coef[4 * lam + 2] = (float)(-4.0 * s / npts);
            coef[4 * lam + 3] = (float)s;
        }
        __syncthreads();
    }
    if (threadIdx.x == 0 && out != nullptr) *out = total;
}

cudaError_t launch_simse_reduce(const double* scratch, long long tiles, int n_lambda, double npts, double beta,
                                float* coef, double* d_loss, cudaStream_t stream)
{
    simse_reduce_kernel<<<1, 1024, 0, stream>>>(scratch, tiles, n_lambda, npts, beta, coef, d_loss);
    return cudaGetLastError();
}

// Rows of the x-pooled plane [cny r][cnx] -> coarse gradient [cny][cnx] (fixed order over the r rows: with the
// lane tree of the store this is the deterministic r x r sum-pool, the adjoint of the nearest up-sampling), and
// optionally the Adam step on the coarse fp32 layout.
__global__ void __launch_bounds__(256) pool_rows_kernel(const float* __restrict__ xpool, float* __restrict__ grad,
                                                        long long cny, long long cnx, int r, int with_adam, AdamParams ap,
                                                        float* __restrict__ layout, float* __restrict__ m,
                                                        float* __restrict__ v)
{
    const long long n = cny * cnx;
    for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < n; i += (long long)gridDim.x * 256) {
        const long long Y = i / cnx, X = i - Y * cnx;
        float g = 0.0f;
        for (int dy = 0; dy < r; ++dy) g += xpool[(Y * r + dy) * cnx + X];
        grad[i] = g;
        if (with_adam) {
            const float mn = ap.b1 * m[i] + ap.c1 * g;
            const float vn = ap.b2 * v[i] + ap.c2 * g * g;
            m[i] = mn;
            v[i] = vn;
            layout[i] = layout[i] - ap.a1 * mn / (sqrtf(vn * ap.rb2) + ap.eps);
        }
    }
}

cudaError_t launch_pool_rows(const float* xpool, float* grad, long long cny, long long cnx, int r, const AdamParams* adam,
                             float* layout, float* m, float* v, cudaStream_t stream)
{
    const long long n = cny * cnx;
    const unsigned blocks = (unsigned)((n + 255) / 256 < 148 * 16 ? (n + 255) / 256 : 148 * 16);
    pool_rows_kernel<<<blocks, 256, 0, stream>>>(xpool, grad, cny, cnx, r, adam != nullptr, adam ? *adam : AdamParams{},
                                                 layout, m, v);
    return cudaGetLastError();
}

__global__ void __launch_bounds__(256) adam_kernel(const float* __restrict__ grad, long long n, AdamParams ap,
                                                   float* __restrict__ layout, float* __restrict__ m, float* __restrict__ v)
{
    for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < n; i += (long long)gridDim.x * 256) {
        const float g = grad[i];
        const float mn = ap.b1 * m[i] + ap.c1 * g;
        const float vn = ap.b2 * v[i] + ap.c2 * g * g;
        m[i] = mn;
        v[i] = vn;
        layout[i] = layout[i] - ap.a1 * mn / (sqrtf(vn * ap.rb2) + ap.eps);
    }
}

cudaError_t launch_adam(const float* grad, long long n, const AdamParams& adam, float* layout, float* m, float* v,
                        cudaStream_t stream)
{
    const unsigned blocks = (unsigned)((n + 255) / 256 < 148 * 16 ? (n + 255) / 256 : 148 * 16);
    adam_kernel<<<blocks, 256, 0, stream>>>(grad, n, adam, layout, m, v);
    return cudaGetLastError();
}

} // namespace dop
