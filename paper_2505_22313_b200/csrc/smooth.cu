// smooth.cu -- plain digit passes (field -> DFT -> field) for the 5-smooth digits of the paper's own grids
// (Table 2: 28 800 = 32 * 900 = 225 * 128, 40 000 = 16 * 2500 = 625 * 64), which until now ran on the
// generic kernel's runtime-radix loops at a fifth of the copy bandwidth.
//
// A digit L = R^2 (225 = 15^2, 625 = 25^2, 900 = 30^2, 2500 = 50^2) is two register steps of R points each, with ONE
// exchange through shared memory between them.  A register step is itself R = R1 R2 R3 mixed-radix (5.3, 5.5, 5.3.2,
// 5.5.2): the thread keeps its R points in registers and runs the three sub-stages of the generic kernel's in-place
// decimation-in-frequency schedule (radix list R1.R2.R3.R1.R2.R3, which is what plan.cu gives these digits) without
// touching memory, so slot order, tables and boundary twiddles are exactly those of the generic kernel -- which stays
// the checker (dop_tuning.no_smooth / force_generic) and the carrier of every fused pass and every other digit.
//   forward : step A (sub-length L: points j + R c of the line, j = thread) -> exchange -> step B (sub-length R: points
//             b R + c, b = thread) -> boundary twiddle -> store;     inverse: the exact mirror (conj twiddles first).
//   in-step twiddles W^(j k): one table load per butterfly for W^j, the powers by multiplication (k <= 4).
// Column-type tiles (y digits, higher x digits): NL adjacent lines, lanes over the lines; the first step loads its
// points straight from global memory (NL * 8 contiguous bytes per point row) and the last stores them straight back.
// Row-type tiles (last x digit): NL contiguous lines; the tile is staged through shared memory with coalesced 16-byte
// accesses on both sides, in a layout padded by P points per R (odd stride between the blocks of step B: no bank
// conflicts in either step).
#include <atomic>

#include "dop_internal.h"
#include "fft_regs.cuh"

namespace dop {
namespace {

// ---- packed fp32x2 butterflies (fft_regs.cuh: one complex add = one FADD2, one complex multiply = FMUL2 + FFMA2; the
//      -i rotation and the negations ride on the operand modifiers).  Same outputs, in the same places, as the scalar
//      butterflies of bfly.cuh that the generic kernel runs.
using fx::add2;
using fx::fma2;
using fx::mul2;
__device__ __forceinline__ float2 bc(float x) { return make_float2(x, x); }
__device__ __forceinline__ float2 neg(float2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ float2 rot_mi(float2 a) { return make_float2(a.y, -a.x); } // -i a

template <int R, int DIR> struct Bfly;
template <int DIR> struct Bfly<1, DIR> { static __device__ __forceinline__ void run(float2*) {} };
template <int DIR> struct Bfly<2, DIR> {
    static __device__ __forceinline__ void run(float2* v)
    {
        const float2 a = v[0], b = v[1];
        v[0] = add2(a, b);
        v[1] = add2(a, neg(b));
    }
};
template <int DIR> struct Bfly<3, DIR> {
    static __device__ __forceinline__ void run(float2* v)
    {
        const float h = 0.86602540378443864676f; // sqrt(3)/2
        const float2 a = v[0], b = v[1], c = v[2];
        const float2 t1 = add2(b, c);
        const float2 t2 = fma2(bc(-0.5f), t1, a);
        const float2 r = rot_mi(add2(b, neg(c)));
        v[0] = add2(a, t1);
        const float2 m = fma2(bc(h), r, t2), q = fma2(bc(-h), r, t2); // t2 -+ i h (b - c)
        if (DIR > 0) { v[1] = m; v[2] = q; } else { v[1] = q; v[2] = m; }
    }
};
template <int DIR> struct Bfly<4, DIR> {
    static __device__ __forceinline__ void run(float2* v) { fx::bf4<DIR>(v[0], v[1], v[2], v[3]); }
};
template <int DIR> struct Bfly<5, DIR> {
    static __device__ __forceinline__ void run(float2* v)
    {
        const float c1 = 0.30901699437494742410f, c2 = -0.80901699437494742410f; // cos(2 pi/5), cos(4 pi/5)
        const float s1 = 0.95105651629515357212f, s2 = 0.58778525229247312917f;  // sin(2 pi/5), sin(4 pi/5)
        const float2 x0 = v[0];
        const float2 a1 = add2(v[1], v[4]), b1 = add2(v[1], neg(v[4])), a2 = add2(v[2], v[3]), b2 = add2(v[2], neg(v[3]));
        v[0] = add2(x0, add2(a1, a2));
        const float2 A1 = fma2(bc(c2), a2, fma2(bc(c1), a1, x0)), A2 = fma2(bc(c1), a2, fma2(bc(c2), a1, x0));
        const float2 r1 = rot_mi(fma2(bc(s2), b2, mul2(bc(s1), b1))), r2 = rot_mi(fma2(bc(-s1), b2, mul2(bc(s2), b1)));
        // forward: y_k = A_k - i B_k, y_{5-k} = A_k + i B_k
        const float2 m1 = add2(A1, r1), q1 = add2(A1, neg(r1)), m2 = add2(A2, r2), q2 = add2(A2, neg(r2));
        if (DIR > 0) { v[1] = m1; v[4] = q1; v[2] = m2; v[3] = q2; }
        else { v[1] = q1; v[4] = m1; v[2] = q2; v[3] = m2; }
    }
};

// a[k] *= w^k (forward: on the outputs) or a[k] *= conj(w)^k (inverse: on the inputs), k = 1 .. R-1
template <int R, bool CONJ>
__device__ __forceinline__ void twiddle_powers(float2* a, float2 w)
{
    float2 wk = w;
#pragma unroll
    for (int k = 1; k < R; ++k) {
        a[k] = CONJ ? fx::cmulc(a[k], wk) : fx::cmul(a[k], wk);
        if (k + 1 < R) wk = fx::cmul(wk, w);
    }
}

// One register step: the sub-stages (R1, R2, R3) of the in-place schedule at sub-length NQ of a digit of length L, on
// the R = R1 R2 R3 points v[c1 R2 R3 + c2 R3 + c3] = x[j + c3 m3 + c2 m2 + c1 m1], m1 = NQ/R1, m2 = m1/R2, m3 = m2/R3,
// j in [0, m3).  W_n^x = wL[x L/n].
template <int DIR, int L, int NQ, int R1, int R2, int R3>
__device__ __forceinline__ void reg_step(float2* v, const float2* __restrict__ wL, int j)
{
    constexpr int R23 = R2 * R3;
    constexpr int m1 = NQ / R1, m2 = m1 / R2, m3 = m2 / R3;
    constexpr bool CJ = DIR < 0;
    auto stage1 = [&]() {
#pragma unroll
        for (int c2 = 0; c2 < R2; ++c2)
#pragma unroll
            for (int c3 = 0; c3 < R3; ++c3) {
                float2 a[R1];
#pragma unroll
                for (int c1 = 0; c1 < R1; ++c1) a[c1] = v[c1 * R23 + c2 * R3 + c3];
                float2 w = make_float2(1.0f, 0.0f);
                if (m1 > 1) w = __ldg(wL + (j + c3 * m3 + c2 * m2) * (L / NQ));
                if (CJ && m1 > 1) twiddle_powers<R1, true>(a, w);
                Bfly<R1, DIR>::run(a);
                if (!CJ && m1 > 1) twiddle_powers<R1, false>(a, w);
#pragma unroll
                for (int c1 = 0; c1 < R1; ++c1) v[c1 * R23 + c2 * R3 + c3] = a[c1];
            }
    };
    auto stage2 = [&]() {
        if (R2 == 1) return;
        float2 w[R3];
#pragma unroll
        for (int c3 = 0; c3 < R3; ++c3) w[c3] = m2 > 1 ? __ldg(wL + (j + c3 * m3) * (L / m1)) : make_float2(1.0f, 0.0f);
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1)
#pragma unroll
            for (int c3 = 0; c3 < R3; ++c3) {
                float2 a[R2];
#pragma unroll
                for (int c2 = 0; c2 < R2; ++c2) a[c2] = v[k1 * R23 + c2 * R3 + c3];
                if (CJ && m2 > 1) twiddle_powers<R2, true>(a, w[c3]);
                Bfly<R2, DIR>::run(a);
                if (!CJ && m2 > 1) twiddle_powers<R2, false>(a, w[c3]);
#pragma unroll
                for (int c2 = 0; c2 < R2; ++c2) v[k1 * R23 + c2 * R3 + c3] = a[c2];
            }
    };
    auto stage3 = [&]() {
        if (R3 == 1) return;
        const float2 w = m3 > 1 ? __ldg(wL + j * (L / m2)) : make_float2(1.0f, 0.0f);
#pragma unroll
        for (int k12 = 0; k12 < R1 * R2; ++k12) {
            float2 a[R3];
#pragma unroll
            for (int c3 = 0; c3 < R3; ++c3) a[c3] = v[k12 * R3 + c3];
            if (CJ && m3 > 1) twiddle_powers<R3, true>(a, w);
            Bfly<R3, DIR>::run(a);
            if (!CJ && m3 > 1) twiddle_powers<R3, false>(a, w);
#pragma unroll
            for (int c3 = 0; c3 < R3; ++c3) v[k12 * R3 + c3] = a[c3];
        }
    };
    if (DIR > 0) { stage1(); stage2(); stage3(); }
    else { stage3(); stage2(); stage1(); }
}

struct TileId { long long base, c0, m; int nl_eff; };

__device__ __forceinline__ TileId decode_tile(const PassDesc& p)
{
    // (the launch has fewer than 2^31 tiles, so its three coordinates divide out in 32 bits)
    unsigned t = blockIdx.x;
    const unsigned ncg = (unsigned)p.n_cgroups, nm = (unsigned)p.n_m;
    const unsigned tq = t / ncg;
    const long long cg = (long long)(t - tq * ncg) + p.cg0;
    const unsigned oq = tq / nm;
    const long long m = tq - oq * nm;
    const long long o = (long long)oq + p.o0;
    TileId id;
    id.c0 = cg * p.nl;
    id.m = m;
    id.nl_eff = (int)((p.NC - id.c0) < (long long)p.nl ? (p.NC - id.c0) : (long long)p.nl);
    id.base = o * p.SO + m * p.SM + id.c0 * p.SCc;
    return id;
}

// ---- column-type tile: NL adjacent lines x L points, thread = (point group bf, line l), lanes over the lines
template <int DIR, int R1, int R2, int R3, int NL>
__global__ void __launch_bounds__(NL * R1 * R2 * R3) smooth_col_kernel(const PassDesc p)
{
    constexpr int R = R1 * R2 * R3, L = R * R;
    extern __shared__ float2 s[]; // [L][NL]
    const TileId id = decode_tile(p);
    const int l = threadIdx.x % NL, bf = threadIdx.x / NL;
    const bool live = l < id.nl_eff;
    float2* __restrict__ g = p.field + id.base + l;
    const long long es = p.es;
    const float2* __restrict__ wL = p.wL;
    // boundary twiddle of (slot, r): y digits tw_b2[r L + slot] (r = m), x digits tw_b2[slot st + r] (r = c0 + l)
    const float2* __restrict__ tb = nullptr;
    long long tbs = 1;
    if (p.tw_b2 != nullptr) {
        if (p.r_from) tb = p.tw_b2 + id.m * L;
        else { tbs = p.twb_n / L; tb = p.tw_b2 + id.c0 + l; }
    }
    float2 v[R];
    // running pointers: A side = points bf + R c (stride R es), B side = points bf R + c (stride es)
    float2* __restrict__ ga = g + (long long)bf * es;
    float2* __restrict__ gb = g + (long long)(bf * R) * es;
    const long long sa = (long long)R * es;
    auto twiddle_b = [&](auto mulop) { // boundary twiddles of the B-side points
        if (tb == nullptr) return;
        if (p.r_from) {
            const float2* __restrict__ t = tb + bf * R;
#pragma unroll
            for (int c = 0; c < R; ++c) v[c] = mulop(v[c], __ldg(t + c));
        } else {
            const float2* __restrict__ t = tb + (long long)(bf * R) * tbs;
#pragma unroll
            for (int c = 0; c < R; ++c) { v[c] = mulop(v[c], __ldg(t)); t += tbs; }
        }
    };
    if (DIR > 0) {
        if (live) {
            const float2* q = ga;
#pragma unroll
            for (int c = 0; c < R; ++c) { v[c] = __ldcs(q); q += sa; }
            reg_step<1, L, L, R1, R2, R3>(v, wL, bf);
#pragma unroll
            for (int c = 0; c < R; ++c) s[(bf + R * c) * NL + l] = v[c];
        }
        __syncthreads();
        if (live) {
#pragma unroll
            for (int c = 0; c < R; ++c) v[c] = s[(bf * R + c) * NL + l];
            reg_step<1, L, R, R1, R2, R3>(v, wL, 0);
            twiddle_b([](float2 a, float2 b) { return fx::cmul(a, b); });
            float2* q = gb;
#pragma unroll
            for (int c = 0; c < R; ++c) { __stcs(q, v[c]); q += es; }
        }
    } else {
        if (live) {
            const float2* q = gb;
#pragma unroll
            for (int c = 0; c < R; ++c) { v[c] = __ldcs(q); q += es; }
            twiddle_b([](float2 a, float2 b) { return fx::cmulc(a, b); });
            reg_step<-1, L, R, R1, R2, R3>(v, wL, 0);
#pragma unroll
            for (int c = 0; c < R; ++c) s[(bf * R + c) * NL + l] = v[c];
        }
        __syncthreads();
        if (live) {
#pragma unroll
            for (int c = 0; c < R; ++c) v[c] = s[(bf + R * c) * NL + l];
            reg_step<-1, L, L, R1, R2, R3>(v, wL, bf);
            float2* q = ga;
#pragma unroll
            for (int c = 0; c < R; ++c) { __stcs(q, v[c]); q += sa; }
        }
    }
}

// ---- row-type tile: NL contiguous lines of L points (the tile is one contiguous run), thread = (line l, point group bf)
// Forward: the A side (points bf + R c: runs of R contiguous points across the lanes) is loaded straight from global
// memory into registers; everything else is staged through shared memory with coalesced 16-byte accesses.
// (R = 50: without a bound the inverse kernel takes 176 registers and runs one 200-thread CTA per SM; the tile's shared
//  memory allows two.  The shorter steps are left to the compiler: a bound of 3-4 CTAs made them spill and slower.)
constexpr int row_min_ctas(int R, int NL) { return R >= 50 ? 2 : 0; } // (0 = no bound)

template <int DIR, int R1, int R2, int R3, int NL>
__global__ void __launch_bounds__(NL * R1 * R2 * R3, row_min_ctas(R1 * R2 * R3, NL)) smooth_row_kernel(const PassDesc p)
{
    constexpr int R = R1 * R2 * R3, L = R * R, P = (R % 2 == 0) ? 1 : 2, LP = L + R * P, T = NL * R;
    constexpr int W = (L % 2 == 0) ? 2 : 1;  // points per staging access: 16-byte where every line starts 16-byte aligned
    constexpr int NIT = L / (R * W);         // staging accesses per thread of a full tile
    extern __shared__ float2 s[];            // [NL][LP], point i of a line at i + (i / R) P
    const TileId id = decode_tile(p);
    const int bf = threadIdx.x % R, l = threadIdx.x / R;
    const bool live = l < id.nl_eff;
    float2* __restrict__ g = p.field + id.base;
    const float2* __restrict__ wL = p.wL;
    const int total = id.nl_eff * L;
    float2* __restrict__ sl = s + l * LP;
    float2 v[R];
    auto smem_of = [&](int q) { const int ln = q / L, i = q - ln * L; return s + ln * LP + i + (i / R) * P; };
    if (DIR > 0) {
        if (live) {
#pragma unroll
            for (int c = 0; c < R; ++c) v[c] = __ldcs(g + l * L + bf + R * c);
            reg_step<1, L, L, R1, R2, R3>(v, wL, bf);
#pragma unroll
            for (int c = 0; c < R; ++c) sl[bf + c * (R + P)] = v[c];
        }
        __syncthreads();
        if (live) {
#pragma unroll
            for (int c = 0; c < R; ++c) v[c] = sl[bf * (R + P) + c];
            reg_step<1, L, R, R1, R2, R3>(v, wL, 0);
#pragma unroll
            for (int c = 0; c < R; ++c) sl[bf * (R + P) + c] = v[c];
        }
        __syncthreads();
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
            const int q = W * (threadIdx.x + it * T);
            if (q < total) {
                const float2* d = smem_of(q); // (W = 2: q even and R even, so q and q + 1 share a block of R)
                if (W == 2) __stcs(reinterpret_cast<float4*>(g + q), make_float4(d[0].x, d[0].y, d[1].x, d[1].y));
                else __stcs(g + q, d[0]);
            }
        }
    } else {
        constexpr int CH = NIT <= 16 ? NIT : (NIT + 1) / 2; // staging accesses in flight per thread (register budget)
#pragma unroll
        for (int it0 = 0; it0 < NIT; it0 += CH) {
            float4 x4[W == 2 ? CH : 1];
            float2 x2[W == 1 ? CH : 1];
#pragma unroll
            for (int k = 0; k < CH; ++k) {
                const int q = W * (threadIdx.x + (it0 + k) * T);
                if (it0 + k < NIT && q < total) {
                    if (W == 2) x4[k] = __ldcs(reinterpret_cast<const float4*>(g + q));
                    else x2[k] = __ldcs(g + q);
                }
            }
#pragma unroll
            for (int k = 0; k < CH; ++k) {
                const int q = W * (threadIdx.x + (it0 + k) * T);
                if (it0 + k < NIT && q < total) {
                    float2* d = smem_of(q);
                    if (W == 2) { d[0] = make_float2(x4[k].x, x4[k].y); d[1] = make_float2(x4[k].z, x4[k].w); }
                    else d[0] = x2[k];
                }
            }
        }
        __syncthreads();
        if (live) {
#pragma unroll
            for (int c = 0; c < R; ++c) v[c] = sl[bf * (R + P) + c];
            reg_step<-1, L, R, R1, R2, R3>(v, wL, 0);
#pragma unroll
            for (int c = 0; c < R; ++c) sl[bf * (R + P) + c] = v[c];
        }
        __syncthreads();
        if (live) {
#pragma unroll
            for (int c = 0; c < R; ++c) v[c] = sl[bf + c * (R + P)];
            reg_step<-1, L, L, R1, R2, R3>(v, wL, bf);
#pragma unroll
            for (int c = 0; c < R; ++c) sl[bf + c * (R + P)] = v[c];
        }
        // (straight stores of the A side -- 8 bytes per lane in runs of R points -- measured slower than this second
        //  staging: 28 800^2 x-inv 3.80 -> 3.07 ms)
        __syncthreads();
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
            const int q = W * (threadIdx.x + it * T);
            if (q < total) {
                const float2* d = smem_of(q);
                if (W == 2) __stcs(reinterpret_cast<float4*>(g + q), make_float4(d[0].x, d[0].y, d[1].x, d[1].y));
                else __stcs(g + q, d[0]);
            }
        }
    }
}

struct SmoothShape { int L, r1, r2, r3, nl_col, nl_row; };
// (L = (r1 r2 r3)^2; lines per column / row tile, measured on B200: 16-line column tiles of 225 and 16-line row tiles
//  of 900 are slower; 0 = no column kernel: the plan never makes 900 or 2500 a column digit)
constexpr SmoothShape kShapes[] = {
    {225, 5, 3, 1, 32, 16},
    {625, 5, 5, 1, 16, 8},
    {900, 5, 3, 2, 0, 8},
    {2500, 5, 5, 2, 0, 4},
};

const SmoothShape* find_shape(long long L)
{
    for (const SmoothShape& sh : kShapes)
        if (sh.L == L) return &sh;
    return nullptr;
}

template <void (*KERNEL)(const PassDesc)>
cudaError_t launch_k(const PassDesc& p, cudaStream_t st)
{
    const long long ntiles = p.n_cgroups * p.n_m * p.n_o;
    if (ntiles <= 0 || ntiles > 2147483647LL) return cudaErrorInvalidConfiguration;
    // the > 48 KiB dynamic shared-memory opt-in is per device function AND per device: once each
    static std::atomic<unsigned long long> attr_mask{0};
    const unsigned long long bit = (p.device >= 0 && p.device < 64) ? 1ull << p.device : 0ull;
    if (p.smem_bytes > 48 * 1024 && (bit == 0 || !(attr_mask.load(std::memory_order_acquire) & bit))) {
        cudaError_t e = cudaFuncSetAttribute(KERNEL, cudaFuncAttributeMaxDynamicSharedMemorySize, p.smem_bytes);
        if (e != cudaSuccess) return e;
        if (bit != 0) attr_mask.fetch_or(bit, std::memory_order_release);
    }
    KERNEL<<<(unsigned)ntiles, p.threads, p.smem_bytes, st>>>(p);
    return cudaGetLastError();
}

template <int R1, int R2, int R3, int NLC, int NLR>
cudaError_t launch_shape(const PassDesc& p, cudaStream_t st)
{
    if (p.col_type) {
        if constexpr (NLC > 0) {
            if (p.nl != NLC) return cudaErrorInvalidConfiguration;
            return p.fft1_dir > 0 ? launch_k<smooth_col_kernel<1, R1, R2, R3, NLC>>(p, st)
                                  : launch_k<smooth_col_kernel<-1, R1, R2, R3, NLC>>(p, st);
        }
        return cudaErrorInvalidConfiguration;
    }
    if (p.nl != NLR) return cudaErrorInvalidConfiguration;
    return p.fft1_dir > 0 ? launch_k<smooth_row_kernel<1, R1, R2, R3, NLR>>(p, st)
                          : launch_k<smooth_row_kernel<-1, R1, R2, R3, NLR>>(p, st);
}

} // namespace

// the radix list plan.cu gives a smooth digit (R1.R2.R3 twice, ones dropped); empty = not a smooth digit
std::vector<int> smooth_radix(long long L)
{
    std::vector<int> r;
    if (const SmoothShape* sh = find_shape(L))
        for (int rep = 0; rep < 2; ++rep)
            for (int q : {sh->r1, sh->r2, sh->r3})
                if (q > 1) r.push_back(q);
    return r;
}

bool smooth_supported(long long L, bool col_type)
{
    const SmoothShape* sh = find_shape(L);
    return sh != nullptr && (!col_type || sh->nl_col > 0);
}

// tile shape of a smooth pass: lines per tile, threads, dynamic shared memory
void smooth_geometry(long long L, bool col_type, int* nl, int* threads, int* smem_bytes)
{
    const SmoothShape* sh = find_shape(L);
    const int R = sh->r1 * sh->r2 * sh->r3;
    *nl = col_type ? sh->nl_col : sh->nl_row;
    *threads = *nl * R;
    const int lp = col_type ? (int)L : (int)L + R * (R % 2 == 0 ? 1 : 2);
    *smem_bytes = *nl * lp * (int)sizeof(float2);
}

cudaError_t launch_tile_pass_smooth(const PassDesc& p, cudaStream_t st, bool* handled)
{
    *handled = false;
    if (!p.smooth) return cudaSuccess;
    const bool plain = p.load_op == LD_C64 && p.mid_op == MID_NONE && p.store_op == ST_C64 && p.fft2_dir == 0;
    if (!plain || find_shape(p.L) == nullptr) return cudaSuccess;
    if (!p.col_type && p.tw_b != nullptr) return cudaSuccess; // (row-type = last x digit: no boundary twiddle)
    if (p.col_type && (p.tw_b != nullptr) != (p.tw_b2 != nullptr)) return cudaSuccess;
    *handled = true;
    switch (p.L) {
    case 225: return launch_shape<5, 3, 1, 32, 16>(p, st);
    case 625: return launch_shape<5, 5, 1, 16, 8>(p, st);
    case 900: return launch_shape<5, 3, 2, 0, 8>(p, st);
    case 2500: return launch_shape<5, 5, 2, 0, 4>(p, st);
    }
    *handled = false;
    return cudaSuccess;
}

} // namespace dop
