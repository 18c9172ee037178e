// fft_regs.cuh -- register-blocked power-of-two line FFT for one CTA tile (sm_100a).
//
// Same mathematics and the same slot order as the generic in-place kernel (kernels_generic.cu):
// in-place decimation in frequency over the radix list (4, 4, ..., 4[, 2]) of a digit of length
// L = 2^p, inverse = exact mirror (decimation in time, conjugate twiddles).  What differs is where
// the data lives: every thread keeps P = 16 points in registers and runs up to two radix-4
// sub-steps (one radix-16 "group") without touching memory; groups exchange data through shared
// memory (one 64-bit store + one 64-bit load per point), and the first / last group load from and
// store to global memory directly from registers.  See DESIGN.md "Kernels".
//
//   group g:  block length n_g, radix R_g = RA*RB (RA in {2,4}, RB in {1,2,4}), m_g = n_g / R_g
//   butterfly id bf in [0, L/R_g):  b = bf / m_g,  j = bf % m_g,  slots  b n_g + j + c m_g, c < R_g
//   register c = ca RB + cb  <->  after the group register c' = ca' RB + cb' holds the output of
//   frequency k = ca' + RA cb' (digit-reversed within the group), times W_{n_g}^{j k}.
#pragma once
#include <cuda_runtime.h>

namespace dop {
namespace fx {

constexpr int P = 16; // points per thread

// ---- packed fp32x2 arithmetic (sm_100a FADD2 / FMUL2 / FFMA2) ----------------------------------
// A complex64 value is a 64-bit register pair, so one complex add is ONE packed instruction and a
// complex multiply is TWO (FMUL2 + FFMA2); the half-swap / per-half-negate operand modifiers of
// the packed instructions (SASS .LO_HI / .NP, scalar broadcast R.F32) make the +-i rotations and
// the (v.y,v.y) x (w.y,w.x) terms free.  The packed pipe retires 2 lanes per instruction at half
// the issue rate: same flop/s as scalar FADD/FFMA, half the issue slots.
__device__ __forceinline__ float2 add2(float2 a, float2 b)
{
    float2 r;
    asm("{ .reg .b64 a,b,c; mov.b64 a,{%2,%3}; mov.b64 b,{%4,%5}; add.rn.f32x2 c,a,b; mov.b64 {%0,%1},c; }"
        : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}
__device__ __forceinline__ float2 mul2(float2 a, float2 b)
{
    float2 r;
    asm("{ .reg .b64 a,b,c; mov.b64 a,{%2,%3}; mov.b64 b,{%4,%5}; mul.rn.f32x2 c,a,b; mov.b64 {%0,%1},c; }"
        : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c)
{
    float2 r;
    asm("{ .reg .b64 a,b,c,d; mov.b64 a,{%2,%3}; mov.b64 b,{%4,%5}; mov.b64 c,{%6,%7}; fma.rn.f32x2 d,a,b,c; "
        "mov.b64 {%0,%1},d; }"
        : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y), "f"(c.x), "f"(c.y));
    return r;
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return add2(a, b); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return add2(a, make_float2(-b.x, -b.y)); }
__device__ __forceinline__ float2 cmul(float2 a, float2 b) // a * b
{
    const float2 t = mul2(make_float2(a.y, a.y), make_float2(b.y, b.x));
    return fma2(make_float2(a.x, a.x), b, make_float2(-t.x, t.y));
}
__device__ __forceinline__ float2 cmulc(float2 a, float2 b) // a * conj(b)
{
    const float2 t = mul2(make_float2(a.x, a.x), b);
    return fma2(make_float2(a.y, a.y), make_float2(b.y, b.x), make_float2(t.x, -t.y));
}

// ---- compile-time schedule of a digit of length L ---------------------------------------------
__host__ __device__ constexpr int ilog2(int x) { return x <= 1 ? 0 : 1 + ilog2(x >> 1); }

template <int L>
struct Sched {
    static constexpr int LG = ilog2(L);
    static constexpr int N4 = LG / 2;       // radix-4 sub-steps
    static constexpr int N2 = LG & 1;       // trailing radix-2 sub-step
    static constexpr int NFULL = N4 / 2;    // radix-16 groups
    static constexpr int REM4 = N4 & 1;
    static constexpr int RLAST = (REM4 ? 4 : 1) * (N2 ? 2 : 1); // 1 = no remainder group
    static constexpr int NG = NFULL + (RLAST > 1 ? 1 : 0);
    __host__ __device__ static constexpr int radix(int g) { return g < NFULL ? 16 : RLAST; }
    __host__ __device__ static constexpr int block(int g) { return g == 0 ? L : block(g - 1) / radix(g - 1); } // n_g
    __host__ __device__ static constexpr int twoff(int g) // offset (float2) of group g's twiddle table
    {
        return g == 0 ? 0 : twoff(g - 1) + (radix(g - 1) - 1) * (block(g - 1) / radix(g - 1));
    }
    static constexpr int TWSIZE = twoff(NG); // the last group's (m = 1) entries are never read
};

// ---- radix-2 / radix-4 butterflies on registers -----------------------------------------------
template <int DIR>
__device__ __forceinline__ void bf2(float2& a, float2& b)
{
    const float2 t = a;
    a = cadd(t, b);
    b = csub(t, b);
}
template <int DIR>
__device__ __forceinline__ void bf4(float2& a, float2& b, float2& c, float2& d)
{
    const float2 s0 = cadd(a, c), s1 = csub(a, c), s2 = cadd(b, d), s3 = csub(b, d);
    a = cadd(s0, s2);
    c = csub(s0, s2);
    const float2 r = make_float2(s3.y, -s3.x); // -i s3 (folded into the operand modifiers)
    if (DIR > 0) { // b = s1 - i s3, d = s1 + i s3
        b = cadd(s1, r);
        d = csub(s1, r);
    } else {
        b = csub(s1, r);
        d = cadd(s1, r);
    }
}

// v *= W_16^{E} (DIR > 0) or its conjugate (DIR < 0), E a compile-time exponent
template <int E, int DIR>
__device__ __forceinline__ void mul_w16(float2& v)
{
    constexpr int e = ((E % 16) + 16) % 16;
    constexpr float C1 = 0.92387953251128675613f, S1 = 0.38268343236508977173f, H = 0.70710678118654752440f;
    // W16^e = cos(2 pi e/16) - i sin(2 pi e/16)
    constexpr float co[16] = {1.f, C1, H, S1, 0.f, -S1, -H, -C1, -1.f, -C1, -H, -S1, 0.f, S1, H, C1};
    constexpr float si[16] = {0.f, S1, H, C1, 1.f, C1, H, S1, 0.f, -S1, -H, -C1, -1.f, -C1, -H, -S1};
    if (e == 0) return;
    const float c = co[e], s = (DIR > 0) ? -si[e] : si[e]; // multiply by (c + i s)
    if (e == 4 || e == 12) { // +-i
        v = s > 0.f ? make_float2(-v.y, v.x) : make_float2(v.y, -v.x);
    } else if (e == 8) {
        v = make_float2(-v.x, -v.y);
    } else if (e % 4 == 2) { // c, s = +-H:  v (c + i s) = H (sc v + ss i v)
        const float2 iv = make_float2(-v.y, v.x);
        const float2 a = c > 0.f ? v : make_float2(-v.x, -v.y);
        const float2 b = s > 0.f ? iv : make_float2(-iv.x, -iv.y);
        v = mul2(make_float2(H, H), add2(a, b));
    } else {
        v = cmul(v, make_float2(c, s));
    }
}

// One group butterfly on R = RA*RB registers v[0], v[ST], ..., v[(R-1) ST] (ST = register stride).
template <int RA, int RB, int DIR, int ST>
__device__ __forceinline__ void group(float2* v)
{
    constexpr int R = RA * RB;
    if (DIR > 0) {
#pragma unroll
        for (int cb = 0; cb < RB; ++cb) {
            if (RA == 4) bf4<DIR>(v[(0 * RB + cb) * ST], v[(1 * RB + cb) * ST], v[(2 * RB + cb) * ST], v[(3 * RB + cb) * ST]);
            else bf2<DIR>(v[(0 * RB + cb) * ST], v[(1 * RB + cb) * ST]);
        }
        if (RB > 1) {
            // internal twiddles W_R^{cb ca'} = W_16^{cb ca' 16/R}
#define DOP_TW(CA, CB) mul_w16<(CA) * (CB) * (16 / R), DIR>(v[((CA) * RB + (CB)) * ST])
            if (RA == 4 && RB == 4) {
                DOP_TW(1, 1); DOP_TW(1, 2); DOP_TW(1, 3);
                DOP_TW(2, 1); DOP_TW(2, 2); DOP_TW(2, 3);
                DOP_TW(3, 1); DOP_TW(3, 2); DOP_TW(3, 3);
            } else if (RA == 4 && RB == 2) {
                DOP_TW(1, 1); DOP_TW(2, 1); DOP_TW(3, 1);
            }
#pragma unroll
            for (int ca = 0; ca < RA; ++ca) {
                if (RB == 4) bf4<DIR>(v[(ca * RB + 0) * ST], v[(ca * RB + 1) * ST], v[(ca * RB + 2) * ST], v[(ca * RB + 3) * ST]);
                else bf2<DIR>(v[(ca * RB + 0) * ST], v[(ca * RB + 1) * ST]);
            }
        }
    } else {
        if (RB > 1) {
#pragma unroll
            for (int ca = 0; ca < RA; ++ca) {
                if (RB == 4) bf4<DIR>(v[(ca * RB + 0) * ST], v[(ca * RB + 1) * ST], v[(ca * RB + 2) * ST], v[(ca * RB + 3) * ST]);
                else bf2<DIR>(v[(ca * RB + 0) * ST], v[(ca * RB + 1) * ST]);
            }
            if (RA == 4 && RB == 4) {
                DOP_TW(1, 1); DOP_TW(1, 2); DOP_TW(1, 3);
                DOP_TW(2, 1); DOP_TW(2, 2); DOP_TW(2, 3);
                DOP_TW(3, 1); DOP_TW(3, 2); DOP_TW(3, 3);
            } else if (RA == 4 && RB == 2) {
                DOP_TW(1, 1); DOP_TW(2, 1); DOP_TW(3, 1);
            }
#undef DOP_TW
        }
#pragma unroll
        for (int cb = 0; cb < RB; ++cb) {
            if (RA == 4) bf4<DIR>(v[(0 * RB + cb) * ST], v[(1 * RB + cb) * ST], v[(2 * RB + cb) * ST], v[(3 * RB + cb) * ST]);
            else bf2<DIR>(v[(0 * RB + cb) * ST], v[(1 * RB + cb) * ST]);
        }
    }
}

template <int R> struct Split;
template <> struct Split<16> { static constexpr int RA = 4, RB = 4; };
template <> struct Split<8> { static constexpr int RA = 4, RB = 2; };
template <> struct Split<4> { static constexpr int RA = 4, RB = 1; };
template <> struct Split<2> { static constexpr int RA = 2, RB = 1; };

// frequency index (within the group) held by register c' after a forward group
template <int R>
__host__ __device__ constexpr int group_freq(int c)
{
    return (c / Split<R>::RB) + Split<R>::RA * (c % Split<R>::RB);
}

// ---- tile-level engine --------------------------------------------------------------------------
// Shared-memory layout of one tile.
//   COL = true : NB (16, 32 or 64) adjacent lines; element (slot, col) at slot*NB + col (conflict-free).
//   COL = false: one line; slot s at s + 2*(s >> 5) (two pad elements per 32 keep every access
//                pattern of the schedule conflict-free and 16-byte alignment of even slots).
template <int L, bool COL, int NB = 16>
struct Tile {
    using S = Sched<L>;
    static constexpr int T = L / P;                                   // threads per line
    static constexpr int LINE_ELEMS = COL ? L * NB : L + 2 * (L / 32); // float2 per tile (COL) / line (row)

    __device__ static __forceinline__ int addr(int slot, int off)
    {
        return COL ? slot * NB + off : slot + ((slot >> 5) << 1) + off;
    }
    // Butterfly handled by thread tt as its u-th one in group G.  Radix-16 groups: one butterfly per
    // thread, bf = tt.  The remainder group (radix R < 16, always last, m = 1) has P/R per thread:
    //   CONTIG  : consecutive ones, so that in the last group's layout a thread owns the 16 adjacent
    //             slots 16 tt .. 16 tt + 15: its exchange with the previous group stays inside that
    //             group's block (warp-local when the block has <= 512 slots), and global accesses
    //             are 128-byte runs that the row kernels stage through shared memory;
    //   !CONTIG : T apart (runs of R slots).  Kept for row tiles with R = 2 (L = 512, 8192), whose
    //             16-byte runs are already perfectly coalesced straight from registers (staging
    //             measured 15 % slower there), and for column tiles (no staging; L = 64 measured
    //             10 % slower with the consecutive assignment).
    static constexpr bool CONTIG = !COL && S::RLAST != 2;
    template <int G>
    __device__ static __forceinline__ int bfly(int tt, int u)
    {
        constexpr int R = S::radix(G);
        return (CONTIG && P / R > 1) ? tt * (P / R) + u : tt + u * T;
    }
    // slot of register i in the layout of group G
    template <int G>
    __device__ static __forceinline__ int slot(int tt, int i)
    {
        constexpr int R = S::radix(G), m = S::block(G) / R;
        const int u = i / R, c = i % R;
        const int bf = bfly<G>(tt, u);
        return (bf & ~(m - 1)) * R + (bf & (m - 1)) + c * m;
    }
    // Shared-memory address of register i in the layout of group G, split into a per-thread base (one
    // per butterfly u = i / R) and a compile-time offset (c = i % R), so that the 16 accesses of an
    // exchange use immediate offsets.  The row padding is separable: the butterfly's base slot is a
    // multiple of R m or has its low part < m, and m | 32, so ((base + c m) >> 5) = (base >> 5) + ((c m) >> 5).
    template <int G>
    __device__ static __forceinline__ int base_addr(int tt, int u, int off)
    {
        constexpr int R = S::radix(G), m = S::block(G) / R;
        const int bf = bfly<G>(tt, u);
        return addr((bf & ~(m - 1)) * R + (bf & (m - 1)), off);
    }
    template <int G>
    __host__ __device__ static constexpr int reg_offset(int c)
    {
        constexpr int R = S::radix(G), m = S::block(G) / R;
        return COL ? c * m * NB : c * m + (((c * m) >> 5) << 1);
    }
    template <int G>
    __device__ static __forceinline__ void to_smem(const float2* v, float2* s, int tt, int off)
    {
        constexpr int R = S::radix(G);
#pragma unroll
        for (int u = 0; u < P / R; ++u) {
            float2* b = s + base_addr<G>(tt, u, off);
#pragma unroll
            for (int c = 0; c < R; ++c) b[reg_offset<G>(c)] = v[u * R + c];
        }
    }
    template <int G>
    __device__ static __forceinline__ void from_smem(float2* v, const float2* s, int tt, int off)
    {
        constexpr int R = S::radix(G);
#pragma unroll
        for (int u = 0; u < P / R; ++u) {
            const float2* b = s + base_addr<G>(tt, u, off);
#pragma unroll
            for (int c = 0; c < R; ++c) v[u * R + c] = b[reg_offset<G>(c)];
        }
    }
    template <int G, int DIR>
    __device__ static __forceinline__ void butterflies(float2* v, int tt, const float2* __restrict__ tw)
    {
        constexpr int R = S::radix(G), m = S::block(G) / R;
#pragma unroll
        for (int u = 0; u < P / R; ++u) {
            float2* w = v + u * R;
            const int j = bfly<G>(tt, u) & (m - 1);
            if (DIR < 0 && m > 1) {
#pragma unroll
                for (int c = 1; c < R; ++c)
                    w[c] = cmulc(w[c], __ldg(tw + S::twoff(G) + (group_freq<R>(c) - 1) * m + j));
            }
            group<Split<R>::RA, Split<R>::RB, DIR, 1>(w);
            if (DIR > 0 && m > 1) {
#pragma unroll
                for (int c = 1; c < R; ++c)
                    w[c] = cmul(w[c], __ldg(tw + S::twoff(G) + (group_freq<R>(c) - 1) * m + j));
            }
        }
    }
    // An exchange between groups GA and GB only moves data inside blocks of block(min(GA, GB)) slots,
    // i.e. among block/16 consecutive threads of a row tile: at most one warp when block <= 512.  Such
    // exchanges need __syncwarp() only; a CTA-wide one additionally needs a leading __syncthreads()
    // when the previous shared-memory activity was only warp-synchronised (PREV_WIDE = false).
    template <int GA, int GB>
    __host__ __device__ static constexpr bool local_exchange()
    {
        return !COL && S::block(GA < GB ? GA : GB) / P <= 32 &&
               (CONTIG || (S::radix(GA) == 16 && S::radix(GB) == 16));
    }
    template <bool LOCAL>
    __device__ static __forceinline__ void xsync()
    {
        if (LOCAL) __syncwarp();
        else __syncthreads();
    }
    // forward: v in the layout of group 0  ->  v in the layout of the last group
    template <int G = 0, bool PREV_WIDE = COL>
    __device__ static __forceinline__ void forward(float2* v, float2* s, int tt, int off, const float2* __restrict__ tw)
    {
        butterflies<G, +1>(v, tt, tw);
        if constexpr (G + 1 < S::NG) {
            constexpr bool loc = local_exchange<G, G + 1>();
            if (!loc && !PREV_WIDE) __syncthreads();
            to_smem<G>(v, s, tt, off);
            xsync<loc>();
            from_smem<G + 1>(v, s, tt, off);
            xsync<loc>();
            forward<G + 1, !loc>(v, s, tt, off, tw);
        }
    }
    // inverse (unnormalised): v in the layout of the last group  ->  layout of group 0
    template <int G = S::NG - 1, bool PREV_WIDE = COL>
    __device__ static __forceinline__ void inverse(float2* v, float2* s, int tt, int off, const float2* __restrict__ tw)
    {
        butterflies<G, -1>(v, tt, tw);
        if constexpr (G > 0) {
            constexpr bool loc = local_exchange<G, G - 1>();
            if (!loc && !PREV_WIDE) __syncthreads();
            to_smem<G>(v, s, tt, off);
            xsync<loc>();
            from_smem<G - 1>(v, s, tt, off);
            xsync<loc>();
            inverse<G - 1, !loc>(v, s, tt, off, tw);
        }
    }
};

} // namespace fx
} // namespace dop
