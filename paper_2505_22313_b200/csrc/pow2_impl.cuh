// pow2_impl.cuh -- register-blocked tile-pass kernels for power-of-two digits (the fast path).
//
// Same pass semantics and slot order as kernels_generic.cu (one CTA = one tile, one read + one
// write of the field, fused pointwise ops; Eq. 1-4, PAPER.md:200 row-column 2-D
// FFT), so a plan may mix the two kernel families pass by pass.  Every thread keeps 16 points in
// registers (fft_regs.cuh) and moves them straight between registers and global memory:
//   column-type tile: 16 adjacent lines x L slots, lanes run over the 16 lines (128-byte segments);
//   row-type tile   : LINES contiguous lines of L points, lanes run over consecutive points.
// Everything structural is a template parameter (digit length, tile type, fused-op variant,
// boundary-twiddle mode), so the emitted code has no per-element branches and its addresses are
// base + compile-time multiples of one stride.
#pragma once
#include <atomic>

#include "dop_internal.h"
#include "fft_regs.cuh"

namespace dop {

// "this (digit, variant, twiddle mode, bundle) combination is not instantiated": the dispatcher then
// falls back to the generic kernel.  Deliberately not a value of the CUDA error enum, so that a real
// launch failure can never be mistaken for it.
constexpr cudaError_t kNotInstantiated = (cudaError_t)0x7fff0001;

// cudaFuncSetAttribute acts on the CURRENT device only: remember, per kernel instantiation, on which
// devices it has been applied (a second plan on another GPU of the same process must set it again).
struct AttrOnce {
    std::atomic<unsigned long long> mask{0};
    template <class F>
    cudaError_t ensure(int dev, F&& set)
    {
        const unsigned long long bit = (dev >= 0 && dev < 64) ? 1ull << dev : 0ull;
        if (bit != 0 && (mask.load(std::memory_order_acquire) & bit)) return cudaSuccess;
        cudaError_t e = set();
        if (e == cudaSuccess && bit != 0) mask.fetch_or(bit, std::memory_order_release);
        return e;
    }
};

using fx::P;

// fused-op variants (what is fused around the digit DFT(s) of a pass)
enum Variant : int {
    V_FWD = 0,     // c64 -> DFT -> c64
    V_INV = 1,     // c64 -> IDFT -> c64
    V_LOSS = 2,    // c64 -> IDFT -> |u|^2, loss, seed -> DFT -> c64          (F6, F7, A1)
    V_H = 3,       // c64 -> DFT -> (x) H or conj H -> IDFT -> c64            (F4 / A3)
    V_GAUSS = 4,   // c64 -> DFT -> (x) Gaussian -> IDFT -> c64               (F0 / A6)
    V_HEIGHT = 5,  // h -> exp(i Phi) -> DFT -> c64                           (F1, F2)
    V_LDOTHER = 6, // seed (2 dL/dI u) or real plane -> DFT -> c64            (runtime load_op)
    V_GRAD = 7,    // c64 -> IDFT -> dL/dh (+=)                               (A5)
    V_STOTHER = 8  // c64 -> IDFT -> (u, |u|^2) or real plane                 (runtime store_op)
};
// boundary twiddle T_j = W_{N_j}^{k_j r_j} of a non-last digit
enum TwbMode : int {
    TWB_NONE = 0,
    TWB_TILE = 1, // r_j is constant over the tile (y digits): table [r][slot], tile's row contiguous
    TWB_LANE = 2  // r_j = the lane's line index (x digits):   table [slot][r], lanes coalesced
};

__host__ __device__ constexpr int variant_dir1(int v)
{
    return (v == V_FWD || v == V_H || v == V_GAUSS || v == V_HEIGHT || v == V_LDOTHER) ? +1 : -1;
}
__host__ __device__ constexpr int variant_dir2(int v) { return v == V_LOSS ? +1 : (v == V_H || v == V_GAUSS) ? -1 : 0; }

__host__ __device__ constexpr int row_lines(int L) { return L >= 4096 ? 1 : 4096 / L; }
__host__ __device__ constexpr int tile_threads(int L, bool col, int nb = 16) { return col ? nb * (L / P) : row_lines(L) * (L / P); }
// resident CTAs per SM the register allocation is asked to allow
#ifndef DOP_RESIDENT_THREADS
#define DOP_RESIDENT_THREADS 1024 // 65536 regs / 1024 threads -> 64 registers per thread (measured best: 768 -> 1024 gave C4 +10%)
#endif
#ifndef DOP_LOSS_THREADS
#define DOP_LOSS_THREADS 512 // the loss variant keeps 16 points + 16 target values live: 128 registers, no spill
#endif
#ifndef DOP_HEAVY_THREADS
#define DOP_HEAVY_THREADS DOP_RESIDENT_THREADS // register budget of the loss / H / Gaussian variants
#endif
__host__ __device__ constexpr int min_blocks(int L, bool col, int v = 0, int nb = 16)
{
    const int rt = v == 2 ? DOP_LOSS_THREADS : (v == 3 || v == 4) ? DOP_HEAVY_THREADS : DOP_RESIDENT_THREADS;
    const int th = tile_threads(L, col, nb);
    return th >= 512 ? (th >= 1024 ? 1 : 2) : (rt / th > 0 ? rt / th : 1);
}

// Cache-hinted global accesses as plain (non-volatile) asm so the unrolled loads can be scheduled
// freely; the loaded field elements are overwritten later by this same thread (a data dependence).
__device__ __forceinline__ float2 ld_cg(const float2* p) // L2 only: streaming field, keeps L1 for tables
{
    float2 v;
    asm("ld.global.cg.v2.f32 {%0,%1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ void st_cg(float2* p, float2 v)
{
    asm volatile("st.global.cg.v2.f32 [%0], {%1,%2};" ::"l"(p), "f"(v.x), "f"(v.y));
}

__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// Inter-CTA software pipelining: CTA b asks L2 for the lines that CTA b + pf_ahead (a couple of
// waves later) will load, so DRAM keeps streaming while the resident CTAs compute and the later
// CTA's loads are L2 hits.  One 128-byte line per thread covers the whole tile.
template <bool COL, int THREADS, int NLINES, bool WANT_FIELD, bool WANT_HEIGHT, bool WANT_PLANE>
__device__ __forceinline__ void prefetch_tile(const PassDesc& p, int slots_per_thread, int L)
{
#ifdef DOP_NO_PF
    return;
#endif
    if (p.pf_ahead <= 0) return;
    unsigned t = blockIdx.x + (unsigned)p.pf_ahead;
    if (t >= gridDim.x) return;
    const unsigned ncg = (unsigned)p.n_cgroups, nm = (unsigned)p.n_m;
    const long long cg = (long long)(t % ncg) + p.cg0;
    t /= ncg;
    const long long m = t % nm;
    const long long o = (long long)(t / nm) + p.o0;
    const long long base = o * p.SO + m * p.SM + cg * NLINES * p.SCc;
    const int tid = threadIdx.x;
    if (COL) { // NLINES adjacent columns of one slot = NLINES/16 lines of the field, one per thread
        constexpr int PER = NLINES / 16;
        const int piece = tid % PER;
        for (int k = 0; k < slots_per_thread; ++k) {
            const long long off = base + (long long)(tid / PER + k * (THREADS / PER)) * p.es;
            if (WANT_FIELD) prefetch_l2(p.field + off + piece * 16);
            if (piece * 32 < NLINES) {
                if (WANT_HEIGHT) prefetch_l2(p.height + off + piece * 32);
                if (WANT_PLANE) prefetch_l2(p.plane_in + off + piece * 32);
            }
        }
    } else { // the tile is NLINES * L contiguous points = THREADS lines of 16 complex64
        const long long off = base + (long long)tid * 16;
        if (WANT_FIELD) prefetch_l2(p.field + off);
        if (tid * 32 < NLINES * L) {
            if (WANT_HEIGHT) prefetch_l2(p.height + base + (long long)tid * 32);
            if (WANT_PLANE) prefetch_l2(p.plane_in + base + (long long)tid * 32);
        }
    }
}

// Field accesses: column-type tiles stream through L2 only (each 128-byte segment is used once;
// L1 is kept for the twiddle tables: y passes 0.244 -> 0.231 ms at C2).  Row-type tiles keep the
// default policy; evict-first / L2-only hints on them and on the fp32 planes measured 10-40% slower.
template <bool CG>
__device__ __forceinline__ float2 field_ld(const float2* p) { return CG ? ld_cg(p) : *p; }
template <bool CG>
__device__ __forceinline__ void field_st(float2* p, float2 v)
{
    if (CG) st_cg(p, v);
    else *p = v;
}

// (cos 2 pi f, sin 2 pi f) for |f| < 2^20 turns, polynomial form: quadrant q = round(4f) mod 4 by the magic-number
// trick (no F2I / FRND), residue |r| <= 1/8 turn, Taylor polynomials in r^2 (truncation 2e-9 / 2.4e-8), then the
// quadrant rotation by selects and sign flips.  ~23 instructions against ~30 for the library sincospif, which also
// has to handle arbitrary arguments.  Used for the phase of H (apply_h; sincos_fixed / h_fixed_nb carry the same
// polynomials): there the hardware sine / cosine measured no gain (three MUFU operations per H value on the
// 16-lane pipe cost what the polynomial's FMAs do: C4 (x) H 17.0 -> 17.5-18.4 ms).
__device__ __forceinline__ void sincos_turn_poly(float f, float* sn, float* cs)
{
    const float MAGIC = 12582912.0f;                 // 1.5 * 2^23
    const float t = fmaf(f, 4.0f, MAGIC);            // low mantissa bits = round(4 f) (two's complement)
    const int q = __float_as_int(t);
    const float r = fmaf(t - MAGIC, -0.25f, f);      // exact: f - q/4
    const float r2 = r * r;
    float sp = fmaf(r2, 42.05869394489765f, -76.70585975306136f);   // (2pi)^9/9!, -(2pi)^7/7!
    sp = fmaf(sp, r2, 81.60524927607504f);                          // (2pi)^5/5!
    sp = fmaf(sp, r2, -41.34170224039976f);                         // -(2pi)^3/3!
    sp = fmaf(sp, r2, 6.283185307179586f);                          // 2pi
    const float s = sp * r;
    float cp = fmaf(r2, 60.24464137187666f, -85.45681720669373f);   // (2pi)^8/8!, -(2pi)^6/6!
    cp = fmaf(cp, r2, 64.93939402266829f);                          // (2pi)^4/4!
    cp = fmaf(cp, r2, -19.739208802178716f);                        // -(2pi)^2/2!
    const float c = fmaf(cp, r2, 1.0f);
    // q mod 4: 0 -> (c, s), 1 -> (-s, c), 2 -> (-c, -s), 3 -> (s, -c)
    const bool odd = (q & 1) != 0;
    const float co = odd ? s : c, so = odd ? c : s;
    *cs = __int_as_float(__float_as_int(co) ^ (((q + 1) & 2) << 30));
    *sn = __int_as_float(__float_as_int(so) ^ ((q & 2) << 30));
}
// u0 = exp(i Phi) (F2, and its recomputation in A5): the residue r = f - rint(f) by the magic-number trick (exact),
// then the hardware sine / cosine (MUFU.SIN / MUFU.COS behind sin.approx / cos.approx; measured on B200 over 2^26
// arguments: max error 3.4e-7, rms 1.2e-7, including the rounding of 2 pi r) -- 8 instructions against 23, in
// passes that are bound by instruction issue (C5 dL/dh pass 20.9 -> 18.7 ms, h -> exp(i Phi) 22.2 -> 21.2 ms).
// -DDOP_POLY_SINCOS keeps the polynomial form.
__device__ __forceinline__ void sincos_turn(float f, float* sn, float* cs)
{
#ifdef DOP_LIB_SINCOS
    sincospif(2.0f * f, sn, cs);
    return;
#endif
#ifndef DOP_POLY_SINCOS
    const float RND = 12582912.0f;                   // 1.5 * 2^23: (f + RND) - RND = rint(f)
    const float r = f - ((f + RND) - RND);           // exact (Sterbenz), |r| <= 1/2 turn
    const float x = r * 6.283185307179586f;
    *sn = __sinf(x);
    *cs = __cosf(x);
#else
    sincos_turn_poly(f, sn, cs);
#endif
}
// Any moderate argument in turns (|ph| < 2^20) needs no separate integer reduction: round(4 ph) mod 4
// is the quadrant whatever the integer part, and ph - round(4 ph)/4 is exact (Sterbenz).
__device__ __forceinline__ void sincos_turns(float ph, float* sn, float* cs) { sincos_turn(ph, sn, cs); }

// F4 / A3: v *= H (or conj H) / N; evanescent bins (a < 0) zeroed.  a and the phase z sqrt(a)
// are fp64; sqrt = fp32 rsqrt seed + one fp64 Newton step.
__device__ __forceinline__ float2 apply_h(float2 v, double c_minus_fx2, double fy2, double z, float scale, bool conj)
{
    const double a = c_minus_fx2 - fy2; // (1/lambda^2 - fx^2) - fy^2, the definition's own order
    if (a >= 0.0) {
        double s = 0.0;
        if (a > 0.0) {
            const double y = (double)rsqrtf((float)a);
            const double hy = 0.5 * y;
            s = a * y;                     // rel. error 2^-22 (fp32 rsqrt)
            s = fma(fma(-s, s, a), hy, s); // one Newton step: ~3e-14, i.e. < 6e-9 turns at z sqrt(a) = 1.8e5
        }
        const double turns = z * s;
        const double RND = 6755399441055744.0;                    // 1.5 * 2^52: (x + RND) - RND = rint(x)
        const float f = (float)(turns - ((turns + RND) - RND));   // fractional turn, |f| <= 0.5
        float sn, cs;
        sincos_turn_poly(f, &sn, &cs);
        const float2 h = make_float2(cs * scale, (conj ? -sn : sn) * scale);
        return fx::cmul(v, h);
    }
    return make_float2(0.0f, 0.0f);
}

// (cos, sin) of a turn fraction given as a 32-bit fixed-point number ph / 2^32: nearest quadrant from
// the top bits, signed residue (units of 2^-32 turn) rounded to 23 bits and turned into a float with
// the magic-number trick (no conversion-pipe instruction), then the polynomials of sincos_turn.
__device__ __forceinline__ void sincos_fixed(unsigned ph, float* sn, float* cs)
{
    const unsigned t = ph + 0x20000000u;
    const int q = (int)(t >> 30);
    const int ri = (int)(t & 0x3FFFFFFFu) - 0x20000000;                 // [-2^29, 2^29)
    const float rf = __int_as_float(0x4B400000 + ((ri + 64) >> 7)) - 12582912.0f; // exact, units of 2^-25 turn
    const float r = rf * 2.98023223876953125e-8f;                      // 2^-25
    const float r2 = r * r;
    float sp = fmaf(r2, 42.05869394489765f, -76.70585975306136f);
    sp = fmaf(sp, r2, 81.60524927607504f);
    sp = fmaf(sp, r2, -41.34170224039976f);
    sp = fmaf(sp, r2, 6.283185307179586f);
    const float s = sp * r;
    float cp = fmaf(r2, 60.24464137187666f, -85.45681720669373f);
    cp = fmaf(cp, r2, 64.93939402266829f);
    cp = fmaf(cp, r2, -19.739208802178716f);
    const float c = fmaf(cp, r2, 1.0f);
    const bool odd = (q & 1) != 0;
    const float co = odd ? s : c, so = odd ? c : s;
    *cs = __int_as_float(__float_as_int(co) ^ (((q + 1) & 2) << 30));
    *sn = __int_as_float(__float_as_int(so) ^ ((q & 2) << 30));
}

// apply_h with the phase taken in fixed point: u = fma(sqrt(a), z 2^32, 1.5 2^52) holds
// round(turns 2^32) in its low word (valid while |turns| < 2^19; the plan checks |z|/lambda), and the
// fp32 rsqrt seed goes through bit-level fp64 <-> fp32 conversions.  Per point this replaces three
// of the four conversion-pipe operations (16 lanes/clk/SM) and three fp64 operations by ~14 integer /
// fp32 ones.
__device__ __forceinline__ float2 apply_h_fixed(float2 v, double c_minus_fx2, double fy2, double z32, float scale, bool conj)
{
    const double a = c_minus_fx2 - fy2;
    if (a >= 0.0) {
        unsigned ph = 0u;
        if (a > 1e-30) {
            const int hi = __double2hiint(a), lo = __double2loint(a);
            const float af = __int_as_float(((hi - 0x38000000) << 3) | (int)((unsigned)lo >> 29)); // truncated (float)a
            const int yb = __float_as_int(rsqrtf(af));
            const double y = __hiloint2double((yb >> 3) + 0x38000000, yb << 29);                    // exact (double)y
            double s = a * y;
            s = fma(fma(-s, s, a), 0.5 * y, s);
            ph = (unsigned)__double2loint(fma(s, z32, 6755399441055744.0));
        }
        float sn, cs;
        sincos_fixed(ph, &sn, &cs);
        const float2 h = make_float2(cs * scale, (conj ? -sn : sn) * scale);
        return fx::cmul(v, h);
    }
    return make_float2(0.0f, 0.0f);
}

// Branch-free flavour of apply_h_fixed for kernels with registers to spare (tma_col.cuh): no divergent region
// around a point's chain, so the 16 chains of a thread interleave (ncu: the branchy form sits at 52 % issue
// utilisation with `wait` and `long_scoreboard` on top).  a < 0 runs the same arithmetic on garbage and the
// result is replaced by 0 with two selects; a == 0 gives s = a y = 0 exactly for any finite seed, i.e. H = 1.
// The 1/(ny nx) scale is folded into the polynomial coefficients (hk, prepared on the host: hk.s[k] =
// scale (2 pi)^(2k+1)/(2k+1)! signed, hk.c[k] likewise for the cosine), conj H into the sign of z32.
struct HCoef { float s[5], c[5]; };
__device__ __forceinline__ float2 h_fixed_nb(double c_minus_fx2, double fy2, double z32, const HCoef& hk)
{
    const double a = c_minus_fx2 - fy2;
    const int hi = __double2hiint(a), lo = __double2loint(a);
    const float af = __int_as_float(((hi - 0x38000000) << 3) | (int)((unsigned)lo >> 29)); // truncated (float)a, a > 0
    const int yb = __float_as_int(rsqrtf(af));
    const double y = __hiloint2double((yb >> 3) + 0x38000000, yb << 29);                    // exact (double)y
    double s = a * y;
    s = fma(fma(-s, s, a), 0.5 * y, s);
    const unsigned ph = (unsigned)__double2loint(fma(s, z32, 6755399441055744.0));
    const bool prop = a >= 0.0; // evanescent bins are zeroed
    const unsigned t = ph + 0x20000000u;
    const int q = (int)(t >> 30);
    const int ri = (int)(t & 0x3FFFFFFFu) - 0x20000000;
    const float rf = __int_as_float(0x4B400000 + ((ri + 64) >> 7)) - 12582912.0f;
    const float r = rf * 2.98023223876953125e-8f;
    const float r2 = r * r;
    float sp = fmaf(r2, hk.s[4], hk.s[3]);
    sp = fmaf(sp, r2, hk.s[2]);
    sp = fmaf(sp, r2, hk.s[1]);
    sp = fmaf(sp, r2, hk.s[0]);
    const float sn0 = sp * r;
    float cp = fmaf(r2, hk.c[4], hk.c[3]);
    cp = fmaf(cp, r2, hk.c[2]);
    cp = fmaf(cp, r2, hk.c[1]);
    const float cs0 = fmaf(cp, r2, hk.c[0]);
    const bool odd = (q & 1) != 0;
    const float co = odd ? sn0 : cs0, so = odd ? cs0 : sn0;
    const float hx = prop ? __int_as_float(__float_as_int(co) ^ (((q + 1) & 2) << 30)) : 0.0f;
    const float hy = prop ? __int_as_float(__float_as_int(so) ^ ((q & 2) << 30)) : 0.0f;
    return make_float2(hx, hy);
}
__device__ __forceinline__ float2 apply_h_fixed_nb(float2 v, double c_minus_fx2, double fy2, double z32, const HCoef& hk)
{
    return fx::cmul(v, h_fixed_nb(c_minus_fx2, fy2, z32, hk));
}

// Height of fine-grid point (row, x) from the caller's design layout: nearest-neighbour up-sampling of the
// coarse feature grid (the adjoint is the sum-pool in the gradient store) and gray
// levels times a height step.
__device__ __forceinline__ float ld_layout(const void* base, int dtype, float step, int up_lg, long long cnx, long long row,
                                           long long x)
{
    const long long ci = (row >> up_lg) * cnx + (x >> up_lg);
    if (dtype == DOP_LAYOUT_F32) return __ldg((const float*)base + ci);
    if (dtype == DOP_LAYOUT_U8) return step * (float)__ldg((const unsigned char*)base + ci);
    return step * (float)__ldg((const unsigned short*)base + ci);
}

// Sum over the r = 2^up_lg adjacent lanes that hold r adjacent x (deterministic xor tree; every lane gets the sum)
__device__ __forceinline__ float pool_lanes(float g, int up_lg, unsigned mask)
{
    for (int d = 1; d < (1 << up_lg); d <<= 1) g += __shfl_xor_sync(mask, g, d);
    return g;
}

// Adam (Kingma & Ba 2014, Alg. 1) on one element: returns the updated layout value
__device__ __forceinline__ float adam_update(float g, float h, float* m, float* v, float b1, float b2, float c1, float c2,
                                             float a1, float rb2, float eps)
{
    const float mn = fmaf(b1, *m, c1 * g);
    const float vn = fmaf(b2, *v, c2 * g * g);
    *m = mn;
    *v = vn;
    return h - a1 * mn / (sqrtf(vn * rb2) + eps);
}

// ---- the tile-pass kernel -------------------------------------------------------------------
template <int L, bool COL, int V, int TWB, int NB>
__global__ void __launch_bounds__(tile_threads(L, COL, NB), min_blocks(L, COL, V, NB))
pow2_kernel(const __grid_constant__ PassDesc p)
{
    using TL = fx::Tile<L, COL, NB>;
    using S = fx::Sched<L>;
    constexpr int T = L / P;            // threads per line
    constexpr int GL = S::NG - 1;       // last group
    constexpr int RL = TL::CONTIG ? P : S::radix(GL); // adjacent slots per run in the last group's layout (fft_regs.cuh bfly)
    constexpr int DIR1 = variant_dir1(V), DIR2 = variant_dir2(V);
    constexpr int LAST = DIR2 != 0 ? DIR2 : DIR1;
    constexpr int LINES = row_lines(L);
    // L2-only field accesses: column tiles except the two variants where it measured slower (C4:
    // loss pass 32 -> 45 ms, height pass 12.5 -> 13.7 ms)
    constexpr bool CG = COL && V != V_LOSS && V != V_HEIGHT;
    // Row tiles: in the last group's layout a thread owns 16 adjacent slots (128 bytes) and a warp 512
    // adjacent slots (4 KiB of contiguous memory: part of one line when T >= 32, 32/T whole lines
    // otherwise).  Global accesses in that layout go through the exchange buffer: the warp moves its 4 KiB
    // with LDG/STG.128 that each cover 512 contiguous bytes, and the threads pick up / drop their own
    // 16 slots in shared memory (x passes at C4: 0.61 / 0.72 -> 0.88 / 0.99 of measured copy bandwidth
    // against 16-byte accesses to 32 different lines per instruction).  Only the warp's own slots are
    // touched, so the hazards are warp-local.
    constexpr bool STAGE = !COL && TL::CONTIG; // (L = 512, 8192: runs of 2 slots, coalesced as they are)
    extern __shared__ float2 s[];

    // ---- which tile (same enumeration as the generic kernel)
    // (32-bit divisions: the launcher guarantees fewer than 2^31 tiles)
    unsigned t = blockIdx.x;
    const unsigned ncg = (unsigned)p.n_cgroups, nm = (unsigned)p.n_m;
    const long long cg = (long long)(t % ncg) + p.cg0;
    t /= ncg;
    const long long m = t % nm;
    const long long o = (long long)(t / nm) + p.o0;
    const int tid = threadIdx.x;
    const int sub = COL ? (tid % NB) : (tid / T); // column in the bundle / line in the tile
    const int tt = COL ? (tid / NB) : (tid % T);
    const long long line = cg * (COL ? NB : LINES) + sub;
    const long long es = COL ? p.es : 1;
    const long long tbase = o * p.SO + m * p.SM + line * p.SCc;
    const int soff = COL ? sub : sub * TL::LINE_ELEMS;
    const float2* __restrict__ tw = p.tw_g;

    // Register i holds slot tt + i T in the first group's layout and slot tt RL + kL(i) in the
    // last group's (fft_regs.cuh Tile::slot with m = T resp. m = 1).
    const long long b0 = tbase + (long long)tt * es;
    const long long bL = tbase + (long long)(tt * RL) * es;
#define DOP_K0(i) ((i) * T)
#define DOP_KL(i) (((i) / RL) * (T * RL) + (i) % RL)
    // Addresses are walked with running offsets (one 64-bit add per access) rather than
    // i * stride products: the stride of a column tile is a run-time 64-bit value.
    const long long step0 = (long long)T * es;                  // first-group layout: register i -> i + 1
    const long long stepLr = (long long)(T * RL - (RL - 1)) * es; // last-group layout: end of a run of RL -> next run
#define DOP_NEXT_L(ptr, i) ptr += ((((i) % RL) == RL - 1) ? stepLr : es)

    // staging geometry (row tiles): shared-memory index (float2 units) of element e (even, 0..510) of the
    // warp's 512 slots, and the global offset of the warp's first slot
    const int lane = tid & 31;
    auto stg_addr = [&](int e) -> int {
        if (T >= 32) return soff + TL::addr((tt - lane) * P + e, 0);
        return (sub - lane / (T >= 32 ? 1 : T) + e / L) * TL::LINE_ELEMS + TL::addr(e % L, 0);
    };
    const long long stg_base = bL - (long long)lane * P;

    // boundary twiddle of the element in register i (last-group layout)
    const float2* __restrict__ twp = nullptr;
    unsigned tws = 1;
    if (TWB == TWB_TILE) {
        twp = p.tw_b2 + m * L + tt * RL;
    } else if (TWB == TWB_LANE) {
        tws = (unsigned)p.NC;
        twp = p.tw_b2 + line + (long long)(tt * RL) * tws;
    }

    // Design-layout addressing (dop_plan_desc.upsample / layout_dtype; only the variants that touch the
    // height plane, a real plane or dL/dh): fine-grid (row, x) of register i in the first group's layout
    constexpr bool LAYV = V == V_HEIGHT || V == V_GRAD || V == V_LDOTHER || V == V_STOTHER;
    const bool lay = LAYV && (p.up_lg | p.h_dtype | p.coarse_in | p.pool_out) != 0; // uniform over the grid
    long long hrow = 0, hx0 = 0;
    if (lay) {
        if (COL) { hrow = o; hx0 = m * p.SM + line + (long long)tt * es; }
        else { hrow = line / p.lpr; hx0 = (line - hrow * p.lpr) * L + tt; }
    }
    const long long hxs = COL ? (long long)T * es : T;

    // (row tiles only: on column tiles it measured as a loss or as a wash that over-fetches DRAM, and
    // its registers cost the fused variants up to 25 %)
    if (!COL)
        prefetch_tile<COL, tile_threads(L, COL, NB), LINES, (V != V_HEIGHT && V != V_LDOTHER),
                      (V == V_HEIGHT || V == V_GRAD), (V == V_LOSS)>(p, 1, L);

    // Touch the tables this tile will need after its DFT now, so they are in L1 by then.
    if (TWB == TWB_TILE && LAST > 0) {
#pragma unroll
        for (int i = 0; i < P; i += (RL >= 16 ? 16 : RL)) asm volatile("prefetch.global.L1 [%0];" ::"l"(twp + DOP_KL(i)));
    }
    if (V == V_H) {
        const double* fyp = p.fy2 + o * p.row_o + m * p.row_m + tt * RL;
#pragma unroll
        for (int i = 0; i < P; i += (RL >= 16 ? 16 : RL)) asm volatile("prefetch.global.L1 [%0];" ::"l"(fyp + DOP_KL(i)));
    }

    __shared__ double red[32];                                     // V_LOSS: per-warp partial sums
    constexpr int NW = (tile_threads(L, COL, NB) + 31) / 32;
    constexpr bool LOSS_DEFER = S::NG > 1 && !TL::template local_exchange<0, 1>();
    float2 v[P];
    // ---- load (+ prologue op, + conj boundary twiddle before an inverse DFT)
    if (DIR1 > 0) {
        long long off = b0;
        if ((V == V_HEIGHT && lay) || (V == V_LDOTHER && p.coarse_in)) {
            // design layout: nearest up-sampling / gray levels inside the read (kept apart from the plain loops
            // below, whose shape the row kernels are sensitive to)
#pragma unroll
            for (int i = 0; i < P; ++i, off += step0) {
                if (V == V_HEIGHT) {
                    const float hv = ld_layout(p.height, p.h_dtype, p.h_step, p.up_lg, p.cnx, hrow, hx0 + i * hxs);
                    sincos_turns(hv * p.phase_coef, &v[i].y, &v[i].x);
                } else {
                    v[i] = make_float2(ld_layout(p.plane_in, p.h_dtype, p.h_step, p.up_lg, p.cnx, hrow, hx0 + i * hxs), 0.0f);
                }
            }
        } else {
#pragma unroll
        for (int i = 0; i < P; ++i, off += step0) {
            if (V == V_HEIGHT) {
                const float ph = __ldg(p.height + off) * p.phase_coef; // Eq. (1) in turns
                sincos_turns(ph, &v[i].y, &v[i].x);                // Eq. (2), E_in = 1
            } else if (V == V_LDOTHER) {
                if (p.load_op == LD_SEED) {
                    const float2 u = field_ld<CG>(p.field + off);
                    const float g = 2.0f * __ldg(p.plane_in + off);
                    v[i] = make_float2(g * u.x, g * u.y);
                } else if (p.load_op == LD_SEED_SIMSE) { // Eq. (6): 2 dL/dI = c0 + cI I + cT T
                    const float2 u = field_ld<CG>(p.field + off);
                    const float I = u.x * u.x + u.y * u.y;
                    const float g = fmaf(__ldg(p.coef + 1), I, fmaf(__ldg(p.coef + 2), __ldg(p.plane_in + off), __ldg(p.coef)));
                    v[i] = make_float2(g * u.x, g * u.y);
                } else {
                    v[i] = make_float2(__ldg(p.plane_in + off), 0.0f);
                }
            } else {
                v[i] = field_ld<CG>(p.field + off);
            }
        }
        }
    } else {
        if (STAGE) {
            const float2* g0 = p.field + stg_base; // the warp's 512 slots
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int e = j * 64 + 2 * lane;
                *reinterpret_cast<float4*>(s + stg_addr(e)) = *reinterpret_cast<const float4*>(g0 + e);
            }
            __syncwarp();
            const float4* own = reinterpret_cast<const float4*>(s + soff + TL::addr(tt * P, 0));
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const float4 w = own[q];
                v[2 * q] = make_float2(w.x, w.y);
                v[2 * q + 1] = make_float2(w.z, w.w);
            }
            __syncwarp();
        } else if (!COL) { // runs of RL = 2 slots: one float4 per lane, 512 contiguous bytes per warp instruction
#pragma unroll
            for (int i = 0; i < P; i += 2) {
                const float4 q = *reinterpret_cast<const float4*>(p.field + bL + DOP_KL(i));
                v[i] = make_float2(q.x, q.y);
                v[i + 1] = make_float2(q.z, q.w);
            }
        } else {
            const float2* lp = p.field + bL;
#pragma unroll
            for (int i = 0; i < P; ++i) {
                v[i] = field_ld<CG>(lp);
                DOP_NEXT_L(lp, i);
            }
        }
        if (TWB != TWB_NONE) {
#pragma unroll
            for (int i = 0; i < P; ++i) v[i] = fx::cmulc(v[i], __ldg(twp + (unsigned)DOP_KL(i) * tws));
        }
    }

    // (PREV_WIDE: no shared-memory activity yet, or it ended with a CTA barrier)
    if (DIR1 > 0) TL::template forward<0, true>(v, s, tt, soff, tw);
    else TL::template inverse<GL, !STAGE>(v, s, tt, soff, tw);

    // ---- middle op
    if (V == V_H) { // registers hold spectrum slots in the last group's layout; this is the last y digit
        const double* __restrict__ fyp = p.fy2 + o * p.row_o + m * p.row_m + tt * RL;
        const double cfx = p.inv_lam2 - __ldg(p.fx2 + line);
        const bool cj = p.mid_op == MID_HCONJ;
        if (p.h_fixed) {
            const double z32 = p.z * 4294967296.0;
#pragma unroll
            for (int i = 0; i < P; ++i) v[i] = apply_h_fixed(v[i], cfx, __ldg(fyp + DOP_KL(i)), z32, p.scale, cj);
        } else {
#pragma unroll
            for (int i = 0; i < P; ++i) v[i] = apply_h(v[i], cfx, __ldg(fyp + DOP_KL(i)), p.z, p.scale, cj);
        }
    } else if (V == V_GAUSS) {
        const float* __restrict__ gyp = p.gy + o * p.row_o + m * p.row_m + tt * RL;
        const float gxs = __ldg(p.gx + line) * p.scale;
#pragma unroll
        for (int i = 0; i < P; ++i) {
            const float g = gxs * __ldg(gyp + DOP_KL(i));
            v[i] = make_float2(v[i].x * g, v[i].y * g);
        }
    } else if (V == V_LOSS) { // registers hold spatial points in the first group's layout
        double acc = 0.0;
        long long off = b0;
#pragma unroll
        for (int i = 0; i < P; ++i, off += step0) {
            const float I = v[i].x * v[i].x + v[i].y * v[i].y; // F6
            const float d = I - __ldg(p.plane_in + off);      // F7
            acc += (double)d * (double)d;
            const float g = p.seed_coef * d;                    // A1: 2 gI = 4 (I - T)/N
            v[i] = make_float2(g * v[i].x, g * v[i].y);
            if (p.write_intensity) p.plane_out[off] = I;
        }
        // deterministic CTA reduction: warp shuffle tree, then thread 0 in warp order
        constexpr int NT = tile_threads(L, COL, NB);
        constexpr int SW = NT < 32 ? NT : 32;                         // a 16-thread CTA (L = 16, 16 columns) is half a warp
        constexpr unsigned SMASK = NT < 32 ? (1u << SW) - 1u : 0xffffffffu;
#pragma unroll
        for (int d = SW / 2; d > 0; d >>= 1) acc += __shfl_down_sync(SMASK, acc, d, SW);
        if ((tid & 31) == 0) red[tid >> 5] = acc;
        // The warp sums are added up by thread 0 after the forward DFT when its first exchange is CTA-wide (a barrier
        // between these writes and that read), so that no warp waits for the serial sum; else behind a barrier here.
        if (!LOSS_DEFER) {
            __syncthreads();
            if (tid == 0) {
                double r = 0.0;
                for (int w = 0; w < NW; ++w) r += red[w];
                p.loss_scratch[p.tile0 + blockIdx.x] = r;
            }
        }
    }

    if (DIR2 > 0) TL::template forward<0, COL>(v, s, tt, soff, tw);
    else if (DIR2 < 0) TL::template inverse<GL, COL>(v, s, tt, soff, tw);
    if (V == V_LOSS && LOSS_DEFER && tid == 0) {
        double r = 0.0;
        for (int w = 0; w < NW; ++w) r += red[w];
        p.loss_scratch[p.tile0 + blockIdx.x] = r;
    }

    // ---- store (+ boundary twiddle after a forward DFT, + epilogue op)
    if (LAST > 0) {
        if (TWB != TWB_NONE) {
#pragma unroll
            for (int i = 0; i < P; ++i) v[i] = fx::cmul(v[i], __ldg(twp + (unsigned)DOP_KL(i) * tws));
        }
        if (STAGE) { // (the last exchange of a row tile is warp-local and ended with a __syncwarp)
            float4* own = reinterpret_cast<float4*>(s + soff + TL::addr(tt * P, 0));
#pragma unroll
            for (int q = 0; q < 8; ++q) own[q] = make_float4(v[2 * q].x, v[2 * q].y, v[2 * q + 1].x, v[2 * q + 1].y);
            __syncwarp();
            float2* g0 = p.field + stg_base;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int e = j * 64 + 2 * lane;
                *reinterpret_cast<float4*>(g0 + e) = *reinterpret_cast<const float4*>(s + stg_addr(e));
            }
        } else if (!COL) {
#pragma unroll
            for (int i = 0; i < P; i += 2)
                *reinterpret_cast<float4*>(p.field + bL + DOP_KL(i)) = make_float4(v[i].x, v[i].y, v[i + 1].x, v[i + 1].y);
        } else {
            float2* sp = p.field + bL;
#pragma unroll
            for (int i = 0; i < P; ++i) {
                field_st<CG>(sp, v[i]);
                DOP_NEXT_L(sp, i);
            }
        }
    } else {
        long long off = b0;
        double st0 = 0.0, st1 = 0.0, st2 = 0.0, st3 = 0.0; // ST_C64_STATS: <I,T>, <I,I>, sum I, <T,T>
        if ((V == V_GRAD && (lay || p.adam_m != nullptr)) || (V == V_STOTHER && p.pool_out)) {
            // design-loop flavours of the two real-plane stores (kept apart from the plain loops below)
            const unsigned am = __activemask();
            const bool leader = ((COL ? sub : tt) & ((1 << p.up_lg) - 1)) == 0;
#pragma unroll
            for (int i = 0; i < P; ++i, off += step0) {
                if (V == V_GRAD) {
                    const float hv = lay ? ld_layout(p.height, p.h_dtype, p.h_step, p.up_lg, p.cnx, hrow, hx0 + i * hxs)
                                         : __ldg(p.height + off);
                    float sn, cs;
                    sincos_turns(hv * p.phase_coef, &sn, &cs);
                    float g = p.grad_coef * (cs * v[i].y - sn * v[i].x); // A5: c Im(conj(u0) g)
                    if (p.pool_out) { // adjoint of the nearest up-sampling along x; rows are pooled afterwards
                        g = pool_lanes(g, p.up_lg, am);
                        const long long ci = hrow * p.cnx + ((hx0 + i * hxs) >> p.up_lg);
                        if (leader) {
                            if (p.store_op == ST_GRAD_ACC) g += p.plane_out[ci];
                            p.plane_out[ci] = g;
                        }
                    } else {
                        if (p.store_op == ST_GRAD_ACC) g += __ldg(p.plane_out + off);
                        p.plane_out[off] = g;
                        if (p.adam_m != nullptr) // the optimiser step rides on the last wavelength's store
                            p.adam_h[off] = adam_update(g, hv, p.adam_m + off, p.adam_v + off, p.adam_b1, p.adam_b2, p.adam_c1,
                                                        p.adam_c2, p.adam_a1, p.adam_rb2, p.adam_eps);
                    }
                } else {
                    const float g = pool_lanes(v[i].x, p.up_lg, am);
                    if (leader) p.plane_out[hrow * p.cnx + ((hx0 + i * hxs) >> p.up_lg)] = g;
                }
            }
        } else {
#pragma unroll
        for (int i = 0; i < P; ++i, off += step0) {
            if (V == V_GRAD) {
                const float ph = __ldg(p.height + off) * p.phase_coef;
                float sn, cs;
                sincos_turns(ph, &sn, &cs); // u0 recomputed, not stored
                float g = p.grad_coef * (cs * v[i].y - sn * v[i].x); // A5: c Im(conj(u0) g)
                if (p.store_op == ST_GRAD_ACC) g += __ldg(p.plane_out + off);
                p.plane_out[off] = g;
            } else if (V == V_STOTHER) {
                if (p.store_op == ST_C64_INTENSITY) {
                    field_st<CG>(p.field + off, v[i]);
                    p.plane_out[off] = v[i].x * v[i].x + v[i].y * v[i].y;
                } else if (p.store_op == ST_C64_STATS) {
                    field_st<CG>(p.field + off, v[i]);
                    const float I = v[i].x * v[i].x + v[i].y * v[i].y;
                    const float Tv = __ldg(p.plane_in + off);
                    st0 += (double)I * (double)Tv;
                    st1 += (double)I * (double)I;
                    st2 += (double)I;
                    st3 += (double)Tv * (double)Tv;
                    if (p.write_intensity) p.plane_out[off] = I;
                } else {
                    p.plane_out[off] = v[i].x;
                }
            } else {
                field_st<CG>(p.field + off, v[i]);
            }
        }
        }
        if (V == V_STOTHER) {
            if (p.store_op == ST_C64_STATS) { // deterministic CTA reduction of the four plane sums
                __shared__ double sred[4][32];
                constexpr int NT = tile_threads(L, COL, NB);
                constexpr int SW = NT < 32 ? NT : 32;
                constexpr unsigned SMASK = NT < 32 ? (1u << SW) - 1u : 0xffffffffu;
#pragma unroll
                for (int d = SW / 2; d > 0; d >>= 1) {
                    st0 += __shfl_down_sync(SMASK, st0, d, SW);
                    st1 += __shfl_down_sync(SMASK, st1, d, SW);
                    st2 += __shfl_down_sync(SMASK, st2, d, SW);
                    st3 += __shfl_down_sync(SMASK, st3, d, SW);
                }
                if ((tid & 31) == 0) {
                    sred[0][tid >> 5] = st0; sred[1][tid >> 5] = st1; sred[2][tid >> 5] = st2; sred[3][tid >> 5] = st3;
                }
                __syncthreads();
                if (tid < 4) {
                    double r = 0.0;
                    constexpr int NW = (NT + 31) / 32;
                    for (int w = 0; w < NW; ++w) r += sred[tid][w];
                    p.loss_scratch[4 * (p.tile0 + blockIdx.x) + tid] = r;
                }
            }
        }
    }
#undef DOP_K0
#undef DOP_KL
#undef DOP_NEXT_L
}

// ---- digits of length 3 * 2^k: one radix-3 step fused in front of three register-blocked 2^k DFTs
// Column-type tiles, plain forward / inverse passes only (the plan puts the factor 3 in a
// non-last digit).  Slot order = the generic kernel's for the radix list (3, 4, 4, ...): slot
// c LP + i' holds output k = c + 3 k'(i').  Each thread keeps the three sub-tiles (48 points).
template <int LP, int V, int TWB, int NB>
__global__ void __launch_bounds__(NB * (LP / P), (512 / (NB * (LP / P))) > 0 ? (512 / (NB * (LP / P))) : 1)
pow2x3_kernel(const __grid_constant__ PassDesc p)
{
    using TL = fx::Tile<LP, true, NB>;
    using S = fx::Sched<LP>;
    constexpr int T = LP / P;
    constexpr int GL = S::NG - 1;
    constexpr int RL = S::radix(GL);
    constexpr int DIR = variant_dir1(V);
    constexpr float HS3 = 0.86602540378443864676f; // sqrt(3)/2
    extern __shared__ float2 s[];

    unsigned t = blockIdx.x;
    const unsigned ncg = (unsigned)p.n_cgroups, nm = (unsigned)p.n_m;
    const long long cg = (long long)(t % ncg) + p.cg0;
    t /= ncg;
    const long long m = t % nm;
    const long long o = (long long)(t / nm) + p.o0;
    const int tid = threadIdx.x;
    const int sub = tid % NB, tt = tid / NB;
    const long long line = cg * NB + sub;
    const long long es = p.es;
    const long long tbase = o * p.SO + m * p.SM + line * p.SCc;
    const float2* __restrict__ tw = p.tw_g;
    const float2* __restrict__ wL = p.wL; // W_L^q, L = 3 LP
#define DOP_K0(i) ((i) * T)
#define DOP_KL(i) (((i) / RL) * (T * RL) + (i) % RL)
    const float2* __restrict__ twp;
    unsigned tws = 1;
    if (TWB == TWB_TILE) {
        twp = p.tw_b2 + m * (3 * LP) + tt * RL;
    } else {
        tws = (unsigned)p.NC;
        twp = p.tw_b2 + line + (long long)(tt * RL) * tws;
    }

    float2 v[3][P];
    if (DIR > 0) {
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int i = 0; i < P; ++i) v[c][i] = ld_cg(p.field + tbase + (long long)(c * LP + tt + DOP_K0(i)) * es);
        // radix-3 step (block length L, stride LP), outputs c = 1, 2 times W_L^{j c}
#pragma unroll
        for (int i = 0; i < P; ++i) {
            const int j = tt + DOP_K0(i);
            const float2 a = v[0][i], b = v[1][i], c = v[2][i];
            const float2 t1 = fx::cadd(b, c), d = fx::csub(b, c);
            const float2 t2 = make_float2(a.x - 0.5f * t1.x, a.y - 0.5f * t1.y);
            const float2 t3 = make_float2(HS3 * d.x, HS3 * d.y);
            v[0][i] = fx::cadd(a, t1);
            v[1][i] = fx::cmul(make_float2(t2.x + t3.y, t2.y - t3.x), __ldg(wL + j));     // t2 - i t3
            v[2][i] = fx::cmul(make_float2(t2.x - t3.y, t2.y + t3.x), __ldg(wL + 2 * j)); // t2 + i t3
        }
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            TL::template forward<0>(v[c], s, tt, sub, tw);
#pragma unroll
            for (int i = 0; i < P; ++i) {
                const float2 w = __ldg(twp + (unsigned)(c * LP + DOP_KL(i)) * tws);
                st_cg(p.field + tbase + (long long)(c * LP + tt * RL + DOP_KL(i)) * es, fx::cmul(v[c][i], w));
            }
        }
    } else {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
#pragma unroll
            for (int i = 0; i < P; ++i) {
                const float2 w = __ldg(twp + (unsigned)(c * LP + DOP_KL(i)) * tws);
                v[c][i] = fx::cmulc(ld_cg(p.field + tbase + (long long)(c * LP + tt * RL + DOP_KL(i)) * es), w);
            }
            TL::template inverse<GL>(v[c], s, tt, sub, tw);
        }
#pragma unroll
        for (int i = 0; i < P; ++i) {
            const int j = tt + DOP_K0(i);
            const float2 a = v[0][i];
            const float2 b = fx::cmulc(v[1][i], __ldg(wL + j));
            const float2 c = fx::cmulc(v[2][i], __ldg(wL + 2 * j));
            const float2 t1 = fx::cadd(b, c), d = fx::csub(b, c);
            const float2 t2 = make_float2(a.x - 0.5f * t1.x, a.y - 0.5f * t1.y);
            const float2 t3 = make_float2(HS3 * d.x, HS3 * d.y);
            v[0][i] = fx::cadd(a, t1);
            v[1][i] = make_float2(t2.x - t3.y, t2.y + t3.x); // inverse: t2 + i t3
            v[2][i] = make_float2(t2.x + t3.y, t2.y - t3.x);
        }
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int i = 0; i < P; ++i) st_cg(p.field + tbase + (long long)(c * LP + tt + DOP_K0(i)) * es, v[c][i]);
    }
#undef DOP_K0
#undef DOP_KL
}

template <int LP, int V, int TWB, int NB>
static cudaError_t launch_x3_one(const PassDesc& p, cudaStream_t stream)
{
    constexpr int smem = fx::Tile<LP, true, NB>::LINE_ELEMS * (int)sizeof(float2);
    static AttrOnce once;
    cudaError_t e = once.ensure(p.device, [] {
        return cudaFuncSetAttribute(pow2x3_kernel<LP, V, TWB, NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    });
    if (e != cudaSuccess) return e;
    const long long ntiles = p.n_cgroups * p.n_m * p.n_o;
    if (ntiles <= 0 || ntiles > 2147483647LL) return cudaErrorInvalidConfiguration;
    pow2x3_kernel<LP, V, TWB, NB><<<(unsigned)ntiles, NB * (LP / P), smem, stream>>>(p);
    return cudaGetLastError();
}

template <int LP, int NB>
cudaError_t launch_x3_nb(const PassDesc& p, int variant, int twb, cudaStream_t st)
{
    if (twb == TWB_TILE) {
        if (variant == V_FWD) return launch_x3_one<LP, V_FWD, TWB_TILE, NB>(p, st);
        if (variant == V_INV) return launch_x3_one<LP, V_INV, TWB_TILE, NB>(p, st);
    } else if (twb == TWB_LANE) {
        if (variant == V_FWD) return launch_x3_one<LP, V_FWD, TWB_LANE, NB>(p, st);
        if (variant == V_INV) return launch_x3_one<LP, V_INV, TWB_LANE, NB>(p, st);
    }
    return kNotInstantiated;
}

template <int LP>
cudaError_t launch_x3(const PassDesc& p, int variant, int twb, cudaStream_t st)
{
    if (p.nl == 16) return launch_x3_nb<LP, 16>(p, variant, twb, st);
    if (p.nl == 32) return launch_x3_nb<LP, 32>(p, variant, twb, st);
    return kNotInstantiated;
}

// ---- host side -------------------------------------------------------------------------------
template <int L, bool COL, int V, int TWB, int NB = 16>
static cudaError_t launch_one(const PassDesc& p, cudaStream_t stream)
{
    using TL = fx::Tile<L, COL, NB>;
    constexpr int threads = tile_threads(L, COL, NB);
    constexpr int smem = (COL ? 1 : row_lines(L)) * TL::LINE_ELEMS * (int)sizeof(float2);
    static AttrOnce once; // per instantiation and device
    cudaError_t e = once.ensure(p.device, [] {
        cudaError_t a = cudaFuncSetAttribute(pow2_kernel<L, COL, V, TWB, NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (a != cudaSuccess) return a;
        return cudaFuncSetAttribute(pow2_kernel<L, COL, V, TWB, NB>, cudaFuncAttributePreferredSharedMemoryCarveout,
                                    cudaSharedmemCarveoutMaxShared);
    });
    if (e != cudaSuccess) return e;
    const long long ntiles = p.n_cgroups * p.n_m * p.n_o;
    if (ntiles <= 0 || ntiles > 2147483647LL) return cudaErrorInvalidConfiguration;
    pow2_kernel<L, COL, V, TWB, NB><<<(unsigned)ntiles, threads, smem, stream>>>(p);
    return cudaGetLastError();
}

// All variants of one (L, tile type).  Returns kNotInstantiated for a combination that is
// never scheduled (the dispatcher then falls back to the generic kernel).
// widest column bundle instantiated for a digit length: 64 columns up to L = 128, 32 up to 256
__host__ __device__ constexpr int max_col_nb(int L) { return L <= 128 ? 64 : (L <= 256 ? 32 : 16); }

template <int L, int NB>
cudaError_t launch_col(const PassDesc& p, int variant, int twb, cudaStream_t st)
{
    if constexpr (NB <= max_col_nb(L)) {
        if (twb == TWB_NONE) {
            if (variant == V_H) return launch_one<L, true, V_H, TWB_NONE, NB>(p, st);
            if (variant == V_GAUSS) return launch_one<L, true, V_GAUSS, TWB_NONE, NB>(p, st);
        } else if (twb == TWB_TILE) {
            if (variant == V_FWD) return launch_one<L, true, V_FWD, TWB_TILE, NB>(p, st);
            if (variant == V_INV) return launch_one<L, true, V_INV, TWB_TILE, NB>(p, st);
        } else {
            switch (variant) {
            case V_FWD: return launch_one<L, true, V_FWD, TWB_LANE, NB>(p, st);
            case V_INV: return launch_one<L, true, V_INV, TWB_LANE, NB>(p, st);
            case V_LOSS: return launch_one<L, true, V_LOSS, TWB_LANE, NB>(p, st);
            case V_HEIGHT: return launch_one<L, true, V_HEIGHT, TWB_LANE, NB>(p, st);
            case V_LDOTHER: return launch_one<L, true, V_LDOTHER, TWB_LANE, NB>(p, st);
            case V_GRAD: return launch_one<L, true, V_GRAD, TWB_LANE, NB>(p, st);
            case V_STOTHER: return launch_one<L, true, V_STOTHER, TWB_LANE, NB>(p, st);
            }
        }
    }
    return kNotInstantiated;
}

// All variants of one (L, tile type).  Returns kNotInstantiated for a combination that is
// never scheduled (the dispatcher then falls back to the generic kernel).
template <int L, bool COL>
cudaError_t launch_L(const PassDesc& p, int variant, int twb, cudaStream_t st)
{
    if constexpr (COL) {
        if (p.nl == 16) return launch_col<L, 16>(p, variant, twb, st);
        if (p.nl == 32) return launch_col<L, 32>(p, variant, twb, st);
        if (p.nl == 64) return launch_col<L, 64>(p, variant, twb, st);
    } else {
        if (twb == TWB_NONE) {
            switch (variant) {
            case V_FWD: return launch_one<L, false, V_FWD, TWB_NONE>(p, st);
            case V_INV: return launch_one<L, false, V_INV, TWB_NONE>(p, st);
            case V_LOSS: return launch_one<L, false, V_LOSS, TWB_NONE>(p, st);
            case V_HEIGHT: return launch_one<L, false, V_HEIGHT, TWB_NONE>(p, st);
            case V_LDOTHER: return launch_one<L, false, V_LDOTHER, TWB_NONE>(p, st);
            case V_GRAD: return launch_one<L, false, V_GRAD, TWB_NONE>(p, st);
            case V_STOTHER: return launch_one<L, false, V_STOTHER, TWB_NONE>(p, st);
            }
        }
    }
    return kNotInstantiated;
}

} // namespace dop
