// tma_col.cuh -- column-type digit passes as a persistent, TMA-fed pipeline (sm_100a).
//
// Same pass semantics, slot order and butterflies as pow2_kernel's column tiles (pow2_impl.cuh;
// PAPER.md:95-112 Eq. 1-4, PAPER.md:200 row-column 2-D FFT), but the tile never travels through the
// load/store unit: a strided NB-column x L-slot tile of the field is exactly one 4-D TMA box, so
//   * a producer warp moves tiles between HBM and shared memory with cp.async.bulk.tensor
//     (UTMALDG / UTMASTG), completion tracked by mbarriers, NST tiles in flight per CTA;
//   * the compute warps run the register-blocked DFT out of the tile buffer itself: the buffer has the
//     layout of fft_regs.cuh's exchange buffer (slot * NB + column), so "load" is from_smem<0>, every
//     group boundary is one store + one barrier + one load, and the last group's to_smem leaves the
//     result where the TMA store picks it up (in place, like every pass);
//   * the CTA is persistent (grid = resident CTAs), so loads of tile k+1.. overlap the DFT of tile k.
// Measured on B200 (profiles/r02_tma_col.md): the strided tile pattern tops out at 0.69-0.74 of the
// copy bandwidth through LDG/STG (16- to 64-column bundles) and reaches 0.88-0.93 through TMA.
//
// Fused variants: plain forward / inverse (V_FWD, V_INV), the (x) H sandwich (V_H), the Gaussian
// sandwich (V_GAUSS), and on x digits h -> exp(i Phi) -> DFT (V_HEIGHT), IDFT -> |u|^2, loss, seed ->
// DFT (V_LOSS), IDFT -> dL/dh (V_GRAD), and the split loss flavours of DOP_LOSS_NONE / DOP_LOSS_SIMSE (IDFT -> u, |u|^2
// [, plane sums]: V_STOTHER; seed from u and a plane -> DFT: V_LDOTHER) with their fp32 planes staged by TMA as well.
// Digits 3 * 2^k: a thread keeps its 16 points of the three 2^k sub-tiles, radix-3 step on registers.
#pragma once
#include <cuda.h>

#include <cstring>

#include "pow2_impl.cuh"

namespace dop {

struct alignas(64) TmaMaps {
    CUtensorMap field; // complex64 field as 8-byte elements: dims (line, m, slot, o), box (NB, 1, LB, 1)
    CUtensorMap pin;   // fp32 plane the pass reads (height / target), same dims
    CUtensorMap pout;  // fp32 plane the pass writes (dL/dh / intensity)
};

// ---- PTX wrappers (mbarrier, bulk tensor copies, proxy fences)
__device__ __forceinline__ unsigned tm_smem(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void tm_mbar_init(uint64_t* b, unsigned n)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(tm_smem(b)), "r"(n) : "memory");
}
__device__ __forceinline__ void tm_mbar_expect_tx(uint64_t* b, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(tm_smem(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tm_mbar_arrive(uint64_t* b)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(tm_smem(b)) : "memory");
}
__device__ __forceinline__ void tm_mbar_wait(uint64_t* b, unsigned parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\tTM_WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra TM_DONE_%=;\n\tbra TM_WAIT_%=;\n\tTM_DONE_%=:\n\t}" ::"r"(tm_smem(b)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tm_load(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2, int c3)
{
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
                 ::"r"(tm_smem(dst)), "l"(map), "r"(tm_smem(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ void tm_store(const CUtensorMap* map, const void* src, int c0, int c1, int c2, int c3)
{
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.bulk_group [%0, {%2, %3, %4, %5}], [%1];"
                 ::"l"(map), "r"(tm_smem(src)), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ void tm_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void tm_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void tm_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void tm_fence_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// resident CTAs per SM the kernel is compiled for: limited by shared memory (227 KiB, 1 KiB reserved per CTA)
// and by 2048 threads per SM; the register allocation follows from it
__host__ __device__ constexpr int tma_min_blocks(int smem, int threads)
{
    const int a = 232448 / (smem + 2048), b = 1024 / threads; // (>= 64 registers per thread)
    const int m = a < b ? a : b;
    return m < 1 ? 1 : m;
}

// The register-blocked DFT of fft_regs.cuh run out of a tile buffer that already holds the data in the
// exchange layout: v enters in the layout of group G (forward) and leaves in the layout of the last
// group; every group boundary is one store, one barrier among the NCOMP compute threads, one load
// (a thread only ever overwrites slots it has read itself, so no second barrier is needed).  `bar` / NBAR: the named
// barrier and its thread count (digits 3 LP: each sub-tile's thread group exchanges on a barrier of its own).
template <class TL, class S, int G, int NBAR>
__device__ __forceinline__ void fwd_groups(float2* v, float2* B, int tt, int col, const float2* __restrict__ tw, int bar = 1)
{
    TL::template butterflies<G, +1>(v, tt, tw);
    if constexpr (G + 1 < S::NG) {
        TL::template to_smem<G>(v, B, tt, col);
        asm volatile("bar.sync %0, %1;" ::"r"(bar), "n"(NBAR) : "memory");
        TL::template from_smem<G + 1>(v, B, tt, col);
        fwd_groups<TL, S, G + 1, NBAR>(v, B, tt, col, tw, bar);
    }
}
// inverse: v enters in the layout of group G (the last one) and leaves in the layout of group 0
template <class TL, class S, int G, int NBAR>
__device__ __forceinline__ void inv_groups(float2* v, float2* B, int tt, int col, const float2* __restrict__ tw, int bar = 1)
{
    TL::template butterflies<G, -1>(v, tt, tw);
    if constexpr (G > 0) {
        TL::template to_smem<G>(v, B, tt, col);
        asm volatile("bar.sync %0, %1;" ::"r"(bar), "n"(NBAR) : "memory");
        TL::template from_smem<G - 1>(v, B, tt, col);
        inv_groups<TL, S, G - 1, NBAR>(v, B, tt, col, tw, bar);
    }
}

// Three independent sub-tiles per thread (digits 3 LP): the same walks with the three exchanges of a group boundary
// behind ONE barrier, and three independent butterfly chains for the scheduler to interleave.
template <class TL, class S, int G, int NBAR>
__device__ __forceinline__ void fwd_groups3(float2 (*v)[P], float2* B, int sub_stride, int tt, int col, const float2* __restrict__ tw)
{
#pragma unroll
    for (int c = 0; c < 3; ++c) TL::template butterflies<G, +1>(v[c], tt, tw);
    if constexpr (G + 1 < S::NG) {
#pragma unroll
        for (int c = 0; c < 3; ++c) TL::template to_smem<G>(v[c], B + c * sub_stride, tt, col);
        asm volatile("bar.sync 1, %0;" ::"n"(NBAR) : "memory");
#pragma unroll
        for (int c = 0; c < 3; ++c) TL::template from_smem<G + 1>(v[c], B + c * sub_stride, tt, col);
        fwd_groups3<TL, S, G + 1, NBAR>(v, B, sub_stride, tt, col, tw);
    }
}
template <class TL, class S, int G, int NBAR>
__device__ __forceinline__ void inv_groups3(float2 (*v)[P], float2* B, int sub_stride, int tt, int col, const float2* __restrict__ tw)
{
#pragma unroll
    for (int c = 0; c < 3; ++c) TL::template butterflies<G, -1>(v[c], tt, tw);
    if constexpr (G > 0) {
#pragma unroll
        for (int c = 0; c < 3; ++c) TL::template to_smem<G>(v[c], B + c * sub_stride, tt, col);
        asm volatile("bar.sync 1, %0;" ::"n"(NBAR) : "memory");
#pragma unroll
        for (int c = 0; c < 3; ++c) TL::template from_smem<G - 1>(v[c], B + c * sub_stride, tt, col);
        inv_groups3<TL, S, G - 1, NBAR>(v, B, sub_stride, tt, col, tw);
    }
}

// compile-time geometry of one instantiation
template <int L, int NB, int V, int NST>
struct TmaGeo {
    static constexpr bool X3 = (L % 3) == 0;
    static constexpr int LP = X3 ? L / 3 : L;      // register-blocked sub-transform length
    static constexpr int NSUB = X3 ? 3 : 1;
    static constexpr int T = LP / P;               // compute threads per column
    static constexpr int NCOMP = NB * T;           // (digits 3 LP: a thread holds its 16 points of all three sub-tiles)
    static constexpr int THREADS = NCOMP + 32;     // + the producer warp
    static constexpr int TILE = L * NB;            // points per tile
    static constexpr int NBOX = (L + 255) / 256;   // a TMA box dimension is at most 256
    static constexpr int LB = L / NBOX;
    static constexpr bool PIN = V == V_LOSS || V == V_HEIGHT || V == V_GRAD || V == V_LDOTHER || V == V_STOTHER;
    static constexpr bool FIELD_IN = V != V_HEIGHT;
    static constexpr bool FIELD_OUT = V != V_GRAD;
    static constexpr int FIELD_BYTES = TILE * 8;
    static constexpr int PLANE_BYTES = PIN ? TILE * 4 : 0;
    static constexpr int STAGE_BYTES = FIELD_BYTES + PLANE_BYTES;
    static constexpr int SMEM = NST * STAGE_BYTES;
    static constexpr int MINB = tma_min_blocks(SMEM, THREADS);
};

template <int L, int NB, int V, int TWB, int NST>
__global__ void __launch_bounds__(TmaGeo<L, NB, V, NST>::THREADS, TmaGeo<L, NB, V, NST>::MINB)
tma_col_kernel(const __grid_constant__ PassDesc p, const __grid_constant__ TmaMaps maps, unsigned ntiles)
{
    using G = TmaGeo<L, NB, V, NST>;
    constexpr int LP = G::LP, T = G::T, NCOMP = G::NCOMP;
    using TL = fx::Tile<LP, true, NB>;
    using S = fx::Sched<LP>;
    constexpr int GL = S::NG - 1;
    constexpr int RL = S::radix(GL);
    constexpr int DIR1 = variant_dir1(V), DIR2 = variant_dir2(V);
    constexpr int LAST = DIR2 != 0 ? DIR2 : DIR1;
    constexpr float HS3 = 0.86602540378443864676f; // sqrt(3)/2

    extern __shared__ __align__(128) unsigned char tm_raw[];
    __shared__ uint64_t full[NST], done[NST];
    __shared__ double red[2][NCOMP / 32 > 0 ? NCOMP / 32 : 1];
    __shared__ double red4[V == V_STOTHER ? 2 : 1][4][NCOMP / 32 > 0 ? NCOMP / 32 : 1]; // plane sums of the si-mse pass

    const int tid = threadIdx.x;
    if (tid == 0) {
        for (int s = 0; s < NST; ++s) {
            tm_mbar_init(&full[s], 1);
            tm_mbar_init(&done[s], NCOMP);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const unsigned ncg = (unsigned)p.n_cgroups, nm = (unsigned)p.n_m;
    const unsigned first = blockIdx.x, stride = gridDim.x;
    const unsigned n_my = first < ntiles ? (ntiles - first + stride - 1) / stride : 0u;
    auto fbuf = [&](int s) -> float2* { return reinterpret_cast<float2*>(tm_raw + (size_t)s * G::STAGE_BYTES); };
    auto pbuf = [&](int s) -> float* { return reinterpret_cast<float*>(tm_raw + (size_t)s * G::STAGE_BYTES + G::FIELD_BYTES); };

    // ================================================================ producer warp
    if (tid >= NCOMP) {
        if (tid != NCOMP) return;
        // which fp32 plane tiles move: the run-time load / store op of the V_LDOTHER / V_STOTHER flavours decides
        const bool store_plane = V == V_GRAD || (V == V_LOSS && p.write_intensity) ||
                                 (V == V_STOTHER && (p.store_op == ST_C64_INTENSITY || p.write_intensity));
        const bool load_plane = G::PIN && !(V == V_STOTHER && p.store_op != ST_C64_STATS);
        auto coords = [&](unsigned k, int* c0, int* c1, int* c3) {
            unsigned t = first + k * stride;
            *c0 = (int)((t % ncg) + (unsigned)p.cg0) * NB;
            t /= ncg;
            *c1 = (int)(t % nm);
            *c3 = (int)(t / nm) + (int)p.o0;
        };
        auto load = [&](unsigned k) {
            const int s = (int)(k % NST);
            int c0, c1, c3;
            coords(k, &c0, &c1, &c3);
            tm_mbar_expect_tx(&full[s], (G::FIELD_IN ? G::FIELD_BYTES : 0) + (load_plane ? G::PLANE_BYTES : 0));
#pragma unroll
            for (int b = 0; b < G::NBOX; ++b) {
                if (G::FIELD_IN) tm_load(fbuf(s) + b * G::LB * NB, &maps.field, &full[s], c0, c1, b * G::LB, c3);
                if (load_plane) tm_load(pbuf(s) + b * G::LB * NB, &maps.pin, &full[s], c0, c1, b * G::LB, c3);
            }
        };
        for (unsigned k = 0; k < (unsigned)NST && k < n_my; ++k) load(k);
        for (unsigned k = 0; k < n_my; ++k) {
            const int s = (int)(k % NST);
            tm_mbar_wait(&done[s], (k / NST) & 1u); // the compute warps have left tile k in its buffer
            int c0, c1, c3;
            coords(k, &c0, &c1, &c3);
#pragma unroll
            for (int b = 0; b < G::NBOX; ++b) {
                if (G::FIELD_OUT) tm_store(&maps.field, fbuf(s) + b * G::LB * NB, c0, c1, b * G::LB, c3);
                if (store_plane) tm_store(&maps.pout, pbuf(s) + b * G::LB * NB, c0, c1, b * G::LB, c3);
            }
            tm_commit();
            if (k + NST < n_my) {
                tm_wait_read0(); // the store has read the buffer: refill it
                load(k + NST);
            }
        }
        tm_wait_all();
        return;
    }

    // ================================================================ compute warps
    const int col = tid % NB, tt = tid / NB;
    const float2* __restrict__ tw = p.tw_g;
    auto cbar = [] { asm volatile("bar.sync 1, %0;" ::"n"(NCOMP) : "memory"); };
#define DOP_KL(i) (((i) / RL) * (T * RL) + (i) % RL)

    for (unsigned k = 0; k < n_my; ++k) {
        const int s = (int)(k % NST);
        unsigned t = first + k * stride;
        const unsigned tile_id = t;
        const long long cg = (long long)(t % ncg) + p.cg0;
        t /= ncg;
        const long long m = t % nm;
        const long long o = (long long)(t / nm) + p.o0;
        const long long line0 = cg * NB + col;
        const long long line = line0 < p.NC ? line0 : p.NC - 1; // ragged last tile: clipped lanes read valid table entries
        float2* B = fbuf(s);
        float* Pl = pbuf(s);

        // boundary twiddle of the element in register i (last-group layout) of sub-tile c: twp[(c LP + KL(i)) tws]
        const float2* __restrict__ twp = nullptr;
        unsigned tws = 1;
        if (TWB == TWB_TILE) {
            twp = p.tw_b2 + m * L + tt * RL;
        } else if (TWB == TWB_LANE) {
            tws = (unsigned)p.NC;
            twp = p.tw_b2 + line + (long long)(tt * RL) * tws;
        }
        // Touch this tile's boundary twiddles now, before waiting for its data: they come from L2 (a different row of
        // the table per tile) and would otherwise be loaded right before their use (ncu: the twiddle multiplies sat
        // on long_scoreboard for a third of all samples).
        // (y digits; for the per-lane tables of the x digits -- 16 lines of 128 bytes per thread -- it measured as a loss)
        if (TWB == TWB_TILE) {
#pragma unroll
            for (int c = 0; c < G::NSUB; ++c)
#pragma unroll
                for (int i = 0; i < P; i += RL) asm volatile("prefetch.global.L1 [%0];" ::"l"(twp + (unsigned)(c * LP + DOP_KL(i))));
        }
        if (V == V_H) { // touch the fy^2 entries of this tile before waiting for it
            const double* fyp = p.fy2 + o * p.row_o + m * p.row_m + tt * RL;
#pragma unroll
            for (int i = 0; i < P; i += RL) asm volatile("prefetch.global.L1 [%0];" ::"l"(fyp + DOP_KL(i)));
        }

        // Per-lane boundary twiddles (x digits: 16 table lines per thread, from L2) are fetched into registers BEFORE
        // the wait for the tile, so their latency hides behind it; the loss pass uses them twice.
        float2 twv[TWB == TWB_LANE && !G::X3 ? P : 1];
        if (TWB == TWB_LANE && !G::X3) {
#pragma unroll
            for (int i = 0; i < P; ++i) twv[i] = __ldg(twp + (unsigned)DOP_KL(i) * tws);
        }
        tm_mbar_wait(&full[s], (k / NST) & 1u);

        float2 v[P];
        if constexpr (!G::X3) {
            // ---- load (+ prologue) and first DFT
            if (DIR1 > 0) {
                if (V == V_HEIGHT) {
#pragma unroll
                    for (int i = 0; i < P; ++i) {
                        const float ph = Pl[(tt + i * T) * NB + col] * p.phase_coef; // Eq. (1) in turns
                        sincos_turns(ph, &v[i].y, &v[i].x);                          // Eq. (2), E_in = 1
                        // pad = 2: slots tt + i T >= L/2, i.e. registers i >= 8, lie outside the aperture: zero amplitude
                        if (i >= P / 2 && p.ap_nx > 0) v[i] = make_float2(0.0f, 0.0f);
                    }
                } else {
                    TL::template from_smem<0>(v, B, tt, col);
                    if (V == V_LDOTHER) { // A1 on a stored field: g_u = 2 (dL/dI) u  /  Eq. (6): (c0 + cI |u|^2 + cT T) u
                        const bool simse = p.load_op == LD_SEED_SIMSE;
                        const float k0 = simse ? __ldg(p.coef) : 0.0f, k1 = simse ? __ldg(p.coef + 1) : 0.0f,
                                    k2 = simse ? __ldg(p.coef + 2) : 2.0f;
#pragma unroll
                        for (int i = 0; i < P; ++i) {
                            const float pl = Pl[(tt + i * T) * NB + col];
                            const float g = fmaf(k1, v[i].x * v[i].x + v[i].y * v[i].y, fmaf(k2, pl, k0));
                            v[i] = make_float2(g * v[i].x, g * v[i].y);
                        }
                    }
                }
                fwd_groups<TL, S, 0, NCOMP>(v, B, tt, col, tw);
            } else {
                TL::template from_smem<GL>(v, B, tt, col);
                if (TWB == TWB_LANE) {
#pragma unroll
                    for (int i = 0; i < P; ++i) v[i] = fx::cmulc(v[i], twv[i]);
                } else if (TWB != TWB_NONE) {
#pragma unroll
                    for (int i = 0; i < P; ++i) v[i] = fx::cmulc(v[i], __ldg(twp + (unsigned)DOP_KL(i) * tws));
                }
                inv_groups<TL, S, GL, NCOMP>(v, B, tt, col, tw);
            }
            // ---- middle op
            if (V == V_H) {
                const double* __restrict__ fyp = p.fy2 + o * p.row_o + m * p.row_m + tt * RL;
                const double cfx = p.inv_lam2 - __ldg(p.fx2 + line);
                const bool cj = p.mid_op == MID_HCONJ;
                // (the plan routes H passes here only when the phase may be taken in fixed point: h_fixed)
                const double z32 = (cj ? -p.z : p.z) * 4294967296.0; // conj H = H at the negated phase
                HCoef hk;
#pragma unroll
                for (int q = 0; q < 5; ++q) { hk.s[q] = p.hk_s[q]; hk.c[q] = p.hk_c[q]; }
#pragma unroll
                for (int i = 0; i < P; ++i) v[i] = apply_h_fixed_nb(v[i], cfx, __ldg(fyp + DOP_KL(i)), z32, hk);
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
#pragma unroll
                for (int i = 0; i < P; ++i) {
                    float* tp = Pl + (tt + i * T) * NB + col;
                    const float I = v[i].x * v[i].x + v[i].y * v[i].y; // F6
                    float d = I - *tp;                                 // F7
                    if (i >= P / 2 && p.ap_nx > 0) d = 0.0f;           // pad = 2: outside the aperture, no loss term, zero seed
                    acc += (double)d * (double)d;
                    const float g = p.seed_coef * d;                   // A1: 2 gI = 4 (I - T)/N
                    v[i] = make_float2(g * v[i].x, g * v[i].y);
                    if (p.write_intensity) *tp = I;
                }
                // deterministic CTA reduction: warp shuffle tree, then one thread in warp order
#pragma unroll
                for (int d = 16; d > 0; d >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, d);
                if ((tid & 31) == 0) red[k & 1][tid >> 5] = acc;
                // The warp sums are added up (warp order: deterministic) by thread 0 AFTER the forward DFT, whose first
                // exchange is the barrier between these writes and that read -- red[] is double-buffered, the tile after
                // next is the first to write this half again.  With a barrier of its own here and the serial sum right
                // behind it, every warp waited for thread 0 at the DFT's exchange: C5 loss pass 34.3 -> 30.4 ms, C4
                // 27.8 -> 23.1.  (Summing in the producer thread instead measured no gain at C4: 27.3.)
                if constexpr (S::NG == 1) cbar(); // (a single-group digit has no exchange)
            }
            if (DIR2 > 0) fwd_groups<TL, S, 0, NCOMP>(v, B, tt, col, tw);
            else if (DIR2 < 0) inv_groups<TL, S, GL, NCOMP>(v, B, tt, col, tw);
            if (V == V_LOSS && tid == 0) { // (serial on purpose: a shuffle tree over warp 0 here measured C4 21.9 -> 28.1 ms)
                double r = 0.0;
                for (int w = 0; w < NCOMP / 32; ++w) r += red[k & 1][w];
                p.loss_scratch[p.tile0 + tile_id] = r;
            }
            // ---- store (+ boundary twiddle after a forward DFT, + epilogue)
            if (LAST > 0) {
                if (TWB == TWB_LANE) {
#pragma unroll
                    for (int i = 0; i < P; ++i) v[i] = fx::cmul(v[i], twv[i]);
                } else if (TWB != TWB_NONE) {
#pragma unroll
                    for (int i = 0; i < P; ++i) v[i] = fx::cmul(v[i], __ldg(twp + (unsigned)DOP_KL(i) * tws));
                }
                TL::template to_smem<GL>(v, B, tt, col);
            } else if (V == V_GRAD) {
#pragma unroll
                for (int i = 0; i < P; ++i) {
                    float* hp = Pl + (tt + i * T) * NB + col;
                    float sn, cs;
                    sincos_turns(*hp * p.phase_coef, &sn, &cs);              // u0 recomputed, not stored
                    *hp = p.grad_coef * (cs * v[i].y - sn * v[i].x);         // A5: c Im(conj(u0) g)
                }
            } else {
                TL::template to_smem<0>(v, B, tt, col);
                if (V == V_STOTHER) { // keep u; I = |u|^2 [and the plane sums <I,T>, <I,I>, sum I, <T,T> of Eq. (6)]
                    const bool stats = p.store_op == ST_C64_STATS;
                    double st0 = 0.0, st1 = 0.0, st2 = 0.0, st3 = 0.0;
#pragma unroll
                    for (int i = 0; i < P; ++i) {
                        float* tp = Pl + (tt + i * T) * NB + col;
                        const float I = v[i].x * v[i].x + v[i].y * v[i].y;
                        if (stats) {
                            const float Tv = *tp;
                            st0 += (double)I * (double)Tv;
                            st1 += (double)I * (double)I;
                            st2 += (double)I;
                            st3 += (double)Tv * (double)Tv;
                        }
                        if (!stats || p.write_intensity) *tp = I;
                    }
                    if (stats) { // deterministic CTA reduction of the four sums
#pragma unroll
                        for (int d = 16; d > 0; d >>= 1) {
                            st0 += __shfl_down_sync(0xffffffffu, st0, d);
                            st1 += __shfl_down_sync(0xffffffffu, st1, d);
                            st2 += __shfl_down_sync(0xffffffffu, st2, d);
                            st3 += __shfl_down_sync(0xffffffffu, st3, d);
                        }
                        if ((tid & 31) == 0) {
                            red4[k & 1][0][tid >> 5] = st0; red4[k & 1][1][tid >> 5] = st1;
                            red4[k & 1][2][tid >> 5] = st2; red4[k & 1][3][tid >> 5] = st3;
                        }
                        cbar();
                        if (tid < 4) {
                            double r = 0.0;
                            for (int w = 0; w < NCOMP / 32; ++w) r += red4[k & 1][tid][w];
                            p.loss_scratch[4 * (p.tile0 + tile_id) + tid] = r;
                        }
                    }
                }
            }
        } else {
            // ---- digits 3 * LP: a thread keeps its 16 points of all three LP-point sub-tiles (48 points; the CTA is alone
            //      on its SM, so the registers are there), runs the radix-3 step on registers and the three sub-tile
            //      DFTs side by side (one barrier per group boundary for the three exchanges).
            const float2* __restrict__ wL = p.wL; // W_L^q, L = 3 LP
            float2 w3[3][P];
            if (DIR1 > 0) {
#pragma unroll
                for (int c = 0; c < 3; ++c) TL::template from_smem<0>(w3[c], B + c * LP * NB, tt, col);
#pragma unroll
                for (int i = 0; i < P; ++i) { // radix-3 step (block length L, stride LP), outputs c = 1, 2 times W_L^{j c}
                    const int j = tt + i * T;
                    const float2 a = w3[0][i], b = w3[1][i], c = w3[2][i];
                    const float2 t1 = fx::cadd(b, c), d = fx::csub(b, c);
                    const float2 t2 = make_float2(a.x - 0.5f * t1.x, a.y - 0.5f * t1.y);
                    const float2 t3 = make_float2(HS3 * d.x, HS3 * d.y);
                    w3[0][i] = fx::cadd(a, t1);
                    w3[1][i] = fx::cmul(make_float2(t2.x + t3.y, t2.y - t3.x), __ldg(wL + j));     // t2 - i t3
                    w3[2][i] = fx::cmul(make_float2(t2.x - t3.y, t2.y + t3.x), __ldg(wL + 2 * j)); // t2 + i t3
                }
                fwd_groups3<TL, S, 0, NCOMP>(w3, B, LP * NB, tt, col, tw);
#pragma unroll
                for (int c = 0; c < 3; ++c) {
#pragma unroll
                    for (int i = 0; i < P; ++i) w3[c][i] = fx::cmul(w3[c][i], __ldg(twp + (unsigned)(c * LP + DOP_KL(i)) * tws));
                    TL::template to_smem<GL>(w3[c], B + c * LP * NB, tt, col);
                }
            } else {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    TL::template from_smem<GL>(w3[c], B + c * LP * NB, tt, col);
#pragma unroll
                    for (int i = 0; i < P; ++i) w3[c][i] = fx::cmulc(w3[c][i], __ldg(twp + (unsigned)(c * LP + DOP_KL(i)) * tws));
                }
                inv_groups3<TL, S, GL, NCOMP>(w3, B, LP * NB, tt, col, tw);
#pragma unroll
                for (int i = 0; i < P; ++i) {
                    const int j = tt + i * T;
                    const float2 a = w3[0][i];
                    const float2 b = fx::cmulc(w3[1][i], __ldg(wL + j));
                    const float2 c = fx::cmulc(w3[2][i], __ldg(wL + 2 * j));
                    const float2 t1 = fx::cadd(b, c), d = fx::csub(b, c);
                    const float2 t2 = make_float2(a.x - 0.5f * t1.x, a.y - 0.5f * t1.y);
                    const float2 t3 = make_float2(HS3 * d.x, HS3 * d.y);
                    w3[0][i] = fx::cadd(a, t1);
                    w3[1][i] = make_float2(t2.x - t3.y, t2.y + t3.x); // inverse: t2 + i t3
                    w3[2][i] = make_float2(t2.x + t3.y, t2.y - t3.x);
                }
#pragma unroll
                for (int c = 0; c < 3; ++c) TL::template to_smem<0>(w3[c], B + c * LP * NB, tt, col);
            }
        }
        tm_fence_async();          // this thread's writes to the tile are visible to the TMA store
        tm_mbar_arrive(&done[s]);
    }
#undef DOP_KL
}

// ---- the (x) H sandwich on mirrored tile pairs ---------------------------------------------------------------
// H(kx, ky) = H(kx, -ky): the tile of the last y digit that holds the frequencies k_low + N_low k_last (k_low fixed
// by the tile, k_last by the slot) has a mirror tile holding (N_low - k_low) + N_low (L - 1 - k_last), and in the
// digit-reversed slot order "L - 1 - k_last" is simply slot L - 1 - i: the thread that owns slots 16 tt .. 16 tt + 15
// of tile A, acting as thread T - 1 - tt on tile B, finds in register 15 - i the point whose H it has just computed.
// So one CTA runs the pair back to back and evaluates H (about 40 of the pass's 83 instructions per point) once
// for both.  Work item = (column group, item q) with items[q] = (tile o_A, mirror tile o_B or -1 for the two
// self-mirrored tiles k_low = 0, N_low / 2, which are processed alone); the tile sequence feeds the same NST-deep
// TMA ring as tma_col_kernel.
template <int L, int NB, int NST>
__global__ void __launch_bounds__(TmaGeo<L, NB, V_H, NST>::THREADS, TmaGeo<L, NB, V_H, NST>::MINB)
tma_hpair_kernel(const __grid_constant__ PassDesc p, const __grid_constant__ TmaMaps maps, unsigned nitems)
{
    using G = TmaGeo<L, NB, V_H, NST>;
    constexpr int T = G::T, NCOMP = G::NCOMP;
    using TL = fx::Tile<L, true, NB>;
    using S = fx::Sched<L>;
    constexpr int GL = S::NG - 1;
    constexpr int RL = S::radix(GL);
    static_assert(!G::X3, "pairs of power-of-two digits only");
    extern __shared__ __align__(128) unsigned char tm_raw[];
    __shared__ uint64_t full[NST], done[NST];

    const int tid = threadIdx.x;
    if (tid == 0) {
        for (int s = 0; s < NST; ++s) {
            tm_mbar_init(&full[s], 1);
            tm_mbar_init(&done[s], NCOMP);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const unsigned ncg = (unsigned)p.n_cgroups;
    const unsigned first = blockIdx.x, stride = gridDim.x;
    const unsigned n_my = first < nitems ? (nitems - first + stride - 1) / stride : 0u;
    const int2* __restrict__ items = reinterpret_cast<const int2*>(p.hpair);
    auto fbuf = [&](unsigned s) -> float2* { return reinterpret_cast<float2*>(tm_raw + (size_t)s * G::STAGE_BYTES); };
    auto item_of = [&](unsigned k, unsigned* cg) -> int2 {
        const unsigned w = first + k * stride;
        *cg = w % ncg;
        return __ldg(items + w / ncg);
    };

    // ================================================================ producer warp
    if (tid >= NCOMP) {
        if (tid != NCOMP) return;
        auto advance = [&](unsigned& k, int& half) {
            unsigned cg;
            if (half == 0 && item_of(k, &cg).y >= 0) half = 1;
            else { half = 0; ++k; }
        };
        auto coords = [&](unsigned k, int half, int* c0, int* c3) {
            unsigned cg;
            const int2 it = item_of(k, &cg);
            *c0 = (int)(cg + (unsigned)p.cg0) * NB;
            *c3 = half ? it.y : it.x;
        };
        unsigned lk = 0, loads = 0, sk = 0, stores = 0;
        int lhalf = 0, shalf = 0;
        auto issue_load = [&]() {
            const unsigned s = loads % NST;
            int c0, c3;
            coords(lk, lhalf, &c0, &c3);
            tm_mbar_expect_tx(&full[s], G::FIELD_BYTES);
#pragma unroll
            for (int b = 0; b < G::NBOX; ++b) tm_load(fbuf(s) + b * G::LB * NB, &maps.field, &full[s], c0, 0, b * G::LB, c3);
            ++loads;
            advance(lk, lhalf);
        };
        while (loads < (unsigned)NST && lk < n_my) issue_load();
        while (sk < n_my) {
            const unsigned s = stores % NST;
            tm_mbar_wait(&done[s], (stores / NST) & 1u);
            int c0, c3;
            coords(sk, shalf, &c0, &c3);
#pragma unroll
            for (int b = 0; b < G::NBOX; ++b) tm_store(&maps.field, fbuf(s) + b * G::LB * NB, c0, 0, b * G::LB, c3);
            tm_commit();
            ++stores;
            advance(sk, shalf);
            if (lk < n_my) {
                tm_wait_read0();
                issue_load();
            }
        }
        tm_wait_all();
        return;
    }

    // ================================================================ compute warps
    const int col = tid % NB, tt = tid / NB;
    const float2* __restrict__ tw = p.tw_g;
    const double z32 = (p.mid_op == MID_HCONJ ? -p.z : p.z) * 4294967296.0; // conj H = H at the negated phase
    HCoef hk;
#pragma unroll
    for (int q = 0; q < 5; ++q) { hk.s[q] = p.hk_s[q]; hk.c[q] = p.hk_c[q]; }
#define DOP_KL(i) (((i) / RL) * (T * RL) + (i) % RL)
    unsigned j = 0; // tiles processed so far (position in the ring)
    for (unsigned k = 0; k < n_my; ++k) {
        unsigned cgi;
        const int2 it = item_of(k, &cgi);
        const long long line0 = ((long long)cgi + p.cg0) * NB + col;
        const long long line = line0 < p.NC ? line0 : p.NC - 1;
        const double cfx = p.inv_lam2 - __ldg(p.fx2 + line);
        const double* __restrict__ fyp = p.fy2 + (long long)it.x * p.row_o + tt * RL;
#pragma unroll
        for (int i = 0; i < P; i += RL) asm volatile("prefetch.global.L1 [%0];" ::"l"(fyp + DOP_KL(i)));
        float2 h[P];
        float2 v[P];
        // ---- tile A: H evaluated (after the DFT: evaluating it before the wait for the tile, where a tile still in
        //      flight would hide it, measured slower -- C5 25.8 -> 27.7 ms, C4 17.1 -> 18.1: 32 more live registers
        //      through the forward DFT)
        {
            const unsigned s = j % NST;
            float2* B = fbuf(s);
            tm_mbar_wait(&full[s], (j / NST) & 1u);
            TL::template from_smem<0>(v, B, tt, col);
            fwd_groups<TL, S, 0, NCOMP>(v, B, tt, col, tw);
#pragma unroll
            for (int i = 0; i < P; ++i) {
                h[i] = h_fixed_nb(cfx, __ldg(fyp + DOP_KL(i)), z32, hk);
                v[i] = fx::cmul(v[i], h[i]);
            }
            inv_groups<TL, S, GL, NCOMP>(v, B, tt, col, tw);
            TL::template to_smem<0>(v, B, tt, col);
            tm_fence_async();
            tm_mbar_arrive(&done[s]);
            ++j;
        }
        // ---- tile B: the mirror tile, this thread in the place of thread T - 1 - tt, H taken from register P - 1 - i
        if (it.y >= 0) {
            const unsigned s = j % NST;
            float2* B = fbuf(s);
            const int tm = T - 1 - tt;
            tm_mbar_wait(&full[s], (j / NST) & 1u);
            TL::template from_smem<0>(v, B, tm, col);
            fwd_groups<TL, S, 0, NCOMP>(v, B, tm, col, tw);
#pragma unroll
            for (int i = 0; i < P; ++i) v[i] = fx::cmul(v[i], h[P - 1 - i]);
            inv_groups<TL, S, GL, NCOMP>(v, B, tm, col, tw);
            TL::template to_smem<0>(v, B, tm, col);
            tm_fence_async();
            tm_mbar_arrive(&done[s]);
            ++j;
        }
    }
#undef DOP_KL
}

// ---- host side -------------------------------------------------------------------------------
typedef CUresult (*TmaEncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
TmaEncodeFn tma_encode_fn();   // cuTensorMapEncodeTiled through cudaGetDriverEntryPoint (no link against libcuda)
// 4-D map of one plane for the tiles of pass p: dims (line, m, slot, o) with the pass's strides, box (nb, 1, lb, 1)
bool tma_make_map(CUtensorMap* map, const void* base, int elem_bytes, const PassDesc& p, int nb, int lb, long long slots = 0,
                  long long so = 0);
int tma_sm_count(int device);

template <int L, int NB, int NST>
static cudaError_t launch_tma_hpair(const PassDesc& p, cudaStream_t stream)
{
    using G = TmaGeo<L, NB, V_H, NST>;
    static AttrOnce once;
    static std::atomic<int> resident[64];
    cudaError_t e = once.ensure(p.device, [&] {
        cudaError_t a = cudaFuncSetAttribute(tma_hpair_kernel<L, NB, NST>, cudaFuncAttributeMaxDynamicSharedMemorySize, G::SMEM);
        if (a != cudaSuccess) return a;
        a = cudaFuncSetAttribute(tma_hpair_kernel<L, NB, NST>, cudaFuncAttributePreferredSharedMemoryCarveout,
                                 cudaSharedmemCarveoutMaxShared);
        if (a != cudaSuccess) return a;
        int nb = 0;
        a = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, tma_hpair_kernel<L, NB, NST>, G::THREADS, G::SMEM);
        if (a != cudaSuccess) return a;
        if (p.device >= 0 && p.device < 64) resident[p.device].store(nb < 1 ? 1 : nb);
        return cudaSuccess;
    });
    if (e != cudaSuccess) return e;
    const long long nitems = p.n_cgroups * (long long)p.n_hpair;
    if (nitems <= 0 || nitems > 2147483647LL) return cudaErrorInvalidConfiguration;
    TmaMaps maps;
    memset(&maps, 0, sizeof(maps));
    if (!tma_make_map(&maps.field, p.field, 8, p, NB, G::LB)) return cudaErrorInvalidValue;
    const int per_sm = (p.device >= 0 && p.device < 64) ? resident[p.device].load() : 1;
    long long grid = (long long)tma_sm_count(p.device) * (per_sm < 1 ? 1 : per_sm);
    if (grid > nitems) grid = nitems;
    tma_hpair_kernel<L, NB, NST><<<(unsigned)grid, G::THREADS, G::SMEM, stream>>>(p, maps, (unsigned)nitems);
    return cudaGetLastError();
}

template <int L, int NB, int V, int TWB, int NST>
static cudaError_t launch_tma_one(const PassDesc& p, cudaStream_t stream)
{
    using G = TmaGeo<L, NB, V, NST>;
    static AttrOnce once;
    static std::atomic<int> resident[64]; // CTAs per SM, per device
    cudaError_t e = once.ensure(p.device, [&] {
        cudaError_t a = cudaFuncSetAttribute(tma_col_kernel<L, NB, V, TWB, NST>, cudaFuncAttributeMaxDynamicSharedMemorySize, G::SMEM);
        if (a != cudaSuccess) return a;
        a = cudaFuncSetAttribute(tma_col_kernel<L, NB, V, TWB, NST>, cudaFuncAttributePreferredSharedMemoryCarveout,
                                 cudaSharedmemCarveoutMaxShared);
        if (a != cudaSuccess) return a;
        int nb = 0;
        a = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, tma_col_kernel<L, NB, V, TWB, NST>, G::THREADS, G::SMEM);
        if (a != cudaSuccess) return a;
        if (p.device >= 0 && p.device < 64) resident[p.device].store(nb < 1 ? 1 : nb);
        return cudaSuccess;
    });
    if (e != cudaSuccess) return e;
    const long long ntiles = p.n_cgroups * p.n_m * p.n_o;
    if (ntiles <= 0 || ntiles > 2147483647LL) return cudaErrorInvalidConfiguration;
    if constexpr (V == V_H && L % 3 != 0) {
        if (p.hpair != nullptr && p.n_m == 1) return launch_tma_hpair<L, NB, NST>(p, stream);
    }
    TmaMaps maps;
    memset(&maps, 0, sizeof(maps));
    if (!tma_make_map(&maps.field, p.field, 8, p, NB, G::LB)) return cudaErrorInvalidValue;
    // pad = 2: the planes are [ap_ny][ap_nx]; along a line only slots < L/2 (x < ap_nx) exist, the TMA unit fills
    // the rest of a loaded tile with zeros and clips the stored one (needs the line to be the whole x axis: n_m = 1)
    const long long pslots = p.ap_nx > 0 ? p.L / 2 : 0, pso = p.ap_nx > 0 ? p.ap_nx : 0;
    if (p.ap_nx > 0 && (p.n_m != 1 || G::PIN == false)) return cudaErrorInvalidValue;
    if (G::PIN && !(V == V_STOTHER && p.store_op != ST_C64_STATS)) {
        const float* src = (V == V_LOSS || V == V_LDOTHER || V == V_STOTHER) ? p.plane_in : p.height;
        if (!tma_make_map(&maps.pin, src, 4, p, NB, G::LB, pslots, pso)) return cudaErrorInvalidValue;
    }
    if (V == V_GRAD || (V == V_LOSS && p.write_intensity) ||
        (V == V_STOTHER && (p.store_op == ST_C64_INTENSITY || p.write_intensity))) {
        if (!tma_make_map(&maps.pout, p.plane_out, 4, p, NB, G::LB, pslots, pso)) return cudaErrorInvalidValue;
    }
    const int per_sm = (p.device >= 0 && p.device < 64) ? resident[p.device].load() : 1;
    long long grid = (long long)tma_sm_count(p.device) * (per_sm < 1 ? 1 : per_sm);
    if (grid > ntiles) grid = ntiles;
    tma_col_kernel<L, NB, V, TWB, NST><<<(unsigned)grid, G::THREADS, G::SMEM, stream>>>(p, maps, (unsigned)ntiles);
    return cudaGetLastError();
}

// all variants of one (digit length, bundle width, pipeline depth)
template <int L, int NB, int NST>
cudaError_t launch_tma(const PassDesc& p, int variant, int twb, cudaStream_t st)
{
    if (twb == TWB_NONE) {
        if constexpr (L % 3 != 0) {
            if (variant == V_H) return launch_tma_one<L, NB, V_H, TWB_NONE, NST>(p, st);
            if (variant == V_GAUSS) return launch_tma_one<L, NB, V_GAUSS, TWB_NONE, NST>(p, st);
        }
    } else if (twb == TWB_TILE) {
        if (variant == V_FWD) return launch_tma_one<L, NB, V_FWD, TWB_TILE, NST>(p, st);
        if (variant == V_INV) return launch_tma_one<L, NB, V_INV, TWB_TILE, NST>(p, st);
    } else {
        if (variant == V_FWD) return launch_tma_one<L, NB, V_FWD, TWB_LANE, NST>(p, st);
        if (variant == V_INV) return launch_tma_one<L, NB, V_INV, TWB_LANE, NST>(p, st);
        if constexpr (L % 3 != 0) {
            if (variant == V_LOSS) return launch_tma_one<L, NB, V_LOSS, TWB_LANE, NST>(p, st);
            if (variant == V_HEIGHT) return launch_tma_one<L, NB, V_HEIGHT, TWB_LANE, NST>(p, st);
            if (variant == V_GRAD) return launch_tma_one<L, NB, V_GRAD, TWB_LANE, NST>(p, st);
            if (variant == V_LDOTHER && (p.load_op == LD_SEED || p.load_op == LD_SEED_SIMSE))
                return launch_tma_one<L, NB, V_LDOTHER, TWB_LANE, NST>(p, st);
            if (variant == V_STOTHER && (p.store_op == ST_C64_INTENSITY || p.store_op == ST_C64_STATS))
                return launch_tma_one<L, NB, V_STOTHER, TWB_LANE, NST>(p, st);
        }
    }
    return kNotInstantiated;
}

} // namespace dop
