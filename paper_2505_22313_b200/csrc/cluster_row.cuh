// cluster_row.cuh -- one pass over a long contiguous row (nx = 16 M, M = 1024 / 2048 / 4096) by a
// thread-block cluster: the two x digit passes (16, M) of pow2_impl.cuh fused into ONE read and ONE
// write of the field, the intermediate crossing the chip through distributed shared memory instead
// of HBM (PAPER.md:200 row-column 2-D FFT; "rows 512 KiB -- a cluster of 4-8 CTAs
// exchanging through DSMEM").
//
// A cluster of C = 16/S CTAs (512 threads each) owns one row.  With n = n1 M + n2 (n1 < 16, n2 < M):
//   natural layout : CTA `rank` holds n2 in [512 rank, 512 rank + 512) for all 16 n1; thread t keeps
//                    the 16 values x[n1 M + 512 rank + t] in registers (coalesced across lanes).
//   line layout    : CTA `rank` holds the S sub-transforms ("lines") slot_c = rank S + sub, each an
//                    M-point line at rbase + slot_c M, in the register layouts of fft_regs.cuh.
// forward : natural -> radix-16 over n1 in registers -> twiddle W_N^{n2 k1} -> all-to-all through
//           DSMEM (st.shared::cluster) -> M-point forward DFT per line -> contiguous store.
// inverse : the exact mirror.  Slot order = that of the digit passes (16, M), so a plan may run
//           either and the H tables are the same.
// Fused pointwise ops ride on the natural layout: exp(i Phi) load (F1, F2), |u|^2 + loss + seed
// (F6, F7, A1) between an inverse and a forward, Im(conj(u0) g) store (A5), and the
// DOP_LOSS_NONE / pre-filter loads and stores.
#pragma once
#include "pow2_impl.cuh"

namespace dop {

__device__ __forceinline__ unsigned cl_smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ unsigned cl_mapa(unsigned addr, unsigned rank)
{
    unsigned r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
__device__ __forceinline__ void cl_st(unsigned addr, float2 v)
{
    asm volatile("st.shared::cluster.v2.f32 [%0], {%1,%2};" ::"r"(addr), "f"(v.x), "f"(v.y) : "memory");
}
__device__ __forceinline__ unsigned cl_rank()
{
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
// cluster-wide barrier with release / acquire semantics: DSMEM writes before it are visible after it
__device__ __forceinline__ void cl_sync()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

template <int M, int S>
constexpr int cluster_smem_bytes() { return S * fx::Tile<M, false>::LINE_ELEMS * (int)sizeof(float2); }

// XCHG selects how the intermediate crosses between the two layouts:
//   XCHG_DSMEM : st.shared::cluster into the peers' exchange buffers.  Measured on B200: the DSMEM
//                all-to-all sustains only 10-13 B/clk/SM (profiles/r02_cluster.md), about half of
//                an SM's share of HBM bandwidth, and needs two extra buffer-free barriers.
//   XCHG_L2    : the intermediate is written to and re-read from the field itself (in place, the
//                positions the digit passes (16, M) would use), ordered by the cluster barrier; it is
//                rewritten with the pass's result a few microseconds later, long before the 126 MB L2
//                would evict it, so HBM sees one read and one write per point.  The cluster then only
//                provides co-scheduling and the hardware barrier.
enum : int { XCHG_DSMEM = 0, XCHG_L2 = 1 };

__device__ __forceinline__ float2 ld_cg_v(const float2* p) // volatile flavour: never hoisted above the cluster barrier
{
    float2 v;
    asm volatile("ld.global.cg.v2.f32 {%0,%1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p) : "memory");
    return v;
}

template <int M, int S, int V, int XCHG>
__global__ void __cluster_dims__(16 / S, 1, 1) __launch_bounds__(S * (M / P), 1024 / (S * (M / P)))
cluster_row_kernel(const __grid_constant__ PassDesc p)
{
    constexpr int kClThreads = S * (M / P); // threads per CTA = points per CTA / 16
    constexpr int kClSeg = kClThreads;      // n2 values per CTA in the natural layout
    using TL = fx::Tile<M, false>;
    using SC = fx::Sched<M>;
    constexpr int C = 16 / S;
    constexpr int T = M / P;                 // threads per line of the local transform
    constexpr int GL = SC::NG - 1;
    constexpr int DIR1 = variant_dir1(V), DIR2 = variant_dir2(V);
    constexpr int LAST = DIR2 != 0 ? DIR2 : DIR1;
    constexpr int PER = kClSeg / T;          // registers of a line thread that go to the same CTA
    static_assert(S * T == kClThreads && M / C == kClSeg && TL::CONTIG && T >= 32, "cluster row geometry");
    extern __shared__ float2 s[];

    const int tid = threadIdx.x;
    const unsigned rank = cl_rank();
    const long long row = (long long)(blockIdx.x / C) + p.o0;
    const long long rbase = row * (16LL * M);
    const int n2 = (int)rank * kClSeg + tid;                 // natural layout: register c <-> n = c M + n2
    const long long nat0 = rbase + n2;
    const int sub = tid / T, tt = tid % T, lane = tid & 31;  // line layout
    const int soff = sub * TL::LINE_ELEMS;
    const long long lbase = rbase + (long long)((int)rank * S + sub) * M;
    const float2* __restrict__ tw = p.tw_g;
    const float2* __restrict__ twp = p.tw_b2 + n2;           // W_N^{n2 pi[c]} at twp[c M]
    const unsigned sbase = cl_smem_u32(s);

    float2 v[P];
    const bool lay = (p.up_lg | p.h_dtype | p.coarse_in | p.pool_out) != 0; // design-layout addressing (uniform)

    // ---- staged contiguous line access (last-group layout: thread owns slots 16 tt .. 16 tt + 15, a
    //      warp 512 adjacent slots = 4 KiB; pow2_impl.cuh "STAGE")
    auto stg_addr = [&](int e) -> int { return soff + TL::addr((tt - lane) * P + e, 0); };
    const long long stg_base = lbase + (long long)(tt - lane) * P;

    auto load_lines = [&]() {
        const float2* g0 = p.field + stg_base;
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
    };
    auto store_lines = [&]() {
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
    };

    // ---- all-to-all, natural -> lines: register c (slot c of digit 0) goes to CTA c / S, line c % S,
    //      position n2 of that line (group-0 layout of the local transform)
    auto send_to_lines = [&]() {
        const unsigned a0 = sbase + (unsigned)TL::addr(n2, 0) * 8u;
#pragma unroll
        for (int c = 0; c < P; ++c)
            cl_st(cl_mapa(a0 + (unsigned)((c % S) * TL::LINE_ELEMS * 8), (unsigned)(c / S)), v[c]);
    };
    auto recv_lines = [&]() { // register i <-> slot tt + i T
        TL::template from_smem<0>(v, s, tt, soff);
    };
    // ---- all-to-all, lines -> natural: register i of line slot_c holds n2' = tt + i T; it goes to CTA
    //      n2' / 512 at [slot_c][n2' % 512]
    auto send_to_natural = [&]() {
        const unsigned a0 = sbase + (unsigned)((((int)rank * S + sub) * kClSeg + tt) * 8);
#pragma unroll
        for (int i = 0; i < P; ++i)
            cl_st(cl_mapa(a0 + (unsigned)((i % PER) * T * 8), (unsigned)(i / PER)), v[i]);
    };
    auto recv_natural = [&]() {
#pragma unroll
        for (int c = 0; c < P; ++c) v[c] = s[c * kClSeg + tid];
    };

    // =========================================================================================
    if (DIR1 > 0) {
        // ---- natural-layout load (+ prologue op)
        if ((V == V_HEIGHT && lay) || (V == V_LDOTHER && p.coarse_in)) {
            // design layout: nearest up-sampling / gray levels inside the read (apart from the plain loop below)
#pragma unroll
            for (int c = 0; c < P; ++c) {
                const float hv = ld_layout(V == V_HEIGHT ? (const void*)p.height : (const void*)p.plane_in, p.h_dtype, p.h_step,
                                           p.up_lg, p.cnx, row, n2 + c * M);
                if (V == V_HEIGHT) sincos_turns(hv * p.phase_coef, &v[c].y, &v[c].x);
                else v[c] = make_float2(hv, 0.0f);
            }
        } else {
#pragma unroll
        for (int c = 0; c < P; ++c) {
            const long long off = nat0 + (long long)c * M;
            if (V == V_HEIGHT) {
                const float ph = __ldg(p.height + off) * p.phase_coef; // Eq. (1) in turns
                sincos_turns(ph, &v[c].y, &v[c].x);                    // Eq. (2), E_in = 1
            } else if (V == V_LDOTHER) {
                if (p.load_op == LD_SEED) {
                    const float2 u = p.field[off];
                    const float g = 2.0f * __ldg(p.plane_in + off);
                    v[c] = make_float2(g * u.x, g * u.y);
                } else if (p.load_op == LD_SEED_SIMSE) {               // Eq. (6): 2 dL/dI = c0 + cI I + cT T
                    const float2 u = p.field[off];
                    const float I = u.x * u.x + u.y * u.y;
                    const float g = fmaf(__ldg(p.coef + 1), I, fmaf(__ldg(p.coef + 2), __ldg(p.plane_in + off), __ldg(p.coef)));
                    v[c] = make_float2(g * u.x, g * u.y);
                } else {
                    v[c] = make_float2(__ldg(p.plane_in + off), 0.0f);
                }
            } else {
                v[c] = p.field[off];
            }
        }
        }
    } else {
        load_lines();
        TL::template inverse<GL, false>(v, s, tt, soff, tw);
        if (XCHG == XCHG_DSMEM) {
            cl_sync();        // every CTA of the cluster is done with its exchange buffer
            send_to_natural();
            cl_sync();
            recv_natural();
        } else {              // group-0 layout: register i <-> position tt + i T of the line, coalesced
#pragma unroll
            for (int i = 0; i < P; ++i) st_cg(p.field + lbase + tt + i * T, v[i]);
            cl_sync();
#pragma unroll
            for (int c = 0; c < P; ++c) v[c] = ld_cg_v(p.field + nat0 + (long long)c * M);
        }
#pragma unroll
        for (int c = 1; c < P; ++c) v[c] = fx::cmulc(v[c], __ldg(twp + c * M));
        fx::group<4, 4, -1, 1>(v);
    }

    // ---- middle op (natural layout)
    __shared__ double red[kClThreads / 32]; // V_LOSS: per-warp partial sums of the tile's loss
    if (V == V_LOSS) {
        double acc = 0.0;
#pragma unroll
        for (int c = 0; c < P; ++c) {
            const long long off = nat0 + (long long)c * M;
            const float I = v[c].x * v[c].x + v[c].y * v[c].y; // F6
            const float d = I - __ldg(p.plane_in + off);       // F7
            acc += (double)d * (double)d;
            const float g = p.seed_coef * d;                   // A1: 2 gI = 4 (I - T)/N
            v[c] = make_float2(g * v[c].x, g * v[c].y);
            if (p.write_intensity) p.plane_out[off] = I;
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, d);
        if (lane == 0) red[tid >> 5] = acc; // (summed by thread 0 after the cluster barriers of the exchange below)
    }

    if (LAST > 0) {
        // ---- radix-16 over n1, twiddle, all-to-all, local forward transform, contiguous store
        fx::group<4, 4, +1, 1>(v);
#pragma unroll
        for (int c = 1; c < P; ++c) v[c] = fx::cmul(v[c], __ldg(twp + c * M));
        if (XCHG == XCHG_DSMEM) {
            cl_sync();        // all CTAs started (DIR1 > 0) / have read their receive buffers (V_LOSS)
            send_to_lines();
            cl_sync();
            recv_lines();
            __syncthreads();
        } else {
#pragma unroll
            for (int c = 0; c < P; ++c) st_cg(p.field + nat0 + (long long)c * M, v[c]);
            cl_sync();
#pragma unroll
            for (int i = 0; i < P; ++i) v[i] = ld_cg_v(p.field + lbase + tt + i * T); // group-0 layout, coalesced
        }
        TL::template forward<0, true>(v, s, tt, soff, tw);
        store_lines();
        if (V == V_LOSS && tid == 0) { // deterministic: warp order; off the path of the other warps
            double r = 0.0;
            for (int w = 0; w < kClThreads / 32; ++w) r += red[w];
            p.loss_scratch[p.tile0 + blockIdx.x] = r;
        }
    } else {
        // ---- natural-layout store (+ epilogue op)
        double st0 = 0.0, st1 = 0.0, st2 = 0.0, st3 = 0.0; // ST_C64_STATS: <I,T>, <I,I>, sum I, <T,T>
        if ((V == V_GRAD && (lay || p.adam_m != nullptr)) || (V == V_STOTHER && p.pool_out)) {
            // design-loop flavours of the two real-plane stores (apart from the plain loop below)
            const bool leader = (tid & ((1 << p.up_lg) - 1)) == 0;
#pragma unroll
            for (int c = 0; c < P; ++c) {
                const long long off = nat0 + (long long)c * M;
                if (V == V_GRAD) {
                    const float hv = lay ? ld_layout(p.height, p.h_dtype, p.h_step, p.up_lg, p.cnx, row, n2 + c * M)
                                         : __ldg(p.height + off);
                    float sn, cs;
                    sincos_turns(hv * p.phase_coef, &sn, &cs);
                    float g = p.grad_coef * (cs * v[c].y - sn * v[c].x); // A5: c Im(conj(u0) g)
                    if (p.pool_out) {
                        g = pool_lanes(g, p.up_lg, 0xffffffffu);
                        const long long ci = row * p.cnx + ((n2 + c * M) >> p.up_lg);
                        if (leader) {
                            if (p.store_op == ST_GRAD_ACC) g += p.plane_out[ci];
                            p.plane_out[ci] = g;
                        }
                    } else {
                        if (p.store_op == ST_GRAD_ACC) g += __ldg(p.plane_out + off);
                        p.plane_out[off] = g;
                        if (p.adam_m != nullptr)
                            p.adam_h[off] = adam_update(g, hv, p.adam_m + off, p.adam_v + off, p.adam_b1, p.adam_b2, p.adam_c1,
                                                        p.adam_c2, p.adam_a1, p.adam_rb2, p.adam_eps);
                    }
                } else {
                    const float g = pool_lanes(v[c].x, p.up_lg, 0xffffffffu);
                    if (leader) p.plane_out[row * p.cnx + ((n2 + c * M) >> p.up_lg)] = g;
                }
            }
        } else {
#pragma unroll
        for (int c = 0; c < P; ++c) {
            const long long off = nat0 + (long long)c * M;
            if (V == V_GRAD) {
                const float ph = __ldg(p.height + off) * p.phase_coef;
                float sn, cs;
                sincos_turns(ph, &sn, &cs); // u0 recomputed, not stored
                float g = p.grad_coef * (cs * v[c].y - sn * v[c].x); // A5: c Im(conj(u0) g)
                if (p.store_op == ST_GRAD_ACC) g += __ldg(p.plane_out + off);
                p.plane_out[off] = g;
            } else if (V == V_STOTHER) {
                if (p.store_op == ST_C64_INTENSITY) {
                    p.field[off] = v[c];
                    p.plane_out[off] = v[c].x * v[c].x + v[c].y * v[c].y;
                } else if (p.store_op == ST_C64_STATS) {
                    p.field[off] = v[c];
                    const float I = v[c].x * v[c].x + v[c].y * v[c].y;
                    const float Tv = __ldg(p.plane_in + off);
                    st0 += (double)I * (double)Tv;
                    st1 += (double)I * (double)I;
                    st2 += (double)I;
                    st3 += (double)Tv * (double)Tv;
                    if (p.write_intensity) p.plane_out[off] = I;
                } else {
                    p.plane_out[off] = v[c].x;
                }
            } else {
                p.field[off] = v[c];
            }
        }
        }
        if (V == V_STOTHER) {
            if (p.store_op == ST_C64_STATS) {
                __shared__ double sred[4][kClThreads / 32];
#pragma unroll
                for (int d = 16; d > 0; d >>= 1) {
                    st0 += __shfl_down_sync(0xffffffffu, st0, d);
                    st1 += __shfl_down_sync(0xffffffffu, st1, d);
                    st2 += __shfl_down_sync(0xffffffffu, st2, d);
                    st3 += __shfl_down_sync(0xffffffffu, st3, d);
                }
                if (lane == 0) {
                    sred[0][tid >> 5] = st0; sred[1][tid >> 5] = st1; sred[2][tid >> 5] = st2; sred[3][tid >> 5] = st3;
                }
                __syncthreads();
                if (tid < 4) {
                    double r = 0.0;
                    for (int w = 0; w < kClThreads / 32; ++w) r += sred[tid][w];
                    p.loss_scratch[4 * (p.tile0 + blockIdx.x) + tid] = r;
                }
            }
        }
    }
}

template <int M, int S, int V, int XCHG>
static cudaError_t launch_cluster_one(const PassDesc& p, cudaStream_t stream)
{
    constexpr int smem = cluster_smem_bytes<M, S>();
    constexpr int kClThreads = S * (M / P);
    static AttrOnce once;
    cudaError_t e = once.ensure(p.device, [] {
        cudaError_t a = cudaFuncSetAttribute(cluster_row_kernel<M, S, V, XCHG>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (a != cudaSuccess) return a;
        if (16 / S > 8) {
            a = cudaFuncSetAttribute(cluster_row_kernel<M, S, V, XCHG>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
            if (a != cudaSuccess) return a;
        }
        return cudaFuncSetAttribute(cluster_row_kernel<M, S, V, XCHG>, cudaFuncAttributePreferredSharedMemoryCarveout,
                                    cudaSharedmemCarveoutMaxShared);
    });
    if (e != cudaSuccess) return e;
    const long long nctas = p.n_o * (16 / S);
    if (nctas <= 0 || nctas > 2147483647LL) return cudaErrorInvalidConfiguration;
    cluster_row_kernel<M, S, V, XCHG><<<(unsigned)nctas, kClThreads, smem, stream>>>(p);
    return cudaGetLastError();
}

template <int M, int S, int XCHG>
cudaError_t launch_cluster_x(const PassDesc& p, int variant, cudaStream_t st)
{
    switch (variant) {
    case V_FWD: return launch_cluster_one<M, S, V_FWD, XCHG>(p, st);
    case V_INV: return launch_cluster_one<M, S, V_INV, XCHG>(p, st);
    case V_LOSS: return launch_cluster_one<M, S, V_LOSS, XCHG>(p, st);
    case V_HEIGHT: return launch_cluster_one<M, S, V_HEIGHT, XCHG>(p, st);
    case V_LDOTHER: return launch_cluster_one<M, S, V_LDOTHER, XCHG>(p, st);
    case V_GRAD: return launch_cluster_one<M, S, V_GRAD, XCHG>(p, st);
    case V_STOTHER: return launch_cluster_one<M, S, V_STOTHER, XCHG>(p, st);
    }
    return kNotInstantiated;
}

template <int M, int S>
cudaError_t launch_cluster(const PassDesc& p, int variant, cudaStream_t st)
{
    return p.cluster == 2 ? launch_cluster_x<M, S, XCHG_DSMEM>(p, variant, st) : launch_cluster_x<M, S, XCHG_L2>(p, variant, st);
}

} // namespace dop
