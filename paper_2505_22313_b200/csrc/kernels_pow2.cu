// kernels_pow2.cu -- dispatcher of the register-blocked power-of-two tile-pass kernels
// (pow2_impl.cuh; instantiated per digit length in pow2_inst.cu) and their host-side tables.
#include <cstdlib>

#include "cluster_row.cuh"
#include "tma_col.cuh"

namespace dop {

extern template cudaError_t launch_cluster<4096, 2>(const PassDesc&, int, cudaStream_t);
extern template cudaError_t launch_cluster<4096, 1>(const PassDesc&, int, cudaStream_t);
extern template cudaError_t launch_cluster<2048, 4>(const PassDesc&, int, cudaStream_t);
extern template cudaError_t launch_cluster<1024, 8>(const PassDesc&, int, cudaStream_t);

// explicit instantiations live in the pow2_inst.cu objects
#define DOP_DECL(L, COL) extern template cudaError_t launch_L<L, COL>(const PassDesc&, int, int, cudaStream_t);
DOP_DECL(16, true) DOP_DECL(32, true) DOP_DECL(64, true) DOP_DECL(128, true) DOP_DECL(256, true) DOP_DECL(512, true)
DOP_DECL(64, false) DOP_DECL(128, false) DOP_DECL(256, false) DOP_DECL(512, false) DOP_DECL(1024, false)
DOP_DECL(2048, false) DOP_DECL(4096, false) DOP_DECL(8192, false)
#undef DOP_DECL
extern template cudaError_t launch_x3<16>(const PassDesc&, int, int, cudaStream_t);
extern template cudaError_t launch_x3<32>(const PassDesc&, int, int, cudaStream_t);
extern template cudaError_t launch_x3<64>(const PassDesc&, int, int, cudaStream_t);
extern template cudaError_t launch_x3<128>(const PassDesc&, int, int, cudaStream_t);

// TMA column kernels (tma_col.cuh): (digit length, bundle width, pipeline depth) instantiated in the tma_inst.cu
// objects -- the same list as TMA_INST in build.py
#define DOP_TMA_LIST(X) \
    X(16, 32, 3) X(32, 32, 3) X(64, 32, 3) X(64, 16, 3) X(128, 32, 3) X(128, 16, 3) X(256, 32, 2) X(256, 16, 3) X(256, 16, 2) X(512, 16, 2) \
    X(96, 32, 3) X(192, 32, 3) X(384, 32, 2)
#define DOP_TMA_DECL(L, NB, NST) extern template cudaError_t launch_tma<L, NB, NST>(const PassDesc&, int, int, cudaStream_t);
DOP_TMA_LIST(DOP_TMA_DECL)
#undef DOP_TMA_DECL

bool tma_instantiated(long long L, int nb, int nst)
{
#define DOP_TMA_HAS(LL, NB, NST) if (L == LL && nb == NB && nst == NST) return true;
    DOP_TMA_LIST(DOP_TMA_HAS)
#undef DOP_TMA_HAS
    return false;
}

TmaEncodeFn tma_encode_fn()
{
    static TmaEncodeFn fn = [] {
        void* f = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess ||
            q != cudaDriverEntryPointSuccess)
            f = nullptr;
        return (TmaEncodeFn)f;
    }();
    return fn;
}

int tma_sm_count(int device)
{
    static std::atomic<int> sms[64];
    if (device < 0 || device >= 64) return 148;
    int n = sms[device].load();
    if (n == 0) {
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, device) != cudaSuccess || n < 1) n = 148;
        sms[device].store(n);
    }
    return n;
}

bool tma_make_map(CUtensorMap* map, const void* base, int eb, const PassDesc& p, int nb, int lb, long long slots, long long so)
{
    TmaEncodeFn enc = tma_encode_fn();
    if (enc == nullptr || base == nullptr || ((uintptr_t)base & 15) != 0) return false;
    // (slots / so: pad = 2 planes -- only the first L/2 slots of a line lie inside the aperture, whose rows are ap_nx long)
    const cuuint64_t dims[4] = {(cuuint64_t)p.NC, (cuuint64_t)p.n_m, (cuuint64_t)(slots > 0 ? slots : p.L), (cuuint64_t)(p.n_o + p.o0)};
    cuuint64_t strides[3] = {(cuuint64_t)p.SM * eb, (cuuint64_t)p.es * eb, (cuuint64_t)(so > 0 ? so : p.SO) * eb};
    for (int i = 0; i < 3; ++i) {
        if (dims[i + 1] == 1 && strides[i] == 0) strides[i] = 16; // (a dimension of extent 1: the stride is never used)
        if (strides[i] % 16 != 0 || strides[i] >= (1ull << 40)) return false;
    }
    for (int i = 0; i < 4; ++i)
        if (dims[i] == 0 || dims[i] > 0xffffffffull) return false;
    const cuuint32_t box[4] = {(cuuint32_t)nb, 1, (cuuint32_t)lb, 1};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    const CUtensorMapDataType dt = eb == 8 ? CU_TENSOR_MAP_DATA_TYPE_UINT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
    // L2 promotion no wider than one row of the box: with 64-byte rows (16 columns of an fp32 plane) a 128-byte
    // promotion fetched every row twice (ncu at C5: the loss pass read 1.17x its algorithmic bytes)
    const CUtensorMapL2promotion promo = nb * eb >= 256 ? CU_TENSOR_MAP_L2_PROMOTION_L2_256B
                                         : nb * eb >= 128 ? CU_TENSOR_MAP_L2_PROMOTION_L2_128B : CU_TENSOR_MAP_L2_PROMOTION_L2_64B;
    return enc(map, dt, 4, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, promo, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

static cudaError_t launch_tma_pass(const PassDesc& p, int v, int twb, cudaStream_t stream)
{
#define DOP_TMA_CASE(LL, NB, NST) if (p.L == LL && p.nl == NB && p.tma == NST) return launch_tma<LL, NB, NST>(p, v, twb, stream);
    DOP_TMA_LIST(DOP_TMA_CASE)
#undef DOP_TMA_CASE
    return kNotInstantiated;
}

bool pow2_supported(long long L, bool col_type)
{
    if (col_type && L % 3 == 0) { // 3 * 2^k, k = 4..7: radix-3 step + three 2^k sub-tiles (plain passes only)
        const long long lp = L / 3;
        return lp >= 16 && lp <= 128 && (lp & (lp - 1)) == 0;
    }
    if (L < 16 || (L & (L - 1)) != 0) return false;
    return col_type ? L <= 512 : (L >= 64 && L <= 8192);
}

// Lines per tile.  Column tiles: the bundle width NB.  `plain` = a plain forward / inverse pass or
// the exp(i Phi) pass: measured on B200, 32-column bundles (256-byte segments) take those from
// 0.67-0.71 to 0.75-0.83 of the measured copy bandwidth (C4 L = 256, C3 L = 128), but cost the
// register-heavy fused variants (H, loss) 15-30 %, and 64 columns lose everywhere.
// nb_override (DOP_COL_NB = 16 | 32 | 64, read at plan creation) applies to every column tile, clamped
// to what is instantiated.
int pow2_lines(long long L, bool col_type, bool plain, int nb_override)
{
    if (!col_type) return row_lines((int)L);
    int nb = (plain && L >= 128) ? 32 : 16;
    if (nb_override == 16 || nb_override == 32 || nb_override == 64) nb = nb_override;
    if (L % 3 == 0) return nb > 32 ? 32 : nb; // 3 * 2^k digits: 16 or 32 columns
    const int mx = max_col_nb((int)L);
    return nb < mx ? nb : mx;
}

// which fused-op variant a pass is, or -1 if the fast kernels do not implement the combination
static int pass_variant(const PassDesc& p)
{
    const int d1 = p.fft1_dir, d2 = p.fft2_dir;
    if (p.mid_op == MID_H || p.mid_op == MID_HCONJ)
        return (d1 > 0 && d2 < 0 && p.load_op == LD_C64 && p.store_op == ST_C64) ? V_H : -1;
    if (p.mid_op == MID_GAUSS) return (d1 > 0 && d2 < 0 && p.load_op == LD_C64 && p.store_op == ST_C64) ? V_GAUSS : -1;
    if (p.mid_op == MID_LOSS) return (d1 < 0 && d2 > 0 && p.load_op == LD_C64 && p.store_op == ST_C64) ? V_LOSS : -1;
    if (d2 != 0) return -1;
    if (d1 > 0) {
        if (p.store_op != ST_C64) return -1;
        if (p.load_op == LD_C64) return V_FWD;
        if (p.load_op == LD_HEIGHT) return V_HEIGHT;
        return V_LDOTHER; // LD_SEED, LD_REAL
    }
    if (p.load_op != LD_C64) return -1;
    if (p.store_op == ST_C64) return V_INV;
    if (p.store_op == ST_GRAD || p.store_op == ST_GRAD_ACC) return V_GRAD;
    return V_STOTHER; // ST_C64_INTENSITY, ST_REAL
}

// x axes of 16 M points (M = 1024, 2048, 4096) can run their two digit passes (16, M) as one
// thread-block-cluster pass (cluster_row.cuh)
bool cluster_supported(long long L0, long long L1) { return L0 == 16 && (L1 == 1024 || L1 == 2048 || L1 == 4096); }
int cluster_size(long long L1) { return L1 == 4096 ? 8 : (L1 == 2048 ? 4 : 2); }
bool cluster_instantiated(long long L1, int lines)
{
    return (L1 == 4096 && (lines == 2 || lines == 1)) || (L1 == 2048 && lines == 4) || (L1 == 1024 && lines == 8);
}

static cudaError_t launch_cluster_pass(const PassDesc& p, cudaStream_t stream)
{
    const int v = pass_variant(p);
    if (v < 0 || p.tw_g == nullptr || p.tw_b2 == nullptr) return cudaErrorInvalidValue;
    switch (p.L * 16 + p.nl) {
    case 4096 * 16 + 2: return launch_cluster<4096, 2>(p, v, stream);
    case 4096 * 16 + 1: return launch_cluster<4096, 1>(p, v, stream);
    case 2048 * 16 + 4: return launch_cluster<2048, 4>(p, v, stream);
    case 1024 * 16 + 8: return launch_cluster<1024, 8>(p, v, stream);
    }
    return cudaErrorInvalidValue;
}

cudaError_t launch_tile_pass_pow2(const PassDesc& p, cudaStream_t stream, bool* handled)
{
    *handled = false;
    if (p.cluster) { // a cluster pass has no other implementation: the plan only schedules supported ones
        *handled = true;
        return launch_cluster_pass(p, stream);
    }
    const bool col = p.col_type != 0;
    if (p.tw_g == nullptr || !pow2_supported(p.L, col)) return cudaSuccess;
    if (col ? !(p.nl == 16 || p.nl == 32 || p.nl == 64) : p.nl != pow2_lines(p.L, false)) return cudaSuccess;
    const int v = pass_variant(p);
    if (v < 0) return cudaSuccess;
    if ((v == V_H || v == V_GAUSS) && (!col || p.row_i != 1)) return cudaSuccess;
    int twb = TWB_NONE;
    if (p.tw_b != nullptr) {
        if (p.tw_b2 == nullptr || !col) return cudaSuccess;
        twb = p.r_from == 1 ? TWB_TILE : TWB_LANE;
    }
    cudaError_t e = kNotInstantiated;
    if (p.tma > 0 && col) { // the plan only marks passes whose variant the TMA kernels implement
        e = launch_tma_pass(p, v, twb, stream);
        if (e != kNotInstantiated) {
            *handled = true;
            return e;
        }
    }
    if (p.NC % p.nl != 0) return cudaSuccess; // (a ragged last tile: only the TMA kernels clip it; else the generic kernel)
    if (p.L % 3 == 0) {
        switch (p.L / 3) {
        case 16: e = launch_x3<16>(p, v, twb, stream); break;
        case 32: e = launch_x3<32>(p, v, twb, stream); break;
        case 64: e = launch_x3<64>(p, v, twb, stream); break;
        case 128: e = launch_x3<128>(p, v, twb, stream); break;
        }
    } else if (col) {
        switch (p.L) {
        case 16: e = launch_L<16, true>(p, v, twb, stream); break;
        case 32: e = launch_L<32, true>(p, v, twb, stream); break;
        case 64: e = launch_L<64, true>(p, v, twb, stream); break;
        case 128: e = launch_L<128, true>(p, v, twb, stream); break;
        case 256: e = launch_L<256, true>(p, v, twb, stream); break;
        case 512: e = launch_L<512, true>(p, v, twb, stream); break;
        }
    } else {
        switch (p.L) {
        case 64: e = launch_L<64, false>(p, v, twb, stream); break;
        case 128: e = launch_L<128, false>(p, v, twb, stream); break;
        case 256: e = launch_L<256, false>(p, v, twb, stream); break;
        case 512: e = launch_L<512, false>(p, v, twb, stream); break;
        case 1024: e = launch_L<1024, false>(p, v, twb, stream); break;
        case 2048: e = launch_L<2048, false>(p, v, twb, stream); break;
        case 4096: e = launch_L<4096, false>(p, v, twb, stream); break;
        case 8192: e = launch_L<8192, false>(p, v, twb, stream); break;
        }
    }
    if (e == kNotInstantiated) return cudaSuccess; // combination not instantiated: generic kernel
    *handled = true;
    return e;
}

// Twiddle tables of the register-blocked schedule of a digit of length L (layout of fft_regs.cuh:
// group g at twoff(g), entry (k-1) m_g + j = W_{n_g}^{j k}), computed in long double.
std::vector<float2> pow2_group_twiddles(long long L)
{
    std::vector<float2> out;
    if (L % 3 == 0) L /= 3; // digits 3 * 2^k: the tables of the 2^k sub-transform
    int lg = 0;
    while ((1LL << lg) < L) ++lg;
    const int n4 = lg / 2, n2 = lg & 1, nfull = n4 / 2, rlast = ((n4 & 1) ? 4 : 1) * (n2 ? 2 : 1);
    const int ng = nfull + (rlast > 1 ? 1 : 0);
    long long n = L;
    const long double pi = 3.141592653589793238462643383279502884L;
    for (int g = 0; g < ng; ++g) {
        const int R = g < nfull ? 16 : rlast;
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
