// dop_internal.h -- shared declarations of the CUDA path (plan <-> kernels <-> C-ABI).
// Nothing here is shared with oracle/ (the oracle is independent test infrastructure).
//
// Vocabulary ("Decomposition"):
//   axis    x (contiguous, length nx) or y (strided, length ny).
//   digit   an axis length N is factored N = L_0 L_1 ... L_{m-1}; index n = sum n_j st_j with
//           st_j = prod_{i>j} L_i.  One *pass* (one kernel launch, one read + one write of the
//           field) transforms one digit of one axis: an L_j-point in-place DFT on every line
//           {base + i*es, i < L_j}.  Forward = decimation in frequency: digits most-significant
//           first, then the "boundary twiddle" T_j = W_{N_j}^{k_j r_j} (N_j = L_j st_j,
//           r_j = n mod st_j).  Spectra stay in this digit-scrambled slot order; the inverse is
//           the exact mirror (conj(T_j) first, digits least-significant first), so no reorder
//           pass ever runs and H is evaluated at the true frequency of each slot from tables.
//   tile    what one CTA holds on chip: nl lines x L points.
//           column-type: the nl lines are adjacent in memory (line stride 1), elements es apart;
//           row-type:    each line is L contiguous elements (es = 1).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include <string>
#include <vector>

#include "../../include/dop.h"

namespace dop {

enum LoadOp : int {
    LD_C64 = 0,     // complex64 field
    LD_HEIGHT = 1,  // Eq. (1)+(2): u0 = exp(i 2 pi (n-1) h / lambda) from the fp32 height plane
    LD_SEED = 2,    // A1 (DOP_LOSS_NONE): g_u = 2 (dL/dI) u
    LD_REAL = 3,    // pre-filter: fp32 plane -> (v, 0)
    LD_SEED_SIMSE = 4 // A1 (DOP_LOSS_SIMSE): g_u = (c0 + cI |u|^2 + cT T) u, coefficients from the plane sums
};
enum MidOp : int {
    MID_NONE = 0,
    MID_H = 1,      // (x) H_lambda of Eq. (3), scaled by 1/(ny nx)
    MID_HCONJ = 2,  // (x) conj(H_lambda) (adjoint), scaled by 1/(ny nx)
    MID_GAUSS = 3,  // pre-filter spectrum factor, scaled by 1/(ny nx)
    MID_LOSS = 4    // I = |u|^2, L2 loss partial, seed g_u = (4/N)(I - T) u  [optional I write]
};
enum StoreOp : int {
    ST_C64 = 0,
    ST_GRAD = 1,           // A5: dL/dh  = c Im(conj(u0) g)   (overwrite)
    ST_GRAD_ACC = 2,       //     dL/dh += ...                (lambda > 0)
    ST_C64_INTENSITY = 3,  // DOP_LOSS_NONE forward end: keep u, write I
    ST_REAL = 4,           // pre-filter: Re(v) -> fp32 plane
    ST_C64_STATS = 5       // DOP_LOSS_SIMSE forward end: keep u, [write I], plane sums <I,T>, <I,I>, sum I, <T,T>
};

constexpr int kMaxRadixSteps = 16;

// Everything one launch of the generic tile kernel needs (passed by value).
struct PassDesc {
    // ---- tile geometry
    int L;        // digit length
    int nl;       // lines per tile
    int col_type; // 1 = column-type tile, 0 = row-type
    long long es; // element stride (elements of the plane)
    long long NC, SCc; // lines along c: count, stride
    long long n_m, SM; // middle coordinate
    long long n_o, SO; // outer coordinate
    long long n_cgroups;
    // ---- slab launch (a launch may cover only a range of column groups / outer indices)
    long long cg0, o0; // added to the decoded cg / o
    long long tile0;   // global tile index of this launch's first tile (loss partial slot)
    int pf_ahead;      // pow2 kernels: CTA b prefetches the lines of tile b + pf_ahead into L2 (0 = off)
    // ---- in-tile DFT
    int n_radix;
    int radix[kMaxRadixSteps];
    int fft1_dir; // +1 forward (exp -), -1 inverse (exp +)
    int fft2_dir; // 0 = none
    const float2* wL;   // [L]  W_L^p = exp(-2 pi i p / L)
    const int* pi;      // [L]  slot within digit -> output index k_j
    const float2* tw_b; // [N_j] boundary twiddles W_{N_j}^p, or nullptr
    const float2* tw_b2; // the same twiddles permuted for the pow2 kernels: y digits [r][slot], x digits [slot][r]
    long long twb_n;    // N_j = L_j st_j
    const float2* tw_g; // group twiddles of the register-blocked schedule (fft_regs.cuh), or nullptr
    int r_from;         // 0: r_j = c (x digit), 1: r_j = m (y digit)
    // ---- pointwise ops
    int load_op, mid_op, store_op;
    int write_intensity;
    float2* field;
    const float* height;  // LD_HEIGHT / ST_GRAD*
    const float* plane_in; // LD_SEED: dL/dI;  LD_REAL: source;  MID_LOSS: target T
    float* plane_out;     // ST_GRAD*: grad;  ST_REAL: destination;  *_INTENSITY: I
    double* loss_scratch; // MID_LOSS: one partial per CTA;  ST_C64_STATS: four per CTA
    const float* coef;    // LD_SEED_SIMSE: (c0, cI, cT) of this wavelength
    // ---- design layout (dop_plan_desc.upsample / layout_dtype): where LD_HEIGHT / ST_GRAD* / LD_REAL (pre-filter
    //      input) find the height of fine-grid point (row, x), and where ST_GRAD* / ST_REAL (pre-filter adjoint) pool
    int up_lg;            // log2 of the up-sampling factor r (0 = none)
    int h_dtype;          // dop_layout_dtype of `height` (LD_HEIGHT, ST_GRAD*) / of plane_in (LD_REAL with coarse_in)
    float h_step;         // metres per level
    long long cnx;        // nx / r: row length of the coarse layout and of the x-pooled plane
    long long lpr;        // row-type tiles: lines per row (nx / L)
    int coarse_in;        // LD_REAL reads the coarse layout (up-sampled on the fly)
    int pool_out;         // ST_GRAD* / ST_REAL write the x-pooled plane [ny][nx / r] (sum over r adjacent lanes)
    // ---- Adam epilogue fused into the A5 store (ST_GRAD* with adam_m != nullptr; no up-sampling)
    float* adam_m;
    float* adam_v;
    float* adam_h;        // the fp32 layout, updated in place
    float adam_b1, adam_b2, adam_c1, adam_c2, adam_a1, adam_rb2, adam_eps; // c = 1 - b; a1 = lr_t / (1 - b1^t), rb2 = 1 / (1 - b2^t)
    float phase_coef;     // (n-1)/lambda   [turns per metre]
    float grad_coef;      // 2 pi (n-1)/lambda
    float scale;          // 1/(ny nx)
    float seed_coef;      // 4/(ny nx)
    double inv_lam2, z;   // H
    float hk_s[5], hk_c[5]; // scale (2 pi)^n/n! with signs: sine / cosine polynomial of H in the TMA kernels (apply_h_fixed_nb)
    int h_fixed;          // pow2 kernels: |z|/lambda < 2^19, the phase of H may be taken in 32-bit fixed point
    const double* fx2;    // [nx] slot -> fx^2   (fp64, same expression as the definition)
    const double* fy2;    // [ny] slot -> fy^2
    const float* gx;      // [nx] slot -> Gaussian factor
    const float* gy;      // [ny]
    long long row_o, row_m, row_i; // y slot of element i: o*row_o + m*row_m + i*row_i
    int smem_bytes;
    int threads;
    int cluster;          // 1 (exchange through L2) | 2 (through DSMEM) = cluster row pass (cluster_row.cuh): L = M, the x digits (16, M) fused; n_o rows
    int device;           // the plan's device (function attributes are set once per device)
    long long ap_nx, ap_ny, grid_nx; // pad = 2 (generic kernel): the caller's planes are [ap_ny][ap_nx], the field window
                          // has rows of grid_nx points; plane accesses outside the aperture are masked (ap_nx = 0: no padding)
    const int* hpair;     // (x) H pass on mirrored tile pairs (tma_hpair_kernel): n_hpair items (o_A, o_B | -1), or nullptr
    int n_hpair;
    int smooth;           // 1: plain pass of a 5-smooth digit on the register-step kernels (smooth.cu); nl / threads / smem are theirs
    int tma;              // > 0: TMA column kernel (tma_col.cuh) with this many tiles in flight per CTA; nl = its bundle width
};

cudaError_t launch_tile_pass(const PassDesc& p, cudaStream_t stream);
// register-blocked power-of-two fast path (kernels_pow2.cu)
bool pow2_supported(long long L, bool col_type);
bool cluster_supported(long long L0, long long L1);
int cluster_size(long long L1);
bool cluster_instantiated(long long L1, int lines);
bool tma_instantiated(long long L, int nb, int nst);
int pow2_lines(long long L, bool col_type, bool plain = false, int nb_override = 0);
std::vector<float2> pow2_group_twiddles(long long L);
// plain passes of the 5-smooth digits 225, 625, 900, 2500 (smooth.cu)
std::vector<int> smooth_radix(long long L);
bool smooth_supported(long long L, bool col_type);
void smooth_geometry(long long L, bool col_type, int* nl, int* threads, int* smem_bytes);
cudaError_t launch_loss_reduce(const double* scratch, long long n, double inv_n, double* d_loss,
                               cudaStream_t stream);
// DOP_LOSS_SIMSE: plane sums -> scale s, loss, seed coefficients per wavelength (kernels_generic.cu)
cudaError_t launch_simse_reduce(const double* scratch, long long tiles, int n_lambda, double npts, double beta,
                                float* coef, double* d_loss, cudaStream_t stream);
// Gaussian pre-filter as a separable spatial stencil (blur.cu): src -> tmp (rows) -> dst (columns)
cudaError_t launch_blur(const float* src, float* tmp, float* dst, long long ny, long long nx, int radius, const float* wx,
                        const float* wy, cudaStream_t st, cudaEvent_t mid_stop, cudaEvent_t mid_start);
struct AdamParams { float b1, b2, c1, c2, a1, rb2, eps; }; // c1 = 1 - b1, c2 = 1 - b2 (rounded from fp64)
// rows of the x-pooled plane -> coarse gradient [ny/r][cnx] (+ optional Adam update of the fp32 layout)
cudaError_t launch_pool_rows(const float* xpool, float* grad, long long cny, long long cnx, int r, const AdamParams* adam,
                             float* layout, float* m, float* v, cudaStream_t stream);
// pointwise Adam on a finished gradient plane (pre-filter configurations)
cudaError_t launch_adam(const float* grad, long long n, const AdamParams& adam, float* layout, float* m, float* v,
                        cudaStream_t stream);

// ------------------------------------------------------------------------------------------
// host-side plan
// ------------------------------------------------------------------------------------------
struct Digit {
    long long L = 0, st = 0;      // length, slot stride within the axis
    std::vector<int> radix;       // in-place DIF radix steps, product = L
    std::vector<int> pi;          // slot -> k_j
    int wl_index = -1;            // which W_L table
    bool has_twb = false;
    std::vector<float2> twb;      // W_{L st}^p, p < L st
    size_t twb_off = 0;           // byte offset into the device arena
    bool fast = false;            // handled by the register-blocked pow2 kernels
    bool smooth = false;          // its plain passes run on the register-step kernels of smooth.cu
    std::vector<float2> twg;      // their group twiddles
    size_t twg_off = 0;
    std::vector<float2> twb2;     // boundary twiddles in the pow2 kernels' layout (fast digits with has_twb)
    size_t twb2_off = 0;
};

struct Axis {
    long long N = 0;
    std::vector<Digit> dig;
    std::vector<long long> kslot; // slot -> frequency index in [0, N)
    std::vector<double> f2;       // slot -> f^2
    std::vector<double> fsigned;  // slot -> signed frequency f (band limit)
    std::vector<float> g;         // slot -> Gaussian factor (pre-filter)
};

enum Buf : int { BUF_NONE = 0, BUF_HEIGHT, BUF_HEFF, BUF_TARGET, BUF_INTENSITY, BUF_DLDI, BUF_GRAD };

// A pass with symbolic buffers; resolved to a PassDesc at launch time.
struct PassTmpl {
    int axis;  // 0 = x, 1 = y
    int digit;
    int fft1_dir, fft2_dir;
    int load_op, mid_op, store_op;
    std::string name;
    double bytes_per_point; // algorithmic HBM bytes per grid point of this launch
    double rd, wr, side;    // its parts: main input read, main output written, side planes (T, I, h, grad)
    int cluster = 0;        // x digits (16, M) fused into one thread-block-cluster pass
};

} // namespace dop

struct dop_plan {
    dop_plan_desc desc;
    dop_tuning tune{};          // copy of desc.tuning (zeros = defaults)
    std::vector<double> lambda, n_refr;
    dop::Axis ax[2]; // 0 = x, 1 = y
    std::vector<std::vector<float2>> wl_tables; // distinct W_L tables
    std::vector<long long> wl_len;
    std::vector<size_t> wl_off;
    int tile_pts = 4096;
    int col_nb = 0;             // DOP_COL_NB override of the column bundle width (0 = per-pass default)
    bool h_float = false;       // DOP_H_FLOAT: never take H's phase in fixed point
    int slab_streams = 2;       // DOP_SLAB_STREAMS
    int pf_waves = 1;           // L2 prefetch distance of the pow2 kernels, in waves of resident CTAs (0 = off)
    long long slab_bytes = 0;   // L2 slab size for multi-pass segments (0 = whole-array launches)
    bool force_generic = false; // dop_tuning.force_generic: generic kernel for every pass
    bool x_cluster = false;     // the x digits are (16, M) and run as one cluster pass
    bool use_tma = true;        // column passes through the TMA kernels where instantiated (dop_tuning.no_tma)
    int tma_nb = 0, tma_stages = 0; // dop_tuning overrides of their bundle width / pipeline depth (0 = default)
    // schedules for one lambda
    std::vector<dop::PassTmpl> fwd, adj, pre; // pre = Gaussian pre-filter (real -> real)
    long long loss_tiles = 0;                 // CTAs of the MID_LOSS pass
    size_t ws_fields = 0, ws_heff_off = 0, ws_loss_off = 0, ws_xpool_off = 0, ws_coef_off = 0, ws_gfine_off = 0, ws_bytes = 0;
    int up_lg = 0;              // log2(upsample)
    long long ap_ny = 0, ap_nx = 0; // pad = 2: the caller's aperture (desc.ny, desc.nx then hold the 2x window); 0 = no padding
    bool pre_stencil = false;   // the pre-filter runs as a separable spatial stencil (blur.cu) instead of the spectral passes
    int blur_radius = 0;
    std::vector<float> blur_wx, blur_wy; // taps g[0 .. radius] of the two axes
    std::vector<int> hpair_items;  // last y digit: (tile, mirror tile | -1) per work item of the paired (x) H pass; empty = unpaired
    int* d_hpair = nullptr;
    std::vector<double*> d_f2_bl[2]; // band_limit: per-wavelength f^2 tables with the clipped bins set to 1e300
    // device tables (lazy)
    bool dev_ready = false;
    int device = -1;
    void* d_arena = nullptr;
    float2* d_tw = nullptr; // W_L tables then boundary twiddles
    int* d_pi = nullptr;
    double* d_f2[2] = {nullptr, nullptr};
    float* d_g[2] = {nullptr, nullptr};
    std::vector<size_t> pi_off[2];
    int state = 0; // 1 after a successful fwd
    const float* target_seen = nullptr; // DOP_LOSS_SIMSE: the target of the last fwd (adj forms the seed from it)
    // slab schedule: auxiliary streams the slabs of a segment are dealt to, so that the launch tails of
    // one slab overlap the next slab's kernels (fork / join around the segment on the caller's stream)
    int n_aux = 0;
    cudaStream_t aux[4] = {nullptr, nullptr, nullptr, nullptr};
    cudaEvent_t ev_fork = nullptr, ev_join[4] = {nullptr, nullptr, nullptr, nullptr};
    // per-launch profiling (dop_plan_set_profiling)
    bool profiling = false;
    std::vector<cudaEvent_t> ev_start, ev_stop;
    std::vector<std::string> prof_name;
    std::vector<double> prof_bpp;
    size_t prof_n = 0;
};

namespace dop {
dop_status build_plan(dop_plan* p);
std::string describe_plan(const dop_plan* p);
void tile_geometry(const dop_plan* p, int axis, int digit, PassDesc* d);
void pass_geometry(const dop_plan* p, const PassTmpl& t, PassDesc* d, bool allow_tma = true);
} // namespace dop
