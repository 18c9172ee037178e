/*
 * dop.h -- C-ABI boundary of the B200-native angular-spectrum (ASM) propagation library.
 *
 * One data-parallel hot path: scalar ASM free-space propagation of a DOE height map on very
 * large grids (forward), and its adjoint (dL/dI -> dL/dh).  Citations are to
 * /root/reference/PAPER.md (arxiv 2505.22313), section 3.1:
 *
 *   Eq. (1) PAPER.md:95-99    Phi_lambda(x,y) = (2 pi / lambda) (n_lambda - 1) h(x,y)
 *   Eq. (2) PAPER.md:99-102   E_doe = E_in * exp(i Phi)                  (E_in == 1 here)
 *   Eq. (3) PAPER.md:104-108  E_dest = F^-1{ F{E_doe} (x) H_lambda }     (F = 2-D FFT)
 *   Eq. (4) PAPER.md:108-112  I_lambda = |E_dest|^2, objective sum_lambda L_p(I_lambda)
 *   back-propagation: PAPER.md:124; "backward pass is realized by another ... 2-D FFT"
 *   PAPER.md:200 (section 4.1); row-column decomposition of the 2-D FFT PAPER.md:200.
 *
 * Readings where the paper is silent ("Readings"):
 *   H_lambda[ky,kx] = exp(+i 2 pi z sqrt(a)) if a >= 0 else 0,
 *       a = (1/lambda^2 - fx^2) - fy^2, fx = kx/(nx pitch), fy = ky/(ny pitch), signed bins
 *       (BASELINE.json north_star; the paper never writes H out);
 *   forward DFT kernel exp(-2 pi i k n/N) unnormalised, inverse exp(+...) scaled 1/(ny nx);
 *   loss (DOP_LOSS_L2) L = sum_lambda (1/(ny nx)) sum_{y,x} (I_lambda - T)^2;
 *   pre-filter (sigma > 0): h <- Re F^-1{ F{h} exp(-2 pi^2 sigma^2 ((kx/nx)^2+(ky/ny)^2)) }.
 *
 * Conventions
 *   Layout     every plane is row-major [ny][nx], x contiguous; [n_lambda][ny][nx] where noted.
 *   Pointers   "host" or "device" is stated per argument.  The caller owns every device buffer
 *              including the workspace; the plan owns host memory and small device tables
 *              (O(nx + ny) bytes, allocated on the current device at the first propagate call,
 *              freed by dop_plan_destroy).  The library never allocates O(ny nx) memory.
 *   Alignment  device planes must be 16-byte aligned (any cudaMalloc / torch allocation is).
 *   Asynchrony dop_propagate_* only enqueue kernels on `cuda_stream` (a cudaStream_t passed as
 *              void*; NULL = the legacy default stream) and never synchronise it.
 *   State      between dop_propagate_fwd and dop_propagate_adj the workspace holds the
 *              destination field (DOP_LOSS_NONE) or the seeded, partly transformed gradient
 *              field (DOP_LOSS_L2); the caller must not touch it.  dop_propagate_adj without a
 *              preceding successful dop_propagate_fwd on the same plan -> DOP_ERR_STATE.
 *   Errors     every call returns a dop_status; argument / size / state errors are detected
 *              before anything is enqueued.  No exception crosses the boundary, there is no
 *              global state, and there is NO CPU fallback: without an sm_100 device the
 *              propagate calls fail with DOP_ERR_ARCH / DOP_ERR_CUDA.
 *
 * Tuning (dop_tuning, passed explicitly through dop_plan_desc.tuning; NULL = defaults).  The library
 * reads NO environment variable and keeps no global state.  None of the fields changes a result
 * beyond rounding order; tests/ exercises every one of them.
 */
#ifndef DOP_H_
#define DOP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dop_plan dop_plan; /* opaque, host-side */

typedef enum {
    DOP_OK = 0,
    DOP_ERR_INVALID_ARG = 1,      /* NULL where a pointer is required, non-finite / non-positive
                                     pitch or lambda, n_lambda < 1, bad enum, missing buffer     */
    DOP_ERR_UNSUPPORTED_SIZE = 2, /* ny or nx < 2, or with a prime factor above 127              */
    DOP_ERR_WORKSPACE = 3,        /* NULL workspace                                              */
    DOP_ERR_STATE = 4,            /* adj called before fwd                                       */
    DOP_ERR_ARCH = 5,             /* current device is not compute capability 10.x (sm_100)      */
    DOP_ERR_CUDA = 6,             /* a CUDA runtime call or launch failed (cudaGetLastError)     */
    DOP_ERR_NOALLOC_LIMIT = 7     /* dop_prefilter_noalloc: ny * nx > DOP_NOALLOC_MAX_POINTS     */
} dop_status;

typedef enum {
    DOP_LOSS_NONE = 0, /* fwd writes I (and keeps the field); adj takes the caller's dL/dI       */
    DOP_LOSS_L2 = 1,   /* L = sum_lambda mean_xy (I_lambda - T)^2, seeded inside the pass (Eq. 4) */
    DOP_LOSS_SIMSE = 2 /* the paper's penalty, Eq. (6): L = sum_lambda [ L_si-mse +
                          energy_beta L_energy ].  The paper defers both definitions to a supplement
                          that is not available; READING: per wavelength
                          L_si-mse = mean_xy (s I - T)^2 with the least-squares scale s = <I,T>/<I,I>,
                          L_energy = 1 - mean_xy I.  The scale needs <I,T>, <I,I> of the whole plane
                          before the seed, so the row pass around the loss splits in two: fwd ends with
                          "x-inv, store u, plane sums", adj starts with "seed from u, T, s; x-fwd".    */
} dop_loss_mode;

/* element type of the design layout handed in as d_height (gray-level layouts) */
typedef enum {
    DOP_LAYOUT_F32 = 0, /* heights in metres                                                       */
    DOP_LAYOUT_U8 = 1,  /* gray levels, height = level * layout_step                               */
    DOP_LAYOUT_U16 = 2  /* gray levels (e.g. the paper's 10-bit layouts), height = level * step    */
} dop_layout_dtype;

/* flags */
#define DOP_WRITE_INTENSITY 0x1u /* DOP_LOSS_L2 only: also write I to d_intensity                */

/* Optional tuning of the pass schedule (measurement and test aid).  Zero-initialise, then set fields. */
typedef struct {
    int32_t n_xdigits;      /* > 0: force the digit decomposition of the x axis (product must be nx,   */
    int64_t xdigits[4];     /*      every digit within the kernels' limits, else UNSUPPORTED_SIZE)     */
    int32_t n_ydigits;      /* the same for the y axis                                                  */
    int64_t ydigits[4];
    int32_t force_generic;  /* != 0: generic shared-memory kernel for every pass                        */
    int32_t col_nb;         /* 16 | 32 | 64: columns per column-tile bundle (0 = per-pass default)      */
    int32_t prefetch_waves; /* 1..64: inter-CTA L2 prefetch distance in waves; -1 = off; 0 = default 1  */
    int32_t slab_mb;        /* > 0: run multi-pass segments slab by slab    */
    int32_t slab_streams;   /* 1..4 auxiliary streams of the slab schedule (0 = default 2)              */
    int32_t h_float;        /* != 0: take the phase of H through an fp32 fraction, never fixed point    */
    int32_t tile_pts;       /* 256..16384: tile size of the generic kernel (0 = default 4096)           */
    int32_t no_cluster;     /* != 0: never use the thread-block-cluster row kernels (cluster_row.cuh)   */
    int32_t no_mirror;      /* != 0: do not pair mirrored ky tiles in the (x) H pass                    */
    int32_t cluster_dsmem;  /* != 0: the cluster row kernels exchange through distributed shared memory  */
                            /*       instead of through L2 (measured slower on B200; kept as evidence)   */
    int32_t cluster_lines;  /* 1 | 2 | 4 | 8: lines per CTA of the cluster row kernels, i.e. cluster size   */
                            /*       16 / lines (0 = default: 512-thread CTAs)                           */
    int32_t cluster_force;  /* != 0: cluster row kernels wherever they exist (nx = 16384, 32768, 65536);  */
                            /*       by default only where measured faster than two digit passes          */
                            /*       (nx = 16384, clusters of 2; profiles/r02_cluster.md)                 */
    int32_t no_tma;         /* != 0: column passes through the LDG/STG kernels (pow2_impl.cuh) instead of the   */
                            /*       persistent TMA pipeline (tma_col.cuh)                                      */
    int32_t tma_nb;         /* 16 | 32: columns per TMA tile (0 = per-pass default)                              */
    int32_t tma_stages;     /* 1..8: tiles in flight per CTA of the TMA kernels (0 = per-pass default)          */
    int32_t no_stencil;     /* != 0: the Gaussian pre-filter always runs in its spectral form (ten FFT passes)  */
                            /*       instead of the separable spatial stencil used for 2 <= sigma <= 4 px (blur.cu) */
    int32_t no_smooth;      /* != 0: plain passes of the 5-smooth digits 225, 625, 900, 2500 (the paper's 28 800 and     */
                            /*       40 000 grids) through the generic kernel instead of the register-step kernels       */
                            /*       (smooth.cu)                                                                         */
} dop_tuning;

typedef struct {
    int64_t ny, nx;            /* rows, columns; x contiguous; each >= 2, prime factors <= 127:  */
                               /* 2^a 3^b run on the specialised kernels, other factors (the     */
                               /* paper's 28 800 = 2^7 3^2 5^2, 40 000 = 2^6 5^4, 128 640 =      */
                               /* 2^7 3 5 67) as direct odd-prime butterflies  */
    double pitch;              /* metres, same in x and y                                        */
    int32_t n_lambda;          /* >= 1                                                           */
    const double* lambda;      /* [n_lambda] metres, HOST memory, copied by dop_plan_create      */
    const double* n_refr;      /* [n_lambda] refractive index n_lambda (Eq. 1), HOST, copied     */
    double z;                  /* metres, any sign, 0 allowed                                    */
    dop_loss_mode loss;
    double prefilter_sigma_px; /* 0 = off; > 0 = Gaussian spectral pre-filter on h (config 3)    */
    uint32_t flags;            /* DOP_WRITE_INTENSITY                                            */
    const dop_tuning* tuning;  /* HOST, copied; NULL = defaults                                  */
    /* ---- the design loop around the path; all zero = the plain path above ---- */
    double energy_beta;        /* DOP_LOSS_SIMSE: weight of L_energy (paper: 5e-3)                */
    int32_t upsample;          /* r = 0 | 1 (none), 2, 4, 8: super-resolved design variable       */
                               /* (PAPER.md:51, 141, 259-264): d_height is the COARSE layout      */
                               /* [ny/r][nx/r], nearest-neighbour up-sampled r x r inside the     */
                               /* first pass's read; d_grad_height is [ny/r][nx/r], the r x r     */
                               /* sum-pool of dL/dh (deterministic: lanes, then rows)             */
    int32_t layout_dtype;      /* dop_layout_dtype of d_height                                    */
    double layout_step;        /* metres per gray level (U8 / U16 layouts)                        */
    /* ---- linear (non-circular) propagation (PAPER.md:436 Matsushima & Shimobaba 2009) ---- */
    int32_t pad;               /* 0 | 1: the circular operator on the given grid (Eq. 3 as it stands);  */
                               /* 2: the aperture [ny][nx] sits in the corner of a [2 ny][2 nx] window  */
                               /* of zero amplitude, the window is propagated and cropped back.  All    */
                               /* caller planes keep their [ny][nx] shape; the workspace holds the      */
                               /* window; rows known to be zero / discarded are pruned from the x       */
                               /* passes.  DOP_LOSS_L2 / DOP_LOSS_NONE, no pre-filter, fp32 layout.     */
    int32_t band_limit;        /* != 0 (needs pad = 2): H is clipped to |fx| <= u_limit, |fy| <= v_limit, */
                               /* u_limit = 1 / (lambda sqrt((2 du z)^2 + 1)), du = 1 / (2 nx pitch)      */
} dop_plan_desc;

/* Adam with a cosine learning-rate schedule (Kingma & Ba 2014, Algorithm 1), applied
 * to the design layout as a pointwise epilogue of the adjoint pass. */
typedef struct {
    double lr0;          /* initial learning rate, in the unit of the layout (metres)                */
    double beta1, beta2; /* 0.9, 0.999                                                                */
    double eps;          /* in the unit of the gradient                                              */
    int64_t iter;        /* 0-based iteration: lr = lr0 (1 + cos(pi iter/total_iters))/2, t = iter+1 */
    int64_t total_iters; /* the schedule reaches zero here (paper: 3000)                             */
} dop_adam;

/*
 * Build a plan (host-only work: validation, factorisation of ny and nx into radix-2/3/4 digit
 * passes, twiddle / frequency tables in fp64, pass schedule).  Touches no GPU.
 *   out              receives the plan (host pointer).
 *   workspace_bytes  (may be NULL) receives the size of the device workspace the caller must
 *                    pass to the propagate calls: n_lambda complex64 fields + (pre-filter on)
 *                    one fp32 plane + loss-reduction scratch.
 * Errors: DOP_ERR_INVALID_ARG, DOP_ERR_UNSUPPORTED_SIZE.
 */
dop_status dop_plan_create(dop_plan** out, const dop_plan_desc* d, size_t* workspace_bytes);

/*
 * Forward pass, Eq. (1)-(4): for every lambda  h -> Phi -> u0 = exp(i Phi) -> F -> (x) H ->
 * F^-1 -> I = |u|^2 [-> L2 loss and the seed g_u = 2 (dL/dI) u of the adjoint, DOP_LOSS_L2].
 *   d_height     the design layout, DEVICE, read-only: [ny][nx] fp32 metres, or with upsample = r
 *                the coarse [ny/r][nx/r] layout of layout_dtype (gray levels times layout_step).
 *   d_target     [ny][nx] fp32 DEVICE (shared by all lambda); required for DOP_LOSS_L2 and
 *                DOP_LOSS_SIMSE, ignored (may be NULL) for DOP_LOSS_NONE.  DOP_LOSS_SIMSE: the seed
 *                is formed from it inside dop_propagate_adj, so the buffer must stay valid and
 *                unchanged until that call has been enqueued and executed.
 *   d_intensity  [n_lambda][ny][nx] fp32 DEVICE; required for DOP_LOSS_NONE and for
 *                DOP_LOSS_L2 with DOP_WRITE_INTENSITY; otherwise ignored (may be NULL).
 *   d_loss       DEVICE double scalar or NULL; DOP_LOSS_L2 / DOP_LOSS_SIMSE: receives L when the
 *                stream reaches that point.  Ignored for DOP_LOSS_NONE.
 *   d_workspace  DEVICE, workspace_bytes from dop_plan_create, 256-byte aligned.
 *                After a DOP_LOSS_NONE forward its first n_lambda*ny*nx complex64 (interleaved
 *                re, im) hold the destination field u of Eq. (3), natural order.
 *   cuda_stream  cudaStream_t.
 */
dop_status dop_propagate_fwd(dop_plan* plan, const void* d_height, const float* d_target,
                             float* d_intensity, double* d_loss, void* d_workspace,
                             void* cuda_stream);

/*
 * Adjoint pass: dL/dI -> g_u = 2 (dL/dI) u -> F -> (x) conj(H) -> F^-1 ->
 * dL/dh = sum_lambda (2 pi (n_lambda-1)/lambda) Im( conj(u0) g_u0 )  [-> pre-filter adjoint].
 *   d_height       the same buffer that was given to dop_propagate_fwd (u0 is recomputed).
 *   d_dLdI         [n_lambda][ny][nx] fp32 DEVICE; required for DOP_LOSS_NONE, ignored for
 *                  DOP_LOSS_L2 (the seed was formed inside the forward pass).
 *   d_grad_height  [ny][nx] fp32 DEVICE, overwritten with dL/dh.
 */
dop_status dop_propagate_adj(dop_plan* plan, const void* d_height, const float* d_dLdI,
                             float* d_grad_height, void* d_workspace, void* cuda_stream);

/*
 * The adjoint pass with the Adam update of the design layout fused into its last store (no up-sampling,
 * no pre-filter: the A5 store of the last wavelength) or into the final row-pooling kernel (up-sampling),
 * else run as one pointwise kernel after the pre-filter adjoint.
 *   d_layout       the fp32 design layout (DOP_LAYOUT_F32 only), the buffer that was given to
 *                  dop_propagate_fwd; UPDATED IN PLACE: l <- l - lr m_hat / (sqrt(v_hat) + eps).
 *   d_grad_height  dL/dl, same shape as the layout; may be NULL when only the update is wanted.
 *   d_m, d_v       Adam's first / second moment, fp32, same shape as the layout, caller-owned,
 *                  zero before the first iteration; updated in place.
 *   hp             HOST, read during the call.
 * Errors as dop_propagate_adj; DOP_ERR_INVALID_ARG for a non-fp32 layout or bad hyper-parameters.
 */
dop_status dop_propagate_adj_adam(dop_plan* plan, float* d_layout, const float* d_dLdI, float* d_grad_height,
                                  float* d_m, float* d_v, const dop_adam* hp, void* d_workspace,
                                  void* cuda_stream);

/*
 * The Gaussian pre-filter F0 / A6 (the blur of the MTF model PAPER.md:184, standing in for G{l} of Eq. 5
 * PAPER.md:114-122; F0) for callers that cannot allocate: code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc.  It is the stencil form of the pre-filter that dop_propagate_fwd /
 * dop_propagate_adj run (rows into a scratch plane, columns out of it), except that the scratch plane is a static
 * device array inside the library (DOP_NOALLOC_MAX_POINTS floats = 16 MiB, held by every GPU that loads the
 * library until the process exits) instead of the caller's workspace, and that it needs no device tables of the
 * plan.  The call reaches no cudaMalloc, cudaFree or allocating library routine, on its first use or later.
 *   plan         a plan whose pre-filter runs as a stencil: prefilter_sigma_px in [2.05, 4], fp32 layout without
 *                up-sampling, nx % 8 == 0, ny % 32 == 0, no tuning.no_stencil / force_generic; only its HOST side
 *                is read (shape and taps), so it may be a plan that never ran, on any device.
 *                Anything else -> DOP_ERR_INVALID_ARG.
 *   d_in         [ny][nx] fp32 DEVICE (current device), read-only: h (F0) or dL/dh_eff (A6; the filter is even).
 *   d_out        [ny][nx] fp32 DEVICE, overwritten; may be d_in itself, must not overlap it otherwise.
 *   cuda_stream  cudaStream_t; the two kernels are enqueued on it, nothing is synchronised.
 * Limit: ny * nx <= DOP_NOALLOC_MAX_POINTS, else DOP_ERR_NOALLOC_LIMIT (nothing is enqueued).
 * Sharing: all calls on a device use the one array, which keeps the previous call's contents; none of it has to
 * start at zero (the row kernel overwrites every element the column kernel reads), so nothing is cleared.  Calls
 * that OVERLAP on the GPU -- two streams, or graph branches with no edge between them -- race on it; order them.
 * The first call on a device looks the array's address up (cudaGetSymbolAddress) and loads the two kernels; make
 * that call outside stream capture.  Errors: DOP_ERR_ARCH off sm_100, DOP_ERR_CUDA.
 */
#define DOP_NOALLOC_MAX_POINTS (4 * 1024 * 1024)
dop_status dop_prefilter_noalloc(const dop_plan* plan, const float* d_in, float* d_out, void* cuda_stream);

/* Frees the plan's host memory and device tables.  NULL -> DOP_ERR_INVALID_ARG. */
dop_status dop_plan_destroy(dop_plan* plan);

/* Static string for a status code (never NULL). */
const char* dop_status_string(dop_status s);

/*
 * Introspection (host only): writes a NUL-terminated, line-oriented description of the pass
 * schedule (one line per kernel launch of one lambda's forward+adjoint, with digit lengths,
 * tile shapes and algorithmic HBM bytes per point) into buf[0..len).  Returns the number of
 * bytes the full text needs (excluding the NUL); output is truncated to len-1 bytes.
 */
size_t dop_plan_describe(const dop_plan* plan, char* buf, size_t len);

/* Number of kernel launches one dop_propagate_fwd + dop_propagate_adj pair enqueues. */
int64_t dop_plan_launch_count(const dop_plan* plan);

/*
 * Per-launch timing (measurement aid for bench.py's roofline line; off by default).
 * dop_plan_set_profiling(plan, 1): every later dop_propagate_fwd/adj records one CUDA event
 * pair around each kernel it enqueues, on the caller's stream (events are owned by the plan;
 * the slots restart at every dop_propagate_fwd).  dop_plan_get_pass_times synchronises those
 * events and writes, for launch i of the last fwd(+adj): ms[i] = its device time in
 * milliseconds and bytes_per_point[i] = its algorithmic HBM bytes per grid point (either array
 * may be NULL); returns the number of recorded launches (<= n are written).
 * dop_plan_pass_name(plan, i): static-lifetime-of-plan name of recorded launch i, or "".
 */
dop_status dop_plan_set_profiling(dop_plan* plan, int enable);
int64_t dop_plan_get_pass_times(dop_plan* plan, float* ms, double* bytes_per_point, int64_t n);
const char* dop_plan_pass_name(const dop_plan* plan, int64_t i);

#ifdef __cplusplus
}
#endif
#endif /* DOP_H_ */
