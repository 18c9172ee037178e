// api.cu -- the C-ABI entry points declared in include/dop.h: validation, lazy upload of the
// plan's small device tables, and the enqueueing of the pass schedule.  No torch types, no
// synchronisation, no CPU fallback.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "dop_internal.h"

namespace dop {
cudaError_t launch_tile_pass_generic(const PassDesc& p, cudaStream_t stream);
cudaError_t launch_tile_pass_pow2(const PassDesc& p, cudaStream_t stream, bool* handled);
cudaError_t launch_tile_pass_smooth(const PassDesc& p, cudaStream_t stream, bool* handled);

cudaError_t launch_tile_pass(const PassDesc& p, cudaStream_t stream)
{
    {
        bool handled = false;
        cudaError_t e = launch_tile_pass_pow2(p, stream, &handled);
        if (handled) return e;
        e = launch_tile_pass_smooth(p, stream, &handled);
        if (handled) return e;
    }
    return launch_tile_pass_generic(p, stream);
}
} // namespace dop

using namespace dop;

namespace {

size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

struct Buffers {
    const void* height = nullptr;  // what LD_HEIGHT / ST_GRAD read: the caller's layout, or the fine fp32 h_eff plane
    bool height_is_layout = false; // -> plan's up-sampling factor and layout dtype apply to `height`
    const float* target = nullptr;
    float* intensity = nullptr;
    const float* dLdI = nullptr;
    float* grad = nullptr;         // where ST_GRAD writes: a fine plane, or (grad_pool) the x-pooled plane
    bool grad_pool = false;
    const void* real_src = nullptr;
    bool real_src_is_layout = false;
    float* real_dst = nullptr;
    bool real_dst_pool = false;
    const AdamParams* adam = nullptr; // fused into the ST_GRAD store of the last wavelength
    float* adam_m = nullptr;
    float* adam_v = nullptr;
    float* adam_h = nullptr;
};

dop_status ensure_device(dop_plan* p)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return DOP_ERR_CUDA;
    if (p->dev_ready && p->device == dev) return DOP_OK;
    if (p->dev_ready) return DOP_ERR_INVALID_ARG; // a plan is bound to the device of its first use
    int major = 0;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) return DOP_ERR_CUDA;
    if (major != 10) return DOP_ERR_ARCH;

    // arena layout: W_L tables | boundary twiddles | pi tables | f2 x,y | g x,y
    size_t off = 0;
    p->wl_off.resize(p->wl_tables.size());
    for (size_t i = 0; i < p->wl_tables.size(); ++i) { p->wl_off[i] = off; off += align256(p->wl_tables[i].size() * sizeof(float2)); }
    for (int a = 0; a < 2; ++a)
        for (Digit& g : p->ax[a].dig)
            if (g.has_twb) { g.twb_off = off; off += align256(g.twb.size() * sizeof(float2)); }
    for (int a = 0; a < 2; ++a)
        for (Digit& g : p->ax[a].dig)
            if (g.fast) { g.twg_off = off; off += align256(g.twg.size() * sizeof(float2)); }
    for (int a = 0; a < 2; ++a)
        for (Digit& g : p->ax[a].dig)
            if (!g.twb2.empty()) { g.twb2_off = off; off += align256(g.twb2.size() * sizeof(float2)); }
    for (int a = 0; a < 2; ++a) {
        p->pi_off[a].resize(p->ax[a].dig.size());
        for (size_t j = 0; j < p->ax[a].dig.size(); ++j) { p->pi_off[a][j] = off; off += align256(p->ax[a].dig[j].pi.size() * sizeof(int)); }
    }
    const size_t hpair_off = off;
    off += align256(p->hpair_items.size() * sizeof(int));
    size_t f2_off[2], g_off[2];
    for (int a = 0; a < 2; ++a) { f2_off[a] = off; off += align256(p->ax[a].f2.size() * sizeof(double)); }
    std::vector<size_t> bl_off[2];
    if (p->desc.band_limit)
        for (int a = 0; a < 2; ++a)
            for (int l = 0; l < p->desc.n_lambda; ++l) { bl_off[a].push_back(off); off += align256(p->ax[a].f2.size() * sizeof(double)); }
    for (int a = 0; a < 2; ++a) { g_off[a] = off; off += align256(p->ax[a].g.size() * sizeof(float)); }

    char* arena = nullptr;
    if (cudaMalloc((void**)&arena, off) != cudaSuccess) return DOP_ERR_CUDA;
    p->d_arena = arena;
    bool ok = true;
    auto up = [&](size_t o, const void* src, size_t bytes) {
        if (bytes && cudaMemcpy(arena + o, src, bytes, cudaMemcpyHostToDevice) != cudaSuccess) ok = false;
    };
    for (size_t i = 0; i < p->wl_tables.size(); ++i) up(p->wl_off[i], p->wl_tables[i].data(), p->wl_tables[i].size() * sizeof(float2));
    for (int a = 0; a < 2; ++a)
        for (Digit& g : p->ax[a].dig)
            if (g.has_twb) up(g.twb_off, g.twb.data(), g.twb.size() * sizeof(float2));
    for (int a = 0; a < 2; ++a)
        for (Digit& g : p->ax[a].dig)
            if (g.fast) up(g.twg_off, g.twg.data(), g.twg.size() * sizeof(float2));
    for (int a = 0; a < 2; ++a)
        for (Digit& g : p->ax[a].dig)
            if (!g.twb2.empty()) up(g.twb2_off, g.twb2.data(), g.twb2.size() * sizeof(float2));
    for (int a = 0; a < 2; ++a)
        for (size_t j = 0; j < p->ax[a].dig.size(); ++j) up(p->pi_off[a][j], p->ax[a].dig[j].pi.data(), p->ax[a].dig[j].pi.size() * sizeof(int));
    up(hpair_off, p->hpair_items.data(), p->hpair_items.size() * sizeof(int));
    p->d_hpair = p->hpair_items.empty() ? nullptr : (int*)(arena + hpair_off);
    for (int a = 0; a < 2; ++a) {
        up(f2_off[a], p->ax[a].f2.data(), p->ax[a].f2.size() * sizeof(double));
        up(g_off[a], p->ax[a].g.data(), p->ax[a].g.size() * sizeof(float));
        p->d_f2[a] = (double*)(arena + f2_off[a]);
        if (p->desc.band_limit) { // H clipped to |f| <= 1 / (lambda sqrt((2 df z)^2 + 1)), df = 1 / (N pitch) of the window
            p->d_f2_bl[a].clear();
            for (int l = 0; l < p->desc.n_lambda; ++l) {
                const double lam = p->lambda[(size_t)l], df = 1.0 / (2.0 * (double)(a == 0 ? p->ap_nx : p->ap_ny) * p->desc.pitch);
                const double lim = 1.0 / (lam * std::sqrt((2.0 * df * p->desc.z) * (2.0 * df * p->desc.z) + 1.0));
                std::vector<double> t = p->ax[a].f2;
                for (size_t sl = 0; sl < t.size(); ++sl)
                    if (std::fabs(p->ax[a].fsigned[sl]) > lim) t[sl] = 1e300; // a < 0: zeroed like an evanescent bin
                up(bl_off[a][(size_t)l], t.data(), t.size() * sizeof(double));
                p->d_f2_bl[a].push_back((double*)(arena + bl_off[a][(size_t)l]));
            }
        }
        p->d_g[a] = (float*)(arena + g_off[a]);
    }
    if (!ok) { cudaFree(arena); p->d_arena = nullptr; return DOP_ERR_CUDA; }
    p->device = dev;
    p->dev_ready = true;
    return DOP_OK;
}

// Resolve one scheduled pass for wavelength `lam` into launch parameters.
PassDesc resolve(const dop_plan* p, const PassTmpl& t, int lam, const Buffers& b, char* ws)
{
    PassDesc d{};
    // (the TMA kernels implement neither the dL/dh accumulate of later wavelengths nor the fused Adam store)
    const bool tma_ok = !(t.store_op == ST_GRAD && (lam > 0 || (b.adam != nullptr && lam == p->desc.n_lambda - 1) || b.grad_pool));
    pass_geometry(p, t, &d, tma_ok);
    // (a cluster pass takes its group twiddles from x digit 1 and its boundary twiddles from x digit 0)
    const Digit& g = p->ax[t.axis].dig[(size_t)(t.cluster ? 1 : t.digit)];
    char* arena = (char*)p->d_arena;
    const size_t npts = (size_t)p->desc.nx * (size_t)p->desc.ny;                           // field window
    const size_t nap = p->ap_nx > 0 ? (size_t)p->ap_nx * (size_t)p->ap_ny : npts;          // caller planes
    d.fft1_dir = t.fft1_dir;
    d.fft2_dir = t.fft2_dir;
    d.wL = (const float2*)(arena + p->wl_off[(size_t)g.wl_index]);
    d.pi = (const int*)(arena + p->pi_off[t.axis][(size_t)t.digit]);
    d.tw_b = g.has_twb ? (const float2*)(arena + g.twb_off) : nullptr;
    d.tw_b2 = g.twb2.empty() ? nullptr : (const float2*)(arena + g.twb2_off);
    d.twb_n = g.L * g.st;
    if (t.cluster) {
        const Digit& g0 = p->ax[0].dig[0];
        d.tw_b = nullptr;
        d.tw_b2 = (const float2*)(arena + g0.twb2_off);
        d.twb_n = g0.L * g0.st;
    }
    d.tw_g = g.fast ? (const float2*)(arena + g.twg_off) : nullptr;
    d.load_op = t.load_op;
    d.mid_op = t.mid_op;
    d.store_op = t.store_op;
    d.field = (float2*)(ws + align256(npts * sizeof(float2)) * (size_t)lam);
    d.height = (const float*)b.height;
    d.write_intensity = 0;
    d.cnx = p->desc.nx >> p->up_lg;
    d.lpr = (d.col_type || d.cluster) ? 0 : p->desc.nx / d.L;
    d.h_step = (float)p->desc.layout_step;
    const bool hl = (t.load_op == LD_HEIGHT || t.store_op == ST_GRAD) && b.height_is_layout;
    if (hl) { d.up_lg = p->up_lg; d.h_dtype = (int)p->desc.layout_dtype; }
    if (t.load_op == LD_SEED) d.plane_in = b.dLdI + nap * (size_t)lam;
    if (t.load_op == LD_SEED_SIMSE) {
        d.plane_in = b.target;
        d.coef = (const float*)(ws + p->ws_coef_off) + 4 * (size_t)lam;
    }
    if (t.load_op == LD_REAL) {
        d.plane_in = (const float*)b.real_src;
        if (b.real_src_is_layout && (p->up_lg > 0 || p->desc.layout_dtype != DOP_LAYOUT_F32)) {
            d.coarse_in = 1;
            d.up_lg = p->up_lg;
            d.h_dtype = (int)p->desc.layout_dtype;
        }
    }
    if (t.store_op == ST_C64_STATS) {
        d.plane_in = b.target;
        d.loss_scratch = (double*)(ws + p->ws_loss_off) + 4 * (size_t)p->loss_tiles * (size_t)lam;
        if (p->desc.flags & DOP_WRITE_INTENSITY) {
            d.write_intensity = 1;
            d.plane_out = b.intensity + nap * (size_t)lam;
        }
    }
    if (t.mid_op == MID_LOSS) {
        d.plane_in = b.target;
        d.loss_scratch = (double*)(ws + p->ws_loss_off) + (size_t)p->loss_tiles * (size_t)lam;
        if (p->desc.flags & DOP_WRITE_INTENSITY) {
            d.write_intensity = 1;
            d.plane_out = b.intensity + nap * (size_t)lam;
        }
    }
    if (t.store_op == ST_GRAD) {
        d.plane_out = b.grad;
        if (lam > 0) d.store_op = ST_GRAD_ACC;
        if (b.grad_pool) { d.pool_out = 1; d.up_lg = p->up_lg; }
        if (b.adam != nullptr && lam == p->desc.n_lambda - 1) {
            d.adam_m = b.adam_m; d.adam_v = b.adam_v; d.adam_h = b.adam_h;
            d.adam_b1 = b.adam->b1; d.adam_b2 = b.adam->b2; d.adam_c1 = b.adam->c1; d.adam_c2 = b.adam->c2;
            d.adam_a1 = b.adam->a1; d.adam_rb2 = b.adam->rb2;
            d.adam_eps = b.adam->eps;
        }
    }
    if (t.store_op == ST_C64_INTENSITY) d.plane_out = b.intensity + nap * (size_t)lam;
    if (t.store_op == ST_REAL) {
        d.plane_out = b.real_dst;
        if (b.real_dst_pool) { d.pool_out = 1; d.up_lg = p->up_lg; }
    }
    const double lambda = p->lambda[(size_t)lam], n = p->n_refr[(size_t)lam];
    d.phase_coef = (float)((n - 1.0) / lambda);
    d.grad_coef = (float)(2.0 * M_PI * (n - 1.0) / lambda);
    d.scale = (float)(1.0 / (double)npts);
    d.seed_coef = (float)(4.0 / (double)nap);
    if (p->ap_nx > 0 && t.axis == 0) { d.ap_nx = p->ap_nx; d.ap_ny = p->ap_ny; d.grid_nx = p->desc.nx; }
    // pad = 2: a pass that touches the caller's planes masks them to the aperture -- in the TMA kernels (tile maps of
    // the aperture's shape) or in the generic kernel; it must never reach the LDG/STG kernels, which do not
    if (d.ap_nx > 0 && d.tma == 0 && (t.load_op != LD_C64 || t.store_op != ST_C64 || t.mid_op == MID_LOSS)) d.tw_g = nullptr;
    if (d.ap_nx > 0 && d.tma > 0 && (d.n_m != 1 || p->ap_nx % 4 != 0)) { d.tma = 0; d.tw_g = nullptr; pass_geometry(p, t, &d, false); d.tw_g = nullptr; }
    d.inv_lam2 = 1.0 / (lambda * lambda);
    d.z = p->desc.z;
    d.h_fixed = (std::fabs(p->desc.z) / lambda < 524288.0 && !p->h_float) ? 1 : 0;
    {
        const double sc = 1.0 / (double)npts, tp = 2.0 * M_PI;
        const double sk[5] = {tp, -tp * tp * tp / 6.0, std::pow(tp, 5) / 120.0, -std::pow(tp, 7) / 5040.0, std::pow(tp, 9) / 362880.0};
        const double ck[5] = {1.0, -tp * tp / 2.0, std::pow(tp, 4) / 24.0, -std::pow(tp, 6) / 720.0, std::pow(tp, 8) / 40320.0};
        for (int q = 0; q < 5; ++q) { d.hk_s[q] = (float)(sc * sk[q]); d.hk_c[q] = (float)(sc * ck[q]); }
    }
    // prefetch distance in tiles: pf_waves x (148 SMs x resident CTAs of ~1024 threads per SM)
    {
        const long long threads = d.cluster ? 512 : (d.col_type ? d.L : (long long)d.nl * d.L / 16);
        const long long per_sm = threads > 0 ? (1024 / threads > 0 ? 1024 / threads : 1) : 1;
        d.pf_ahead = (int)(p->pf_waves * 148 * per_sm);
        // Measured (C2 / C3 / C4): a gain on row-type tiles (C3 x passes 0.86 -> 0.75 ms, C2 loss pass
        // 0.57 -> 0.52 ms); on column tiles a loss, or a wash that over-fetches DRAM by 15-50 %
        // (ncu) -- with 32-column bundles the C2 y passes run 0.217 ms with it and 0.204 ms without.
        if (d.col_type || d.cluster) d.pf_ahead = 0;
    }
    d.device = p->device;
    if ((t.mid_op == MID_H || t.mid_op == MID_HCONJ) && d.tma > 0 && p->d_hpair != nullptr && d.n_m == 1 && d.cg0 == 0 && d.o0 == 0) {
        d.hpair = p->d_hpair;
        d.n_hpair = (int)(p->hpair_items.size() / 2);
    }
    d.fx2 = p->d_f2[0];
    d.fy2 = p->d_f2[1];
    if (p->desc.band_limit) { d.fx2 = p->d_f2_bl[0][(size_t)lam]; d.fy2 = p->d_f2_bl[1][(size_t)lam]; }
    d.gx = p->d_g[0];
    d.gy = p->d_g[1];
    return d;
}

// profiling slot for the next launch: records the start event, returns the slot (or -1)
long long prof_begin(dop_plan* p, const std::string& name, double bpp, cudaStream_t st)
{
    if (!p->profiling) return -1;
    const size_t i = p->prof_n++;
    if (i >= p->ev_start.size()) {
        cudaEvent_t a = nullptr, b = nullptr;
        if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) { p->prof_n--; return -1; }
        p->ev_start.push_back(a);
        p->ev_stop.push_back(b);
        p->prof_name.emplace_back();
        p->prof_bpp.push_back(0.0);
    }
    p->prof_name[i] = name;
    p->prof_bpp[i] = bpp;
    cudaEventRecord(p->ev_start[i], st);
    return (long long)i;
}
void prof_end(dop_plan* p, long long slot, cudaStream_t st)
{
    if (slot >= 0) cudaEventRecord(p->ev_stop[(size_t)slot], st);
}

// pad = 2: rows [ap_ny, 2 ap_ny) of wavelength lam's window are known zeros (forward) / discarded (adjoint): the x
// passes are launched on the aperture rows only and those rows are cleared instead (a write, no read, no DFT)
bool zero_pruned_rows(const dop_plan* p, char* ws, int lam, cudaStream_t st)
{
    if (p->ap_nx == 0) return true;
    const size_t npts = (size_t)p->desc.nx * (size_t)p->desc.ny;
    char* field = ws + align256(npts * sizeof(float2)) * (size_t)lam;
    const size_t row = (size_t)p->desc.nx * sizeof(float2);
    return cudaMemsetAsync(field + (size_t)p->ap_ny * row, 0, (size_t)(p->desc.ny - p->ap_ny) * row, st) == cudaSuccess;
}

// the Gaussian pre-filter as two stencil passes (blur.cu), one profiling slot each
dop_status run_stencil(dop_plan* p, const float* src, float* tmp, float* dst, cudaStream_t st, const char* tag)
{
    long long s0 = prof_begin(p, std::string(tag) + ":blur-x", 8.0, st);
    long long s1 = -1;
    cudaEvent_t mid_stop = s0 >= 0 ? p->ev_stop[(size_t)s0] : nullptr, mid_start = nullptr;
    if (p->profiling) {
        s1 = prof_begin(p, std::string(tag) + ":blur-y", 8.0, st); // (its start event is re-recorded between the kernels)
        if (s1 >= 0) mid_start = p->ev_start[(size_t)s1];
    }
    cudaError_t e = launch_blur(src, tmp, dst, p->desc.ny, p->desc.nx, p->blur_radius, p->blur_wx.data(), p->blur_wy.data(), st,
                                mid_stop, mid_start);
    if (s1 >= 0) prof_end(p, s1, st);
    return e == cudaSuccess ? DOP_OK : DOP_ERR_CUDA;
}

long long gcdll(long long a, long long b) { while (b) { long long t = a % b; a = b; b = t; } return a; }
long long lcmll(long long a, long long b) { return a / gcdll(a, b) * b; }


// Slab unit (columns for y segments, rows for x segments) and slab size of a segment; false when the
// segment runs as whole-array launches.
template <class D>
bool slab_layout(const dop_plan* p, const std::vector<D>& d, int axis, long long* total, long long* per)
{
    const long long nx = p->desc.nx, ny = p->desc.ny;
    *total = axis == 1 ? nx : ny;
    *per = *total;
    if (!(p->slab_bytes > 0 && d.size() >= 2)) return false;
    long long unit = 1;
    for (const D& q : d) {
        if (axis == 1) unit = lcmll(unit, q.nl);
        else if (!q.col_type) {
            const long long lpr = nx / q.L; // lines per row
            if (q.nl > lpr) unit = lcmll(unit, (q.nl + lpr - 1) / lpr);
        }
    }
    const long long group_bytes = (axis == 1 ? ny : nx) * (long long)sizeof(float2);
    *per = p->slab_bytes / group_bytes / unit * unit;
    if (*per < unit) *per = unit;
    if (*per >= *total) { *per = *total; return false; }
    return true;
}

std::string pass_label(const char* tag, const PassTmpl& t)
{
    if (t.cluster) return std::string(tag) + ":x0+x1:" + t.name;
    return std::string(tag) + ":" + (t.axis == 0 ? "x" : "y") + std::to_string(t.digit) + ":" + t.name;
}

// One segment = consecutive passes along the same axis.  Its passes exchange data only inside
// independent groups (y passes: inside a column group; x passes: inside a row), so the segment
// is run slab by slab -- a slab being a set of whole groups of about slab_bytes -- and every pass
// after the first finds its input in L2.
dop_status run_segment(dop_plan* p, const std::vector<PassTmpl>& sched, size_t b, size_t e, int lam,
                       const Buffers& bufs, char* ws, cudaStream_t st, const char* tag)
{
    const long long nx = p->desc.nx, ny = p->desc.ny;
    const int axis = sched[b].axis;
    std::vector<PassDesc> d;
    for (size_t i = b; i < e; ++i) d.push_back(resolve(p, sched[i], lam, bufs, ws));
    long long total = 0, per = 0;
    const bool slabbed = slab_layout(p, d, axis, &total, &per);
    if (!slabbed) { // whole-array launches, one profiling slot per launch
        for (size_t i = b; i < e; ++i) {
            // (the dL/dh accumulate of every wavelength after the first re-reads grad: +4 B/point)
            const double bpp = sched[i].bytes_per_point + ((lam > 0 && sched[i].store_op == ST_GRAD) ? 4.0 : 0.0);
            long long slot = prof_begin(p, pass_label(tag, sched[i]), bpp, st);
            cudaError_t er = launch_tile_pass(d[i - b], st);
            prof_end(p, slot, st);
            if (er != cudaSuccess) return DOP_ERR_CUDA;
        }
        return DOP_OK;
    }
    // lazily create the auxiliary streams (DOP_SLAB_STREAMS, default 2)
    if (p->n_aux == 0) {
        const int ns = p->slab_streams;
        if (cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming) != cudaSuccess) return DOP_ERR_CUDA;
        for (int k = 0; k < ns; ++k) {
            if (cudaStreamCreateWithFlags(&p->aux[k], cudaStreamNonBlocking) != cudaSuccess) return DOP_ERR_CUDA;
            if (cudaEventCreateWithFlags(&p->ev_join[k], cudaEventDisableTiming) != cudaSuccess) return DOP_ERR_CUDA;
        }
        p->n_aux = ns;
    }
    std::string name = std::string(tag) + ":" + (axis == 0 ? "x" : "y") + "-seg[";
    double dram = sched[b].rd + sched[e - 1].wr;
    for (size_t i = b; i < e; ++i) {
        name += (i > b ? " | " : "") + sched[i].name;
        dram += sched[i].side;
    }
    name += "]";
    long long slot = prof_begin(p, name, dram, st);
    if (cudaEventRecord(p->ev_fork, st) != cudaSuccess) return DOP_ERR_CUDA;
    for (int k = 0; k < p->n_aux; ++k)
        if (cudaStreamWaitEvent(p->aux[k], p->ev_fork, 0) != cudaSuccess) return DOP_ERR_CUDA;
    long long slab_index = 0;
    for (long long g0 = 0; g0 < total; g0 += per, ++slab_index) {
        cudaStream_t ss = p->aux[slab_index % p->n_aux];
        const long long g1 = g0 + per < total ? g0 + per : total;
        for (PassDesc q : d) {
            if (axis == 1) { // columns [g0, g1)
                q.cg0 = g0 / q.nl;
                q.n_cgroups = (g1 - g0 + q.nl - 1) / q.nl;
            } else if (q.col_type) { // rows [g0, g1)
                q.tile0 = g0 * q.n_m * q.n_cgroups;
                q.o0 = g0;
                q.n_o = g1 - g0;
            } else {
                const long long lpr = nx / q.L;
                q.cg0 = g0 * lpr / q.nl;
                q.n_cgroups = ((g1 - g0) * lpr + q.nl - 1) / q.nl;
                q.tile0 = q.cg0;
            }
            if (launch_tile_pass(q, ss) != cudaSuccess) return DOP_ERR_CUDA;
        }
    }
    for (int k = 0; k < p->n_aux; ++k) {
        if (cudaEventRecord(p->ev_join[k], p->aux[k]) != cudaSuccess) return DOP_ERR_CUDA;
        if (cudaStreamWaitEvent(st, p->ev_join[k], 0) != cudaSuccess) return DOP_ERR_CUDA;
    }
    prof_end(p, slot, st);
    return DOP_OK;
}

dop_status run(dop_plan* p, const std::vector<PassTmpl>& sched, int lam, const Buffers& b, char* ws,
               cudaStream_t st, const char* tag)
{
    size_t i = 0;
    while (i < sched.size()) {
        size_t j = i + 1;
        while (j < sched.size() && sched[j].axis == sched[i].axis) ++j;
        dop_status s = run_segment(p, sched, i, j, lam, b, ws, st, tag);
        if (s != DOP_OK) return s;
        i = j;
    }
    return DOP_OK;
}

} // namespace

extern "C" {

dop_status dop_plan_create(dop_plan** out, const dop_plan_desc* d, size_t* workspace_bytes)
{
    if (out == nullptr) return DOP_ERR_INVALID_ARG;
    *out = nullptr;
    if (d == nullptr || d->lambda == nullptr || d->n_refr == nullptr) return DOP_ERR_INVALID_ARG;
    if (d->n_lambda < 1 || d->n_lambda > 4096) return DOP_ERR_INVALID_ARG;
    if (!(d->pitch > 0.0) || !std::isfinite(d->pitch) || !std::isfinite(d->z)) return DOP_ERR_INVALID_ARG;
    if (!(d->prefilter_sigma_px >= 0.0) || !std::isfinite(d->prefilter_sigma_px)) return DOP_ERR_INVALID_ARG;
    if (d->loss != DOP_LOSS_NONE && d->loss != DOP_LOSS_L2 && d->loss != DOP_LOSS_SIMSE) return DOP_ERR_INVALID_ARG;
    if (d->flags & ~DOP_WRITE_INTENSITY) return DOP_ERR_INVALID_ARG;
    for (int i = 0; i < d->n_lambda; ++i) {
        if (!(d->lambda[i] > 0.0) || !std::isfinite(d->lambda[i])) return DOP_ERR_INVALID_ARG;
        if (!std::isfinite(d->n_refr[i])) return DOP_ERR_INVALID_ARG;
    }
    if (d->ny < 2 || d->nx < 2) return DOP_ERR_UNSUPPORTED_SIZE;
    if (d->pad != 0 && d->pad != 1 && d->pad != 2) return DOP_ERR_INVALID_ARG;
    if (d->pad == 2 && (d->loss == DOP_LOSS_SIMSE || d->prefilter_sigma_px > 0.0 || (d->upsample != 0 && d->upsample != 1) ||
                        d->layout_dtype != DOP_LAYOUT_F32))
        return DOP_ERR_INVALID_ARG;
    if (d->band_limit != 0 && d->pad != 2) return DOP_ERR_INVALID_ARG;
    dop_plan* p = new (std::nothrow) dop_plan();
    if (p == nullptr) return DOP_ERR_INVALID_ARG;
    p->desc = *d;
    p->lambda.assign(d->lambda, d->lambda + d->n_lambda);
    p->n_refr.assign(d->n_refr, d->n_refr + d->n_lambda);
    p->desc.lambda = p->lambda.data();
    p->desc.n_refr = p->n_refr.data();
    if (d->tuning != nullptr) p->tune = *d->tuning;
    p->desc.tuning = nullptr;
    if (d->pad == 2) { // the plan is built for the [2 ny][2 nx] window; the caller's planes keep the aperture shape
        p->ap_ny = d->ny;
        p->ap_nx = d->nx;
        p->desc.ny = 2 * d->ny;
        p->desc.nx = 2 * d->nx;
    }
    dop_status s;
    try {
        s = build_plan(p);
    } catch (...) {
        s = DOP_ERR_INVALID_ARG;
    }
    if (s != DOP_OK) { delete p; return s; }
    if (workspace_bytes) *workspace_bytes = p->ws_bytes;
    *out = p;
    return DOP_OK;
}

dop_status dop_propagate_fwd(dop_plan* p, const void* d_height, const float* d_target, float* d_intensity,
                             double* d_loss, void* d_workspace, void* cuda_stream)
{
    if (p == nullptr || d_height == nullptr) return DOP_ERR_INVALID_ARG;
    const bool l2 = p->desc.loss == DOP_LOSS_L2, simse = p->desc.loss == DOP_LOSS_SIMSE;
    const bool need_I = !(l2 || simse) || (p->desc.flags & DOP_WRITE_INTENSITY);
    if ((l2 || simse) && d_target == nullptr) return DOP_ERR_INVALID_ARG;
    if (need_I && d_intensity == nullptr) return DOP_ERR_INVALID_ARG;
    if (d_workspace == nullptr) return DOP_ERR_WORKSPACE;
    dop_status s = ensure_device(p);
    if (s != DOP_OK) return s;
    p->state = 0;
    p->prof_n = 0;
    p->target_seen = d_target;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    char* ws = (char*)d_workspace;
    Buffers b;
    b.height = d_height;
    b.height_is_layout = true;
    b.target = d_target;
    b.intensity = d_intensity;
    if (p->pre_stencil) { // F0 as a separable stencil: rows into the (still unused) field area, columns into h_eff
        float* heff = (float*)(ws + p->ws_heff_off);
        if ((s = run_stencil(p, (const float*)d_height, (float*)ws, heff, st, "pre")) != DOP_OK) return s;
        b.height = heff;
        b.height_is_layout = false;
    } else if (!p->pre.empty()) { // F0: h_eff = Re F^-1{ F{U l} G } (the layout is up-sampled inside the first read)
        float* heff = (float*)(ws + p->ws_heff_off);
        Buffers pb;
        pb.real_src = d_height;
        pb.real_src_is_layout = true;
        pb.real_dst = heff;
        if ((s = run(p, p->pre, 0, pb, ws, st, "pre")) != DOP_OK) return s;
        b.height = heff;
        b.height_is_layout = false;
    }
    for (int lam = 0; lam < p->desc.n_lambda; ++lam) {
        if (!zero_pruned_rows(p, ws, lam, st)) return DOP_ERR_CUDA; // pad = 2: the window rows below the aperture enter as zeros
        if ((s = run(p, p->fwd, lam, b, ws, st, "fwd")) != DOP_OK) return s;
        // ... and leave the loss pass as a zero seed (DOP_LOSS_L2: the x passes only touch the aperture rows)
        if (l2 && !zero_pruned_rows(p, ws, lam, st)) return DOP_ERR_CUDA;
    }
    const double npts = p->ap_nx > 0 ? (double)p->ap_nx * (double)p->ap_ny : (double)p->desc.nx * (double)p->desc.ny;
    if (l2 && d_loss != nullptr) {
        long long slot = prof_begin(p, "fwd:loss-reduce", 0.0, st);
        cudaError_t e = launch_loss_reduce((const double*)(ws + p->ws_loss_off), p->loss_tiles * p->desc.n_lambda,
                                           1.0 / npts, d_loss, st);
        prof_end(p, slot, st);
        if (e != cudaSuccess) return DOP_ERR_CUDA;
    }
    if (simse) { // plane sums -> s, L, seed coefficients (needed by adj even when the caller does not want L)
        long long slot = prof_begin(p, "fwd:si-mse-reduce", 0.0, st);
        cudaError_t e = launch_simse_reduce((const double*)(ws + p->ws_loss_off), p->loss_tiles, p->desc.n_lambda, npts,
                                            p->desc.energy_beta, (float*)(ws + p->ws_coef_off), d_loss, st);
        prof_end(p, slot, st);
        if (e != cudaSuccess) return DOP_ERR_CUDA;
    }
    p->state = 1;
    return DOP_OK;
}

static dop_status propagate_adj(dop_plan* p, const void* d_height, const float* d_dLdI, float* d_grad_height,
                                void* d_workspace, void* cuda_stream, const dop_adam* hp, float* d_m, float* d_v)
{
    if (p == nullptr || d_height == nullptr || d_grad_height == nullptr) return DOP_ERR_INVALID_ARG;
    if (p->desc.loss == DOP_LOSS_NONE && d_dLdI == nullptr) return DOP_ERR_INVALID_ARG;
    if (d_workspace == nullptr) return DOP_ERR_WORKSPACE;
    AdamParams ap{};
    if (hp != nullptr) {
        if (d_m == nullptr || d_v == nullptr || p->desc.layout_dtype != DOP_LAYOUT_F32) return DOP_ERR_INVALID_ARG;
        if (!(hp->lr0 >= 0.0) || !(hp->beta1 >= 0.0 && hp->beta1 < 1.0) || !(hp->beta2 >= 0.0 && hp->beta2 < 1.0) ||
            !(hp->eps >= 0.0) || hp->iter < 0 || hp->total_iters < 1 || !std::isfinite(hp->lr0) || !std::isfinite(hp->eps))
            return DOP_ERR_INVALID_ARG;
        const double t = (double)hp->iter + 1.0;
        const double frac = (double)(hp->iter < hp->total_iters ? hp->iter : hp->total_iters) / (double)hp->total_iters;
        const double lr = hp->lr0 * 0.5 * (1.0 + std::cos(M_PI * frac));
        ap.b1 = (float)hp->beta1;
        ap.b2 = (float)hp->beta2;
        ap.c1 = (float)(1.0 - hp->beta1);
        ap.c2 = (float)(1.0 - hp->beta2);
        ap.a1 = (float)(lr / (1.0 - std::pow(hp->beta1, t)));
        ap.rb2 = (float)(1.0 / (1.0 - std::pow(hp->beta2, t)));
        ap.eps = (float)hp->eps;
    }
    if (p->state != 1) return DOP_ERR_STATE;
    dop_status s = ensure_device(p);
    if (s != DOP_OK) return s;
    p->state = 0;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    char* ws = (char*)d_workspace;
    const bool has_pre = p->desc.prefilter_sigma_px > 0.0;
    const bool pooled = p->up_lg > 0;
    const bool plain_layout = !pooled && p->desc.layout_dtype == DOP_LAYOUT_F32;
    float* xpool = (float*)(ws + p->ws_xpool_off);
    Buffers b;
    b.dLdI = d_dLdI;
    b.target = nullptr;
    if (has_pre) {
        b.height = ws + p->ws_heff_off; // the filtered fine plane
        b.grad = plain_layout ? d_grad_height : (float*)(ws + p->ws_gfine_off);
    } else {
        b.height = d_height;
        b.height_is_layout = true;
        b.grad = pooled ? xpool : d_grad_height;
        b.grad_pool = pooled;
        if (hp != nullptr && !pooled) { // Adam rides on the A5 store of the last wavelength
            b.adam = &ap;
            b.adam_m = d_m;
            b.adam_v = d_v;
            b.adam_h = (float*)const_cast<void*>(d_height);
        }
    }
    if (p->desc.loss == DOP_LOSS_SIMSE) b.target = p->target_seen;
    for (int lam = 0; lam < p->desc.n_lambda; ++lam) {
        // pad = 2, caller-seeded adjoint: the seed is zero below the aperture rows
        if (p->desc.loss == DOP_LOSS_NONE && !zero_pruned_rows(p, ws, lam, st)) return DOP_ERR_CUDA;
        if ((s = run(p, p->adj, lam, b, ws, st, "adj")) != DOP_OK) return s;
    }
    if (p->pre_stencil) { // A6 = F0 (g is even): rows into the field area (dead by now), columns back into dL/dh
        if ((s = run_stencil(p, d_grad_height, (float*)ws, d_grad_height, st, "pre-adj")) != DOP_OK) return s;
    } else if (has_pre) { // A6: the Gaussian spectrum is real and even, so the filter is self-adjoint
        Buffers pb;
        pb.real_src = b.grad;
        pb.real_dst = pooled ? xpool : d_grad_height;
        pb.real_dst_pool = pooled;
        if ((s = run(p, p->pre, 0, pb, ws, st, "pre-adj")) != DOP_OK) return s;
    }
    const long long cny = p->desc.ny >> p->up_lg, cnx = p->desc.nx >> p->up_lg;
    if (pooled) { // rows of the x-pooled plane -> coarse dL/dl (+ Adam on the coarse layout)
        long long slot = prof_begin(p, "adj:pool-rows", 4.0 / (double)(1 << p->up_lg), st);
        cudaError_t e = launch_pool_rows(xpool, d_grad_height, cny, cnx, 1 << p->up_lg, hp != nullptr ? &ap : nullptr,
                                         (float*)const_cast<void*>(d_height), d_m, d_v, st);
        prof_end(p, slot, st);
        if (e != cudaSuccess) return DOP_ERR_CUDA;
    } else if (hp != nullptr && has_pre) {
        long long slot = prof_begin(p, "adj:adam", 28.0, st);
        cudaError_t e = launch_adam(d_grad_height, cny * cnx, ap, (float*)const_cast<void*>(d_height), d_m, d_v, st);
        prof_end(p, slot, st);
        if (e != cudaSuccess) return DOP_ERR_CUDA;
    }
    return DOP_OK;
}

dop_status dop_propagate_adj(dop_plan* p, const void* d_height, const float* d_dLdI, float* d_grad_height,
                             void* d_workspace, void* cuda_stream)
{
    return propagate_adj(p, d_height, d_dLdI, d_grad_height, d_workspace, cuda_stream, nullptr, nullptr, nullptr);
}

dop_status dop_propagate_adj_adam(dop_plan* p, float* d_layout, const float* d_dLdI, float* d_grad_height, float* d_m,
                                  float* d_v, const dop_adam* hp, void* d_workspace, void* cuda_stream)
{
    if (hp == nullptr) return DOP_ERR_INVALID_ARG;
    return propagate_adj(p, d_layout, d_dLdI, d_grad_height, d_workspace, cuda_stream, hp, d_m, d_v);
}

dop_status dop_plan_destroy(dop_plan* p)
{
    if (p == nullptr) return DOP_ERR_INVALID_ARG;
    if (p->d_arena != nullptr) cudaFree(p->d_arena);
    for (int k = 0; k < p->n_aux; ++k) {
        if (p->aux[k]) cudaStreamDestroy(p->aux[k]);
        if (p->ev_join[k]) cudaEventDestroy(p->ev_join[k]);
    }
    if (p->ev_fork) cudaEventDestroy(p->ev_fork);
    for (cudaEvent_t e : p->ev_start) cudaEventDestroy(e);
    for (cudaEvent_t e : p->ev_stop) cudaEventDestroy(e);
    delete p;
    return DOP_OK;
}

const char* dop_status_string(dop_status s)
{
    switch (s) {
    case DOP_OK: return "DOP_OK";
    case DOP_ERR_INVALID_ARG: return "DOP_ERR_INVALID_ARG: bad or missing argument";
    case DOP_ERR_UNSUPPORTED_SIZE: return "DOP_ERR_UNSUPPORTED_SIZE: ny and nx must be >= 2 with no prime factor above 127";
    case DOP_ERR_WORKSPACE: return "DOP_ERR_WORKSPACE: workspace missing";
    case DOP_ERR_STATE: return "DOP_ERR_STATE: dop_propagate_adj needs a preceding dop_propagate_fwd";
    case DOP_ERR_ARCH: return "DOP_ERR_ARCH: device is not sm_100";
    case DOP_ERR_CUDA: return "DOP_ERR_CUDA: CUDA runtime error (see cudaGetLastError)";
    case DOP_ERR_NOALLOC_LIMIT: return "DOP_ERR_NOALLOC_LIMIT: dop_prefilter_noalloc takes at most DOP_NOALLOC_MAX_POINTS = 4194304 points (its static scratch array)";
    }
    return "DOP_ERR_UNKNOWN";
}

size_t dop_plan_describe(const dop_plan* p, char* buf, size_t len)
{
    if (p == nullptr) return 0;
    std::string s = describe_plan(p);
    if (buf != nullptr && len > 0) {
        size_t n = s.size() < len - 1 ? s.size() : len - 1;
        std::memcpy(buf, s.data(), n);
        buf[n] = '\0';
    }
    return s.size();
}

int64_t dop_plan_launch_count(const dop_plan* p)
{
    if (p == nullptr) return 0;
    auto count = [&](const std::vector<PassTmpl>& sched) {
        int64_t n = 0;
        size_t i = 0;
        while (i < sched.size()) {
            size_t j = i + 1;
            while (j < sched.size() && sched[j].axis == sched[i].axis) ++j;
            std::vector<PassDesc> d(j - i);
            for (size_t k = i; k < j; ++k) pass_geometry(p, sched[k], &d[k - i]);
            long long total = 0, per = 0;
            const bool slabbed = slab_layout(p, d, sched[i].axis, &total, &per);
            n += (int64_t)(j - i) * (slabbed ? (total + per - 1) / per : 1);
            i = j;
        }
        return n;
    };
    int64_t n = (count(p->fwd) + count(p->adj)) * p->desc.n_lambda + 2 * count(p->pre) + (p->pre_stencil ? 4 : 0);
    if (p->desc.loss == DOP_LOSS_L2 || p->desc.loss == DOP_LOSS_SIMSE) n += 1; // loss / plane-sum reduction
    if (p->up_lg > 0) n += 1;                                                  // row pooling
    return n;
}

dop_status dop_plan_set_profiling(dop_plan* p, int enable)
{
    if (p == nullptr) return DOP_ERR_INVALID_ARG;
    p->profiling = enable != 0;
    p->prof_n = 0;
    return DOP_OK;
}

int64_t dop_plan_get_pass_times(dop_plan* p, float* ms, double* bytes_per_point, int64_t n)
{
    if (p == nullptr) return 0;
    for (size_t i = 0; i < p->prof_n && (int64_t)i < n; ++i) {
        if (ms != nullptr) {
            float t = 0.0f;
            if (cudaEventSynchronize(p->ev_stop[i]) != cudaSuccess ||
                cudaEventElapsedTime(&t, p->ev_start[i], p->ev_stop[i]) != cudaSuccess)
                t = -1.0f;
            ms[i] = t;
        }
        if (bytes_per_point != nullptr) bytes_per_point[i] = p->prof_bpp[i];
    }
    return (int64_t)p->prof_n;
}

const char* dop_plan_pass_name(const dop_plan* p, int64_t i)
{
    if (p == nullptr || i < 0 || (size_t)i >= p->prof_n) return "";
    return p->prof_name[(size_t)i].c_str();
}

} // extern "C"
