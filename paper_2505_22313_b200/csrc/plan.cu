// plan.cu -- host-only plan construction: digit factorisation, twiddle and frequency tables
// (computed in fp64 / long double, rounded once to fp32), pass schedule.  Touches no GPU.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <functional>
#include <sstream>

#include "dop_internal.h"

namespace dop {

static const long double kPiL = 3.141592653589793238462643383279502884L;

constexpr int kMaxPrime = 127; // largest prime factor a digit may carry (direct butterfly in the generic kernel)

static std::vector<long long> prime_factors(long long n) // with multiplicity, ascending; empty if a factor > kMaxPrime
{
    std::vector<long long> f;
    for (long long q = 2; q <= kMaxPrime && n > 1; ++q)
        while (n % q == 0) { f.push_back(q); n /= q; }
    if (n != 1) f.clear();
    return f;
}

static bool supported_size(long long n) { return n >= 2 && !prime_factors(n).empty(); }

static bool is_23_smooth(long long n)
{
    if (n < 2) return false;
    while (n % 2 == 0) n /= 2;
    while (n % 3 == 0) n /= 3;
    return n == 1;
}

// radix steps for one digit: odd primes > 3 first (largest first), then 3s, then 4s, then one 2 if needed
static std::vector<int> radix_steps(long long L)
{
    std::vector<int> r = smooth_radix(L); // 225, 625, 900, 2500: the order the register-step kernels run (smooth.cu)
    if (!r.empty()) return r;
    for (long long q = kMaxPrime; q >= 5; --q)
        while (L % q == 0 && prime_factors(q).size() == 1) { r.push_back((int)q); L /= q; }
    while (L % 3 == 0) { r.push_back(3); L /= 3; }
    while (L % 4 == 0) { r.push_back(4); L /= 4; }
    if (L % 2 == 0) { r.push_back(2); L /= 2; }
    return r;
}

// In-place DIF over radices (r_0..r_{t-1}): slot i = sum c_q m_q (m_q = L/(r_0..r_q)) holds
// output index k = sum c_q (r_0..r_{q-1}).
static std::vector<int> dif_permutation(long long L, const std::vector<int>& radix)
{
    std::vector<int> pi((size_t)L);
    for (long long i = 0; i < L; ++i) {
        long long rem = i, m = L, k = 0, w = 1;
        for (int r : radix) {
            m /= r;
            long long c = rem / m;
            rem -= c * m;
            k += c * w;
            w *= r;
        }
        pi[(size_t)i] = (int)k;
    }
    return pi;
}

static std::vector<float2> twiddle_table(long long n)
{
    std::vector<float2> w((size_t)n);
    for (long long k = 0; k < n; ++k) {
        long double a = 2.0L * kPiL * (long double)k / (long double)n;
        w[(size_t)k] = make_float2((float)cosl(a), (float)(-sinl(a)));
    }
    return w;
}

// Split N into the fewest digits with every digit <= lmax_first (all but the last) and the last
// <= lmax_last, as balanced as possible.  A forced decomposition (dop_tuning) overrides; it must
// multiply to N and respect the same limits.
static bool split_digits(long long N, long long lmax_first, long long lmax_last, int n_forced,
                         const int64_t* forced, std::vector<long long>* out, bool last_is_row, bool tu_no_smooth)
{
    out->clear();
    if (n_forced > 0) {
        if (n_forced > 4) return false;
        long long prod = 1;
        for (int i = 0; i < n_forced; ++i) {
            const long long x = forced[i];
            if (x < 2 || x > (i + 1 < n_forced ? lmax_first : lmax_last)) return false;
            out->push_back(x);
            prod *= x;
        }
        return prod == N;
    }
    if (N <= lmax_last) { out->push_back(N); return true; }
    // divisors of N
    std::vector<long long> divs{1};
    {
        const std::vector<long long> pf = prime_factors(N);
        for (size_t i = 0; i < pf.size();) {
            size_t j = i;
            while (j < pf.size() && pf[j] == pf[i]) ++j;
            const size_t base = divs.size();
            long long pw = 1;
            for (size_t e = i; e < j; ++e) {
                pw *= pf[i];
                for (size_t k = 0; k < base; ++k) divs.push_back(divs[k] * pw);
            }
            i = j;
        }
    }
    std::sort(divs.begin(), divs.end());
    if (!is_23_smooth(N)) {
        // General sizes: a digit the register-blocked / TMA kernels handle costs 1, a digit of the generic kernel
        // 4 plus its largest prime factor / 8 (direct butterflies); the cheapest decomposition into at most four
        // digits wins, ties go to the smaller largest digit.
        // The first x digit carries the fused exp(i Phi) / loss / dL/dh ops and the last y digit the (x) H
        // sandwich: only pure powers of two run those on the specialised kernels (3 * 2^k digits: plain passes).
        auto digit_cost = [&](long long dgt, bool first, bool last) {
            const bool col = !(last && last_is_row);
            const bool fused = last_is_row ? first : last;
            // (fused x passes stage their fp32 planes by TMA: the line count N / dgt must be a multiple of 4)
            const bool planes_ok = !(last_is_row && first && !last) || (N / dgt) % 4 == 0;
            if (pow2_supported(dgt, col) && !(fused && dgt % 3 == 0) && planes_ok) return 1.0;
            if (!fused && !tu_no_smooth && smooth_supported(dgt, col)) return 1.5; // register-step kernels (smooth.cu)
            const std::vector<long long> f = prime_factors(dgt);
            return (fused ? 6.0 : 4.0) + (f.back() > 7 ? (double)f.back() / 4.0 : 0.0);
        };
        double best_c = -1.0;
        long long best_m = 0;
        std::vector<long long> cur, bestv;
        std::function<void(long long, double, long long)> rec = [&](long long rem, double cost, long long mx) {
            if (best_c >= 0.0 && cost >= best_c + 1e-9 && !(cost <= best_c + 1e-9 && mx < best_m)) return;
            if (rem >= 2 && rem <= lmax_last) { // close with `rem` as the last digit
                const double c = cost + digit_cost(rem, cur.empty(), true);
                const long long m2 = std::max(mx, rem);
                if (best_c < 0.0 || c < best_c - 1e-9 || (c <= best_c + 1e-9 && m2 < best_m)) {
                    best_c = c; best_m = m2; bestv = cur; bestv.push_back(rem);
                }
            }
            if (cur.size() >= 3) return;
            for (long long d0 : divs) {
                // (generic column digits: 16 lines x d0 points, twice that with an out-of-place prime step, in 200 KiB)
                const std::vector<long long> f0 = prime_factors(d0);
                const long long lim = (!f0.empty() && f0.back() > 7) ? 512 : 1024;
                if (d0 < 2 || d0 > std::max(lmax_first, lim) || d0 > lim || rem % d0 != 0 || rem / d0 < 2) continue;
                cur.push_back(d0);
                rec(rem / d0, cost + digit_cost(d0, cur.size() == 1, false), std::max(mx, d0));
                cur.pop_back();
            }
        };
        rec(N, 0.0, 0);
        if (best_c < 0.0) return false;
        *out = bestv;
        return true;
    }
    // two digits
    long long best = -1, best_cost = 0;
    for (long long d0 : divs) {
        long long d1 = N / d0;
        if (d0 < 2 || d1 < 2 || d0 > lmax_first || d1 > lmax_last) continue;
        long long cost = std::max(d0, d1);
        if (best < 0 || cost < best_cost || (cost == best_cost && d0 > best)) { best = d0; best_cost = cost; }
    }
    if (best > 0) { out->push_back(best); out->push_back(N / best); return true; }
    // three digits
    long long b0 = -1, b1 = -1;
    best_cost = 0;
    for (long long d0 : divs)
        for (long long d1 : divs) {
            if (d0 < 2 || d1 < 2 || (N / d0) % d1 != 0) continue;
            long long d2 = N / d0 / d1;
            if (d2 < 2 || d0 > lmax_first || d1 > lmax_first || d2 > lmax_last) continue;
            long long cost = std::max(d0, std::max(d1, d2));
            if (b0 < 0 || cost < best_cost) { b0 = d0; b1 = d1; best_cost = cost; }
        }
    if (b0 > 0) { out->push_back(b0); out->push_back(b1); out->push_back(N / b0 / b1); return true; }
    return false;
}

static int wl_table_index(dop_plan* p, long long L)
{
    for (size_t i = 0; i < p->wl_len.size(); ++i)
        if (p->wl_len[i] == L) return (int)i;
    p->wl_len.push_back(L);
    p->wl_tables.push_back(twiddle_table(L));
    return (int)p->wl_len.size() - 1;
}

static bool build_axis(dop_plan* p, int a, long long N, const std::vector<long long>& Ls)
{
    const bool tu_no_tma = p->tune.no_tma != 0;
    Axis& ax = p->ax[a];
    ax.N = N;
    ax.dig.resize(Ls.size());
    long long st = N;
    for (size_t j = 0; j < Ls.size(); ++j) {
        Digit& d = ax.dig[j];
        d.L = Ls[j];
        st /= Ls[j];
        d.st = st;
        d.radix = radix_steps(d.L);
        if ((int)d.radix.size() > kMaxRadixSteps) return false;
        d.pi = dif_permutation(d.L, d.radix);
        d.wl_index = wl_table_index(p, d.L);
        d.has_twb = (j + 1 < Ls.size());
        if (d.has_twb) d.twb = twiddle_table(d.L * d.st);
        // column-type unless it is the last x digit
        const bool col_type = !(a == 0 && d.st == 1);
        const long long lines = col_type ? (a == 0 ? d.st : p->desc.nx) : p->desc.ny * (N / d.L);
        // (a column digit whose line count is not a multiple of 16 still counts as fast: the TMA kernels clip ragged
        // tiles in hardware; the LDG/STG kernels decline such a pass at dispatch and the generic kernel runs it)
        d.fast = !p->force_generic && pow2_supported(d.L, col_type) &&
                 (col_type ? (lines % 16 == 0 || !tu_no_tma) : lines % pow2_lines(d.L, false) == 0);
        // pad = 2: the fused x passes mask their plane accesses to the aperture, which only the generic kernel
        // implements (the plain x passes and every y pass keep the specialised kernels)
        // ... unless the x axis has two digits and the first is a power of two: its fused passes then run on the TMA
        // kernels, where the TMA unit itself masks the planes to the aperture (resolve() sends anything else to the generic kernel)
        const bool pad_tma = Ls.size() == 2 && (d.L & (d.L - 1)) == 0 && d.L >= 16 && !tu_no_tma && !p->force_generic;
        if (p->ap_nx > 0 && a == 0 && j == 0 && !pad_tma) d.fast = false;
        // 5-smooth digits with register-step kernels for their plain passes (smooth.cu)
        d.smooth = !p->force_generic && !p->tune.no_smooth && !d.fast && smooth_supported(d.L, col_type);
        if (d.fast) d.twg = pow2_group_twiddles(d.L);
        if ((d.fast || (d.smooth && col_type)) && d.has_twb) { // W_{N_j}^{r pi[slot]}: y digits [r][slot], x digits [slot][r]
            const long long Nj = d.L * d.st;
            d.twb2.resize((size_t)Nj);
            for (long long r = 0; r < d.st; ++r)
                for (long long sl = 0; sl < d.L; ++sl) {
                    const float2 w = d.twb[(size_t)((r * d.pi[(size_t)sl]) % Nj)];
                    d.twb2[(size_t)(a == 1 ? r * d.L + sl : sl * d.st + r)] = w;
                }
        }
    }
    // slot -> true frequency index:  k = sum_j pi_j(p_j) (L_0 .. L_{j-1})
    ax.kslot.resize((size_t)N);
    ax.f2.resize((size_t)N);
    ax.fsigned.resize((size_t)N);
    ax.g.resize((size_t)N);
    const double pitch = p->desc.pitch, sigma = p->desc.prefilter_sigma_px;
    for (long long s = 0; s < N; ++s) {
        long long k = 0, w = 1;
        for (const Digit& d : ax.dig) {
            long long pj = (s / d.st) % d.L;
            k += (long long)d.pi[(size_t)pj] * w;
            w *= d.L;
        }
        ax.kslot[(size_t)s] = k;
        // signed bin, then the definition's own fp64 expressions (F4 / O4)
        double kb = (double)(k < (N + 1) / 2 ? k : k - N);
        double f = kb / ((double)N * pitch);
        ax.f2[(size_t)s] = f * f;
        ax.fsigned[(size_t)s] = f;
        double v = kb / (double)N;
        ax.g[(size_t)s] = (float)std::exp(-2.0 * M_PI * M_PI * sigma * sigma * (v * v));
    }
    return true;
}

static PassTmpl mk(int axis, int digit, int d1, int d2, int ld, int mid, int st, const char* nm, double rd,
                   double wr, double side = 0.0)
{
    PassTmpl t;
    t.axis = axis; t.digit = digit; t.fft1_dir = d1; t.fft2_dir = d2;
    t.load_op = ld; t.mid_op = mid; t.store_op = st; t.name = nm;
    t.rd = rd; t.wr = wr; t.side = side;
    t.bytes_per_point = rd + wr + side;
    return t;
}

// passes of  F^-1{ mid (x) F{.} }  minus the first forward x digit and the last inverse x digit
static void sandwich_core(const dop_plan* p, int mid, bool with_xfwd, std::vector<PassTmpl>* out)
{
    const int a = p->x_cluster ? 1 : (int)p->ax[0].dig.size(), b = (int)p->ax[1].dig.size();
    if (with_xfwd)
        for (int j = 1; j < a; ++j) out->push_back(mk(0, j, +1, 0, LD_C64, MID_NONE, ST_C64, "x-fwd", 8, 8));
    for (int j = 0; j + 1 < b; ++j) out->push_back(mk(1, j, +1, 0, LD_C64, MID_NONE, ST_C64, "y-fwd", 8, 8));
    out->push_back(mk(1, b - 1, +1, -1, LD_C64, mid, ST_C64,
                      mid == MID_H ? "y-fwd*H*y-inv" : mid == MID_HCONJ ? "y-fwd*conjH*y-inv" : "y-fwd*G*y-inv", 8, 8));
    for (int j = b - 2; j >= 0; --j) out->push_back(mk(1, j, -1, 0, LD_C64, MID_NONE, ST_C64, "y-inv", 8, 8));
    for (int j = a - 1; j >= 1; --j) out->push_back(mk(0, j, -1, 0, LD_C64, MID_NONE, ST_C64, "x-inv", 8, 8));
}

static void build_schedule(dop_plan* p)
{
    const bool l2 = p->desc.loss == DOP_LOSS_L2;
    const bool wi = l2 && (p->desc.flags & DOP_WRITE_INTENSITY);
    // with cluster row passes the x digits (16, M) always run fused: one x pass per transform pair
    const int a = p->x_cluster ? 1 : (int)p->ax[0].dig.size();
    p->fwd.clear(); p->adj.clear(); p->pre.clear();
    // forward
    p->fwd.push_back(mk(0, 0, +1, 0, LD_HEIGHT, MID_NONE, ST_C64, "h->u0,x-fwd", 4, 8));
    sandwich_core(p, MID_H, true, &p->fwd);
    if (l2) {
        // the seed's forward x transform belongs to the same row sandwich as the loss pass, so in
        // L2 mode all of it runs inside dop_propagate_fwd (dop.h: the workspace then holds "the
        // seeded, partly transformed gradient field")
        p->fwd.push_back(mk(0, 0, -1, +1, LD_C64, MID_LOSS, ST_C64, "x-inv,|u|^2,loss,seed,x-fwd", 8, 8, wi ? 8 : 4));
        for (int j = 1; j < a; ++j) p->fwd.push_back(mk(0, j, +1, 0, LD_C64, MID_NONE, ST_C64, "x-fwd", 8, 8));
    } else if (p->desc.loss == DOP_LOSS_SIMSE) {
        // Eq. (6): the least-squares scale s needs the sums of the whole plane before the seed, so the row
        // sandwich around the loss splits at the call boundary (as for DOP_LOSS_NONE)
        const bool wis = (p->desc.flags & DOP_WRITE_INTENSITY) != 0;
        p->fwd.push_back(mk(0, 0, -1, 0, LD_C64, MID_NONE, ST_C64_STATS, "x-inv,|u|^2,plane sums", 8, 8, wis ? 8 : 4));
        p->adj.push_back(mk(0, 0, +1, 0, LD_SEED_SIMSE, MID_NONE, ST_C64, "si-mse seed,x-fwd", 8, 8, 4));
    } else {
        p->fwd.push_back(mk(0, 0, -1, 0, LD_C64, MID_NONE, ST_C64_INTENSITY, "x-inv,|u|^2", 8, 8, 4));
        p->adj.push_back(mk(0, 0, +1, 0, LD_SEED, MID_NONE, ST_C64, "seed,x-fwd", 8, 8, 4));
    }
    // adjoint
    sandwich_core(p, MID_HCONJ, !l2, &p->adj);
    p->adj.push_back(mk(0, 0, -1, 0, LD_C64, MID_NONE, ST_GRAD, "x-inv,grad", 8, 4, 4));
    // Gaussian pre-filter (real plane -> real plane through the complex field buffer), unless it runs as a stencil
    if (p->desc.prefilter_sigma_px > 0.0 && !p->pre_stencil) {
        p->pre.push_back(mk(0, 0, +1, 0, LD_REAL, MID_NONE, ST_C64, "real,x-fwd", 4, 8));
        sandwich_core(p, MID_GAUSS, true, &p->pre);
        p->pre.push_back(mk(0, 0, -1, 0, LD_C64, MID_NONE, ST_REAL, "x-inv,real", 8, 4));
    }
    if ((p->up_lg > 0 || p->desc.layout_dtype != DOP_LAYOUT_F32) && p->pre.empty()) {
        // super-resolved layout: the height is read from the coarse plane (hb bytes per fine point) and dL/dh
        // leaves as the x-pooled plane (4 / r bytes per fine point).  (With the pre-filter the phase passes work
        // on the filtered fine plane; the coarse read / pooled write then sit at the two ends of the filter.)
        const double r = (double)(1 << p->up_lg);
        const double hb = (p->desc.layout_dtype == DOP_LAYOUT_U8 ? 1.0 : p->desc.layout_dtype == DOP_LAYOUT_U16 ? 2.0 : 4.0) / (r * r);
        for (std::vector<PassTmpl>* v : {&p->fwd, &p->adj})
            for (PassTmpl& t : *v) {
                if (t.load_op == LD_HEIGHT) t.rd = hb;
                if (t.store_op == ST_GRAD) { t.side = hb; t.wr = 4.0 / r; }
                t.bytes_per_point = t.rd + t.wr + t.side;
            }
    }
    if (p->x_cluster)
        for (std::vector<PassTmpl>* v : {&p->fwd, &p->adj, &p->pre})
            for (PassTmpl& t : *v)
                if (t.axis == 0) t.cluster = 1;
}

void tile_geometry(const dop_plan* p, int axis, int digit, PassDesc* d)
{
    const long long nx = p->desc.nx, ny = p->desc.ny;
    const Digit& g = p->ax[axis].dig[(size_t)digit];
    const long long L = g.L, st = g.st;
    d->L = (int)L;
    d->n_radix = (int)g.radix.size();
    for (int i = 0; i < d->n_radix; ++i) d->radix[i] = g.radix[(size_t)i];
    long long nl_target = std::max<long long>(1, p->tile_pts / L);
    const bool fast = g.fast;
    d->row_o = d->row_m = d->row_i = 0;
    if (axis == 0 && st == 1) { // last x digit: row-type, lines are contiguous runs of L
        d->col_type = 0;
        d->es = 1;
        d->NC = ny * nx / L;
        d->SCc = L;
        d->n_m = 1; d->SM = 0; d->n_o = 1; d->SO = 0;
        d->r_from = 0;
        d->nl = fast ? pow2_lines(L, false) : (int)std::min<long long>(nl_target, d->NC);
    } else if (axis == 0) { // higher x digit: lines r..r+nl-1 adjacent, elements st apart
        d->col_type = 1;
        d->es = st;
        d->NC = st; d->SCc = 1;
        d->n_m = nx / (L * st); d->SM = L * st;
        d->n_o = ny; d->SO = nx;
        d->r_from = 0;
        d->nl = fast ? 16 : (int)std::min<long long>(std::max<long long>(nl_target, 16), st);
    } else { // y digit: lines are adjacent columns, elements st rows apart
        d->col_type = 1;
        d->es = st * nx;
        d->NC = nx; d->SCc = 1;
        d->n_m = st; d->SM = nx;
        d->n_o = ny / (L * st); d->SO = L * st * nx;
        d->r_from = 1;
        d->row_o = L * st; d->row_m = 1; d->row_i = st;
        d->nl = fast ? 16 : (int)std::min<long long>(std::max<long long>(nl_target, 16), nx);
    }
    d->n_cgroups = (d->NC + d->nl - 1) / d->nl;
    d->smem_bytes = (int)((long long)d->nl * L * (long long)sizeof(float2));
    for (int rr : g.radix)
        if (rr > 7) { d->smem_bytes *= 2; break; } // out-of-place scratch of the larger odd-prime steps (kernels_generic.cu)
    d->threads = 256;
}

// Geometry of one scheduled pass: tile_geometry of its digit, then the column bundle width, which
// is a property of the pass (it does not change where data lives): plain forward / inverse
// passes (and the exp(i Phi) pass of short digits) take wider bundles (pow2_lines), the register-heavy fused
// variants stay at 16 columns.
static void pass_geometry_full(const dop_plan* p, const PassTmpl& t, PassDesc* d, bool allow_tma);

// pad = 2: every x pass runs on the aperture rows only (rows below are known zeros on the way in and discarded on
// the way out: "pruned" passes); the geometry of the full window is cut down to the first ap_ny rows here, so that
// describe, the loss partial count and the launches all see the same tiles.
void pass_geometry(const dop_plan* p, const PassTmpl& t, PassDesc* d, bool allow_tma)
{
    pass_geometry_full(p, t, d, allow_tma);
    if (p->ap_nx == 0 || t.axis != 0) return;
    if (d->col_type) {
        d->n_o = p->ap_ny;
    } else {
        const long long lpr = p->desc.nx / d->L; // lines per row
        d->NC = p->ap_ny * lpr;
        d->n_cgroups = (d->NC + d->nl - 1) / d->nl;
    }
}

static void pass_geometry_full(const dop_plan* p, const PassTmpl& t, PassDesc* d, bool allow_tma)
{
    if (t.cluster) { // one cluster of C CTAs per row; CTA = S lines of M points
        const long long M = p->ax[0].dig[1].L;
        const int C = p->tune.cluster_lines > 0 ? 16 / p->tune.cluster_lines : cluster_size(M);
        *d = PassDesc{};
        d->cluster = p->tune.cluster_dsmem ? 2 : 1;
        d->L = (int)M;
        d->nl = 16 / C;
        d->col_type = 0;
        d->es = 1;
        d->NC = C; d->SCc = 0;
        d->n_cgroups = C;
        d->n_m = 1; d->SM = 0;
        d->n_o = p->desc.ny; d->SO = p->desc.nx;
        d->smem_bytes = (int)((16 / C) * (M + 2 * (M / 32)) * (long long)sizeof(float2));
        d->threads = (int)((16 / C) * (M / 16));
        return;
    }
    tile_geometry(p, t.axis, t.digit, d);
    const Digit& g = p->ax[t.axis].dig[(size_t)t.digit];
    if (g.smooth && t.mid_op == MID_NONE && t.fft2_dir == 0 && t.load_op == LD_C64 && t.store_op == ST_C64) {
        smooth_geometry(g.L, d->col_type != 0, &d->nl, &d->threads, &d->smem_bytes);
        d->n_cgroups = (d->NC + d->nl - 1) / d->nl;
        d->smooth = 1;
        return;
    }
    if (!g.fast || !d->col_type) return;
    // Column passes the TMA kernels implement (tma_col.cuh) run there: bundle width and pipeline depth per
    // digit length and variant (measured, profiles/r02_tma_col.md), dop_tuning.tma_nb / tma_stages override.
    if (allow_tma && p->use_tma) {
        const bool x3 = g.L % 3 == 0;
        const bool plain_layout = p->up_lg == 0 && p->desc.layout_dtype == DOP_LAYOUT_F32;
        const bool sandwich = t.fft1_dir > 0 && t.fft2_dir < 0 && t.load_op == LD_C64 && t.store_op == ST_C64 &&
                              (t.mid_op == MID_H || t.mid_op == MID_HCONJ || t.mid_op == MID_GAUSS);
        const bool plainpass = t.mid_op == MID_NONE && t.fft2_dir == 0 && t.load_op == LD_C64 && t.store_op == ST_C64;
        const bool lossp = t.mid_op == MID_LOSS && t.fft1_dir < 0 && t.fft2_dir > 0 && t.load_op == LD_C64 && t.store_op == ST_C64;
        const bool heightp = t.mid_op == MID_NONE && t.fft2_dir == 0 && t.load_op == LD_HEIGHT && t.store_op == ST_C64 && plain_layout;
        const bool gradp = t.mid_op == MID_NONE && t.fft2_dir == 0 && t.load_op == LD_C64 && t.store_op == ST_GRAD && plain_layout;
        // (h -> exp(i Phi) -> DFT through TMA: 16-column tiles measured SLOWER than the LDG/STG kernel -- C4 14.6 against
        // 13.7 ms, C5 22.0 against 21.0 -- and 32-column tiles of 256 slots faster -- C4 12.9, C5 19.7; so digits of 256
        // go there, and otherwise only what that kernel cannot run: a line count that is not a multiple of 16, pad = 2)
        const bool height_wide = heightp && g.L == 256 && d->NC % 32 == 0 && p->ap_nx == 0;
        const bool heightp_tma = heightp && (height_wide || d->NC % 16 != 0 || p->ap_nx > 0); // (pad = 2: only the TMA kernel masks)
        // the split loss flavours: IDFT -> u, |u|^2 [, plane sums]  and  seed from u and dL/dI (or T) -> DFT
        const bool statp = t.mid_op == MID_NONE && t.fft2_dir == 0 && t.load_op == LD_C64 &&
                           (t.store_op == ST_C64_INTENSITY || t.store_op == ST_C64_STATS) && t.axis == 0;
        const bool seedp = t.mid_op == MID_NONE && t.fft2_dir == 0 && t.store_op == ST_C64 &&
                           (t.load_op == LD_SEED || t.load_op == LD_SEED_SIMSE) && t.axis == 0;
        const bool has_plane = lossp || heightp_tma || gradp || statp || seedp;
        // (the TMA (x) H kernel takes the phase in 32-bit fixed point: |z|/lambda < 2^19 for every wavelength)
        bool h_ok = !p->h_float;
        for (double lam : p->lambda) h_ok = h_ok && std::fabs(p->desc.z) / lam < 524288.0;
        const bool sandwich_ok = sandwich && (t.mid_op == MID_GAUSS || h_ok);
        if (plainpass || (!x3 && (sandwich_ok || has_plane))) {
            // measured per variant at L = 256 (C4): plain passes and the dL/dh store are near the pattern's ceiling
            // with 32-column tiles, the register-heavy fused variants want 16 columns (two CTAs per SM)
            int nb = 32, nst = g.L <= 128 ? 3 : 2;
            if (sandwich || lossp || statp || seedp) { nb = 16; nst = 3; }
            if (heightp_tma) { nb = height_wide ? 32 : 16; nst = g.L == 256 ? 2 : 3; }
            if (g.L == 512) { nb = 16; nst = 2; }
            if (x3) { nb = 32; nst = g.L == 384 ? 2 : 3; }
            if (p->tma_nb) nb = p->tma_nb;
            if (p->tma_stages) nst = p->tma_stages;
            auto fits = [&](int b, int n) {
                // (TMA global strides are multiples of 16 bytes: complex64 field and, for the fused x variants, fp32 planes)
                const long long sa = has_plane ? 4 : 2;
                if (d->es % sa != 0 || (d->n_m > 1 && d->SM % sa != 0) || (d->n_o > 1 && d->SO % sa != 0)) return false;
                return tma_instantiated(g.L, b, n) && d->NC >= b &&
                       (long long)n * g.L * b * (has_plane ? 12 : 8) <= 227 * 1024 - 2048;
            };
            if (!fits(nb, nst)) { // nearest instantiated choice
                bool found = false;
                for (int n = nst; n >= 1 && !found; --n)
                    for (int b : {nb, 16, 32})
                        if (fits(b, n)) { nb = b; nst = n; found = true; break; }
                if (!found) nst = 0;
            }
            if (nst > 0) {
                d->tma = nst;
                d->nl = nb;
                d->n_cgroups = (d->NC + nb - 1) / nb; // (a ragged last tile is clipped by the TMA unit)
                d->smem_bytes = (int)((long long)nst * g.L * nb * (has_plane ? 12 : 8));
                d->threads = (int)(nb * ((x3 ? g.L / 3 : g.L) / 16) + 32);
                return;
            }
        }
    }
    // (the exp(i Phi) pass: measured better at 32 columns for L = 128, worse for L = 256)
    // and the gradient / real-plane stores: +5-10 % at 32 columns for L = 128, no change for L = 256)
    const bool short_digit = g.L <= 128;
    const bool plain = t.mid_op == MID_NONE && t.fft2_dir == 0 &&
                       ((t.store_op == ST_C64 && (t.load_op == LD_C64 || (t.load_op == LD_HEIGHT && short_digit))) ||
                        (t.load_op == LD_C64 && short_digit &&
                         (t.store_op == ST_GRAD || t.store_op == ST_GRAD_ACC || t.store_op == ST_REAL)));
    const int nb = pow2_lines(g.L, true, plain, p->col_nb);
    if (nb != d->nl && d->NC % nb == 0) {
        d->nl = nb;
        d->n_cgroups = d->NC / nb;
        d->smem_bytes = (int)((long long)nb * g.L * (long long)sizeof(float2));
    }
}

dop_status build_plan(dop_plan* p)
{
    const dop_plan_desc& d = p->desc;
    if (!supported_size(d.nx) || !supported_size(d.ny)) return DOP_ERR_UNSUPPORTED_SIZE;
    const dop_tuning& tu = p->tune;
    p->force_generic = tu.force_generic != 0;
    // ---- design-loop options
    if (d.loss == DOP_LOSS_SIMSE && !(std::isfinite(d.energy_beta) && d.energy_beta >= 0.0)) return DOP_ERR_INVALID_ARG;
    if (d.layout_dtype != DOP_LAYOUT_F32 && d.layout_dtype != DOP_LAYOUT_U8 && d.layout_dtype != DOP_LAYOUT_U16)
        return DOP_ERR_INVALID_ARG;
    if (d.layout_dtype != DOP_LAYOUT_F32 && !(std::isfinite(d.layout_step) && d.layout_step > 0.0)) return DOP_ERR_INVALID_ARG;
    p->up_lg = 0;
    if (d.upsample != 0 && d.upsample != 1) {
        if (d.upsample != 2 && d.upsample != 4 && d.upsample != 8) return DOP_ERR_INVALID_ARG;
        p->up_lg = d.upsample == 2 ? 1 : (d.upsample == 4 ? 2 : 3);
        if (d.nx % d.upsample != 0 || d.ny % d.upsample != 0) return DOP_ERR_UNSUPPORTED_SIZE;
    }
    if (tu.tile_pts != 0) {
        if (tu.tile_pts < 256 || tu.tile_pts > 16384) return DOP_ERR_INVALID_ARG;
        p->tile_pts = tu.tile_pts;
    }
    if (tu.col_nb != 0 && tu.col_nb != 16 && tu.col_nb != 32 && tu.col_nb != 64) return DOP_ERR_INVALID_ARG;
    p->col_nb = tu.col_nb;
    p->h_float = tu.h_float != 0;
    if (tu.slab_streams < 0 || tu.slab_streams > 4) return DOP_ERR_INVALID_ARG;
    p->slab_streams = tu.slab_streams == 0 ? 2 : tu.slab_streams;
    if (tu.prefetch_waves < -1 || tu.prefetch_waves > 64) return DOP_ERR_INVALID_ARG;
    p->pf_waves = tu.prefetch_waves == 0 ? 1 : (tu.prefetch_waves < 0 ? 0 : tu.prefetch_waves);
    // Multi-pass segments can run slab by slab so that the passes after the first hit L2.  Off by
    // default: measured slower than whole-array launches on B200.
    if (tu.slab_mb < 0 || tu.slab_mb > 4096) return DOP_ERR_INVALID_ARG;
    p->slab_bytes = (long long)tu.slab_mb << 20;
    if (tu.tma_nb != 0 && tu.tma_nb != 16 && tu.tma_nb != 32 && tu.tma_nb != 64) return DOP_ERR_INVALID_ARG;
    if (tu.tma_stages < 0 || tu.tma_stages > 8) return DOP_ERR_INVALID_ARG;
    p->use_tma = !tu.no_tma && !p->force_generic;
    p->tma_nb = tu.tma_nb;
    p->tma_stages = tu.tma_stages;
    if (tu.cluster_lines != 0 && tu.cluster_lines != 1 && tu.cluster_lines != 2 && tu.cluster_lines != 4 && tu.cluster_lines != 8)
        return DOP_ERR_INVALID_ARG;
    // generic kernel limits: a row-type line <= 8192 points (64 KiB), a column-type digit
    // <= 512 points (x 16 adjacent lines = 64 KiB)
    std::vector<long long> lx, ly;
    // Cluster row passes: measured on B200 a gain for clusters of 2 (nx = 16384: C3 +7 %), a loss of
    // 5-15 % against two digit passes for clusters of 4-16 (profiles/r02_cluster.md), so only the
    // former is a default; dop_tuning.cluster_force selects them wherever they exist.
    const bool may_cluster = !tu.no_cluster && !p->force_generic;
    const bool want_cluster = may_cluster && p->ap_nx == 0 && d.nx % 16 == 0 && cluster_supported(16, d.nx / 16) &&
                              (tu.cluster_force || d.nx == 16384);
    if (want_cluster && tu.n_xdigits == 0) {
        lx = {16, d.nx / 16}; // rows of 16 M points: one thread-block-cluster pass per transform pair
    } else if (!split_digits(d.nx, 512, 8192, tu.n_xdigits, tu.xdigits, &lx, true, tu.no_smooth != 0)) return DOP_ERR_UNSUPPORTED_SIZE;
    if (!split_digits(d.ny, 512, 512, tu.n_ydigits, tu.ydigits, &ly, false, tu.no_smooth != 0)) return DOP_ERR_UNSUPPORTED_SIZE;
    if (!build_axis(p, 0, d.nx, lx) || !build_axis(p, 1, d.ny, ly)) return DOP_ERR_UNSUPPORTED_SIZE;
    p->x_cluster = want_cluster && lx.size() == 2 && cluster_supported(lx[0], lx[1]) && p->ax[0].dig[0].fast &&
                   p->ax[0].dig[1].fast;
    if (p->x_cluster && tu.cluster_lines > 0 && !cluster_instantiated(lx[1], tu.cluster_lines)) return DOP_ERR_INVALID_ARG;
    // Pre-filter as a separable spatial stencil (blur.cu) when its kernel is short: taps = the definition's own
    // inverse DFT g[n] = (1/N) sum_k Ghat(k) cos(2 pi k n / N), n <= R = ceil(6 sigma), summed here in fp64.
    p->pre_stencil = false;
    if (d.prefilter_sigma_px > 0.0 && !tu.no_stencil && !p->force_generic && p->up_lg == 0 && d.layout_dtype == DOP_LAYOUT_F32) {
        const int R = (int)std::ceil(6.0 * d.prefilter_sigma_px);
        // (below sigma ~ 2 px the sampled spectrum is still 1e-9 or more at Nyquist: its inverse DFT then rings far beyond 6 sigma)
        if (d.prefilter_sigma_px >= 2.05 && R <= 24 && d.nx % 8 == 0 && d.ny % 32 == 0 && d.nx >= 2 * R + 8 && d.ny >= 2 * R + 32) {
            auto taps = [&](long long N, std::vector<float>* w) {
                w->assign((size_t)R + 1, 0.0f);
                const double sg = d.prefilter_sigma_px;
                for (int n = 0; n <= R; ++n) {
                    long double acc = 0.0L;
                    for (long long k = 0; k < N; ++k) {
                        const double kb = (double)(k < (N + 1) / 2 ? k : k - N), v = kb / (double)N;
                        acc += (long double)std::exp(-2.0 * M_PI * M_PI * sg * sg * (v * v)) *
                               cosl(2.0L * kPiL * (long double)((k * n) % N) / (long double)N);
                    }
                    (*w)[(size_t)n] = (float)(acc / (long double)N);
                }
            };
            taps(d.nx, &p->blur_wx);
            taps(d.ny, &p->blur_wy);
            p->blur_radius = R;
            p->pre_stencil = true;
        }
    }
    build_schedule(p);
    // (x) H on mirrored tile pairs (tma_col.cuh): tile o of the last y digit holds k_low(o) + N_low k_last; its mirror
    // holds N_low - k_low(o).  Needs a pure power-of-two last digit (slot L - 1 - i <-> k_last L - 1 - k_last).
    p->hpair_items.clear();
    {
        const Axis& ay = p->ax[1];
        const Digit& last = ay.dig.back();
        const bool pow2 = (last.L & (last.L - 1)) == 0 && last.L >= 16;
        if (ay.dig.size() >= 2 && pow2 && last.fast && !tu.no_mirror && p->use_tma) {
            const long long L = last.L, nlow = ay.N / L;
            std::vector<long long> o_of((size_t)nlow, -1);
            for (long long o = 0; o < nlow; ++o) o_of[(size_t)(ay.kslot[(size_t)(o * L)] % nlow)] = o;
            std::vector<int> singles;
            for (long long o = 0; o < nlow; ++o) {
                const long long kl = ay.kslot[(size_t)(o * L)] % nlow, om = o_of[(size_t)((nlow - kl) % nlow)];
                if (om == o) singles.push_back((int)o);
                else if (o < om) { p->hpair_items.push_back((int)o); p->hpair_items.push_back((int)om); }
            }
            for (int o : singles) { p->hpair_items.push_back(o); p->hpair_items.push_back(-1); }
        }
    }
    // CTAs of the MID_LOSS / plane-sum pass, in the geometry it is launched with (partials per CTA)
    p->loss_tiles = 0;
    for (const PassTmpl& t : p->fwd)
        if (t.mid_op == MID_LOSS || t.store_op == ST_C64_STATS) {
            PassDesc g{};
            pass_geometry(p, t, &g);
            p->loss_tiles = g.n_cgroups * g.n_m * g.n_o;
        }
    // The sum-pool along x is a shuffle reduction over r adjacent lanes of the register-blocked kernels: the
    // pass that stores dL/dh (and the pre-filter's real-plane store) must be one of them, with r | its lane run
    if (p->up_lg > 0) {
        const int r = 1 << p->up_lg;
        for (const std::vector<PassTmpl>* v : {&p->adj, &p->pre})
            for (const PassTmpl& t : *v) {
                if (t.store_op != ST_GRAD && t.store_op != ST_REAL) continue;
                PassDesc g{};
                pass_geometry(p, t, &g);
                const Digit& dg = p->ax[0].dig[0];
                bool ok = t.cluster || dg.fast;
                if (ok && !t.cluster) ok = g.col_type ? (g.nl % r == 0 && dg.st % r == 0) : (g.L / 16 >= r && g.L % r == 0);
                if (!ok) return DOP_ERR_UNSUPPORTED_SIZE;
            }
    }
    // workspace: [n_lambda fields][h_eff plane][loss partials]
    const size_t npts = (size_t)d.nx * (size_t)d.ny;
    auto align256 = [](size_t x) { return (x + 255) & ~(size_t)255; };
    p->ws_fields = align256(npts * sizeof(float2)) * (size_t)d.n_lambda;
    p->ws_heff_off = p->ws_fields;
    size_t off = p->ws_fields;
    if (d.prefilter_sigma_px > 0.0) off += align256(npts * sizeof(float));
    p->ws_loss_off = off;
    if (d.loss == DOP_LOSS_L2) off += align256((size_t)p->loss_tiles * (size_t)d.n_lambda * sizeof(double));
    if (d.loss == DOP_LOSS_SIMSE) off += align256((size_t)p->loss_tiles * (size_t)d.n_lambda * 4 * sizeof(double));
    p->ws_coef_off = off;
    if (d.loss == DOP_LOSS_SIMSE) off += align256((size_t)d.n_lambda * 4 * sizeof(float));
    p->ws_xpool_off = off;
    if (p->up_lg > 0) off += align256(npts / (size_t)(1 << p->up_lg) * sizeof(float));
    // pre-filter on a coarse / integer layout: A5 writes the fine dL/dh_eff plane here, the filter's adjoint pools it
    p->ws_gfine_off = off;
    if (d.prefilter_sigma_px > 0.0 && (p->up_lg > 0 || d.layout_dtype != DOP_LAYOUT_F32)) off += align256(npts * sizeof(float));
    p->ws_bytes = off;
    return DOP_OK;
}

std::string describe_plan(const dop_plan* p)
{
    std::ostringstream os;
    const dop_plan_desc& d = p->desc;
    os << "grid ny=" << d.ny << " nx=" << d.nx << " n_lambda=" << d.n_lambda
       << " loss=" << (d.loss == DOP_LOSS_L2 ? "L2" : d.loss == DOP_LOSS_SIMSE ? "si-mse+energy" : "none")
       << " upsample=" << (1 << p->up_lg) << " layout=" << (d.layout_dtype == DOP_LAYOUT_U8 ? "u8" : d.layout_dtype == DOP_LAYOUT_U16 ? "u16" : "f32")
       << " prefilter_sigma_px=" << d.prefilter_sigma_px << " pad=" << (p->ap_nx > 0 ? 2 : 1) << " band_limit=" << (d.band_limit ? 1 : 0)
       << " workspace_bytes=" << p->ws_bytes << " loss_tiles=" << p->loss_tiles << "\n";
    for (int a = 0; a < 2; ++a) {
        os << (a == 0 ? "x" : "y") << "-digits:";
        for (const Digit& g : p->ax[a].dig) {
            os << " " << g.L << "(st=" << g.st << ",radix=";
            for (size_t i = 0; i < g.radix.size(); ++i) os << (i ? "." : "") << g.radix[i];
            os << ")";
        }
        os << "\n";
    }
    double total = 0;
    auto dump = [&](const char* tag, const std::vector<PassTmpl>& v) {
        for (const PassTmpl& t : v) {
            PassDesc g{};
            pass_geometry(p, t, &g);
            if (t.cluster)
                os << tag << " x0+x1 L=16x" << g.L << " tile=" << g.nl << "x" << g.L << " row cluster=" << g.n_cgroups;
            else
                os << tag << " " << (t.axis == 0 ? "x" : "y") << t.digit << " L=" << g.L << " tile=" << g.nl << "x" << g.L
                   << (g.col_type ? " col" : " row") << (p->ax[t.axis].dig[(size_t)t.digit].fast ? (g.tma ? " tma" : " pow2") : (g.smooth ? " smooth" : " generic"));
            if (g.tma) os << " stages=" << g.tma;
            os << " ctas=" << g.n_cgroups * g.n_m * g.n_o
               << " smem=" << g.smem_bytes << " B/pt=" << t.bytes_per_point << " [" << t.name << "]\n";
            total += t.bytes_per_point;
        }
    };
    if (p->pre_stencil) {
        os << "pre blur-x rows stencil radius=" << p->blur_radius << " B/pt=8 [gaussian taps along x]\n"
           << "pre blur-y cols stencil radius=" << p->blur_radius << " B/pt=8 [gaussian taps along y]\n";
        total += 16;
    }
    dump("pre", p->pre);
    dump("fwd", p->fwd);
    dump("adj", p->adj);
    dump("pre-adj", p->pre);
    if (p->pre_stencil) {
        os << "pre-adj blur-x rows stencil radius=" << p->blur_radius << " B/pt=8 [gaussian taps along x]\n"
           << "pre-adj blur-y cols stencil radius=" << p->blur_radius << " B/pt=8 [gaussian taps along y]\n";
        total += 16;
    }
    if (!p->hpair_items.empty()) {
        size_t yp = 0;
        for (size_t i = 1; i < p->hpair_items.size(); i += 2) yp += p->hpair_items[i] >= 0;
        os << "H on mirrored tiles: " << p->hpair_items.size() / 2 << " work items per column group (" << yp << " ky-mirror pairs)\n";
    }
    os << "algorithmic_bytes_per_point=" << total << "\n";
    if (d.n_lambda > 1)
        os << "(per wavelength; every wavelength after the first re-reads dL/dh to accumulate: +4 B/point on its last pass)\n";
    return os.str();
}

} // namespace dop
