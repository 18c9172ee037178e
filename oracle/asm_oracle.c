/*
 * oracle/asm_oracle.c -- fp64 CPU oracle for scalar angular-spectrum (ASM) propagation
 * of a DOE height map and its adjoint.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares
 * no code, header, table or constant with the CUDA path under paper_2505_22313_b200/csrc/.
 *
 * What it computes is the plain definition, in the paper's order and notation
 * (PAPER.md = /root/reference/PAPER.md, arxiv 2505.22313, section 3.1):
 *
 *   Eq. (1)  PAPER.md:95-99    Phi_lambda(x,y) = (2 pi / lambda) (n_lambda - 1) h(x,y)
 *   Eq. (2)  PAPER.md:99-102   E_doe = E_in * exp(i Phi)            (E_in == 1, plane wave)
 *   Eq. (3)  PAPER.md:104-108  E_dest = F^-1{ F{E_doe} (x) H_lambda }   (F = 2-D DFT, (x) = Hadamard)
 *   Eq. (4)  PAPER.md:108-112  I_lambda = |E_dest|^2 ; objective sum_lambda L_p(I_lambda)
 *   back-propagation, "backward pass is realized by another ... 2-D FFT" PAPER.md:200
 *   row-column decomposition of the 2-D DFT  PAPER.md:200 (section 4.1)
 *
 * Readings where the paper is silent (repeated in DESIGN.md):
 *   - H_lambda is not written out in the paper; BASELINE.json north_star fixes
 *       H = exp(i 2 pi z sqrt(1/lambda^2 - fx^2 - fy^2)), 0 where the radicand is negative.
 *   - forward DFT kernel exp(-2 pi i k n / N), unnormalised; inverse exp(+...), scaled 1/N.
 *   - f = k/(N pitch) with signed bins (k in [-N/2, N/2)), no fftshift.
 *   - loss L = sum_lambda (1/N) sum_{y,x} (I_lambda - T)^2  (plain L2 stand-in for Eq. 6).
 *   - pre-filter (config 3): h <- Re F^-1{ F{h} * exp(-2 pi^2 sigma^2 ((kx/Nx)^2 + (ky/Ny)^2)) }.
 *
 * The DFT is this file's own: a textbook recursive decimation-in-time Cooley-Tukey for any
 * factorisation (smallest prime factor first, O(p^2) butterfly for a prime factor p), with
 * twiddles taken from a table filled by direct long-double sin/cos of 2 pi k / N (no
 * recurrences).  No FFT library is used.  Everything is double precision.
 *
 * Pins (tests/test_oracle_*.py, run with -m "not gpu"): brute-force O(N^2) DFT, numpy.fft as a
 * library cross-check, plane wave, z = 0 identity / band projector, composition in z, Parseval,
 * analytic Gaussian beam, tilted-plane-wave eigenfunction, Jacobi-Anger phase grating,
 * periodic tiling, <Ax,y> = <x,A^H y>, adjoint gradient vs central finite differences.
 * No function in this file is "parity unpinned".
 *
 * Build:  gcc -O2 -fopenmp -shared -fPIC -o liboracle_asm.so asm_oracle.c -lm   (see build.py)
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

#ifndef M_PIl
#define M_PIl 3.141592653589793238462643383279502884L
#endif

/* ------------------------------------------------------------------------------------------
 * 1-D DFT of any length: X[k] = sum_n x[n] exp(-/+ 2 pi i k n / N)
 * ---------------------------------------------------------------------------------------- */

/* w[k] = exp(-2 pi i k / n), k = 0..n-1, each from a direct long-double sin/cos. */
static void fill_twiddles(int64_t n, cplx *w)
{
    for (int64_t k = 0; k < n; ++k) {
        long double a = 2.0L * M_PIl * (long double)k / (long double)n;
        w[k] = (double)cosl(a) - I * (double)sinl(a);
    }
}

static int64_t smallest_prime_factor(int64_t n)
{
    for (int64_t p = 2; p * p <= n; ++p)
        if (n % p == 0) return p;
    return n;
}

/* table lookup of exp(-/+ 2 pi i j / nfull) for any j >= 0 */
static inline cplx tw(const cplx *w, int64_t nfull, int64_t j, int inverse)
{
    cplx v = w[j % nfull];
    return inverse ? conj(v) : v;
}

/*
 * Decimation in time.  With n = p*m and input index  j = p*j' + r  (r = 0..p-1):
 *   X[k + q m] = sum_{r<p}  W_n^{r (k + q m)}  E_r[k],      E_r = DFT_m of x[p j' + r],
 * for k = 0..m-1, q = 0..p-1  (W_n = exp(-2 pi i / n)).  `w` is the table for length nfull and
 * n divides nfull, so W_n^j = w[j * (nfull/n)].
 * in: n samples `istride` apart.  out: n contiguous.  tmp: scratch of n.
 */
static void dft_rec(int64_t n, const cplx *in, int64_t istride, cplx *out, cplx *tmp,
                    const cplx *w, int64_t nfull, int inverse)
{
    if (n == 1) { out[0] = in[0]; return; }
    const int64_t p = smallest_prime_factor(n);
    const int64_t m = n / p;
    const int64_t ws = nfull / n;            /* W_n^j = w[j*ws] */
    for (int64_t r = 0; r < p; ++r)          /* E_r -> tmp[r*m .. r*m+m) (out is their scratch) */
        dft_rec(m, in + r * istride, istride * p, tmp + r * m, out + r * m, w, nfull, inverse);
    if (p == 2) {                            /* the p = 2 case of the formula, written out */
        for (int64_t k = 0; k < m; ++k) {
            cplx e = tmp[k], o = tw(w, nfull, k * ws, inverse) * tmp[m + k];
            out[k]     = e + o;              /* W_n^{k+m} = -W_n^k */
            out[k + m] = e - o;
        }
        return;
    }
    for (int64_t k = 0; k < m; ++k)
        for (int64_t q = 0; q < p; ++q) {
            cplx s = 0.0;
            for (int64_t r = 0; r < p; ++r)
                s += tw(w, nfull, ((r * (k + q * m)) % n) * ws, inverse) * tmp[r * m + k];
            out[k + q * m] = s;
        }
}

/* In-place 1-D DFT of n samples `stride` apart (gathered to a contiguous line first). */
static void dft_line(int64_t n, cplx *a, int64_t stride, const cplx *w, int inverse,
                     cplx *line, cplx *out, cplx *tmp)
{
    for (int64_t j = 0; j < n; ++j) line[j] = a[j * stride];
    dft_rec(n, line, 1, out, tmp, w, n, inverse);
    for (int64_t j = 0; j < n; ++j) a[j * stride] = out[j];
}

/* out[k] = sum_n in[n] exp(-/+ 2 pi i k n / N); exported so the 1-D routine can be pinned alone */
int oracle_dft1(int64_t n, const cplx *in, cplx *out, int inverse)
{
    if (n < 1) return 1;
    cplx *w = malloc(sizeof(cplx) * n), *tmp = malloc(sizeof(cplx) * n);
    if (!w || !tmp) { free(w); free(tmp); return 2; }
    fill_twiddles(n, w);
    dft_rec(n, in, 1, out, tmp, w, n, inverse);
    free(w); free(tmp);
    return 0;
}

/*
 * 2-D DFT in place, rows then columns:
 *   forward (inverse = 0):  U[ky,kx] = sum_y sum_x a[y,x] exp(-2 pi i (kx x/Nx + ky y/Ny))
 *   inverse (inverse = 1):  a[y,x]  = (1/N) sum sum U[ky,kx] exp(+2 pi i (...)),  N = Ny Nx
 * a is row-major [ny][nx], x contiguous.
 */
int oracle_dft2(int64_t ny, int64_t nx, cplx *a, int inverse)
{
    if (ny < 1 || nx < 1) return 1;
    cplx *wx = malloc(sizeof(cplx) * nx), *wy = malloc(sizeof(cplx) * ny);
    if (!wx || !wy) { free(wx); free(wy); return 2; }
    fill_twiddles(nx, wx);
    fill_twiddles(ny, wy);
    int err = 0;
#pragma omp parallel
    {
        int64_t nmax = nx > ny ? nx : ny;
        cplx *line = malloc(sizeof(cplx) * nmax), *out = malloc(sizeof(cplx) * nmax),
             *tmp = malloc(sizeof(cplx) * nmax);
        if (!line || !out || !tmp) {
#pragma omp atomic write
            err = 2;
        } else {
#pragma omp for schedule(static)
            for (int64_t y = 0; y < ny; ++y)                      /* rows: along x */
                dft_line(nx, a + y * nx, 1, wx, inverse, line, out, tmp);
#pragma omp for schedule(static)
            for (int64_t x = 0; x < nx; ++x)                      /* columns: along y */
                dft_line(ny, a + x, nx, wy, inverse, line, out, tmp);
            if (inverse) {
                const double s = 1.0 / ((double)ny * (double)nx);
#pragma omp for schedule(static)
                for (int64_t i = 0; i < ny * nx; ++i) a[i] *= s;
            }
        }
        free(line); free(out); free(tmp);
    }
    free(wx); free(wy);
    return err;
}

/* signed bin index of k in a length-n DFT: k for k < n/2 (rounded up), k - n otherwise */
static inline double signed_bin(int64_t k, int64_t n) { return (double)(k < (n + 1) / 2 ? k : k - n); }

/* ------------------------------------------------------------------------------------------
 * Pointwise steps O1..O10 (SURVEY.md section 8(c) numbering)
 * ---------------------------------------------------------------------------------------- */

/* O1 + O2, Eq. (1)-(2):  t = (n-1) h / lambda ; Phi = 2 pi t ; u0 = cos Phi + i sin Phi */
void oracle_phase_field(int64_t npts, const double *h, double lambda, double n_refr, cplx *u0)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < npts; ++i) {
        double t = (n_refr - 1.0) * h[i] / lambda;
        double phi = 2.0 * M_PI * t;
        u0[i] = cos(phi) + I * sin(phi);
    }
}

/*
 * O4, the (x) H_lambda of Eq. (3) with north_star's H:
 *   fx = kx/(Nx pitch), fy = ky/(Ny pitch) (signed bins); a = (1/lambda^2 - fx^2) - fy^2;
 *   U *= exp(+i 2 pi z sqrt(a)) if a >= 0, else U = 0.   conj_h != 0 multiplies by conj(H) (adjoint).
 */
void oracle_transfer_multiply(int64_t ny, int64_t nx, cplx *U, double pitch, double lambda,
                              double z, int conj_h)
{
#pragma omp parallel for schedule(static)
    for (int64_t ky = 0; ky < ny; ++ky) {
        double fy = signed_bin(ky, ny) / ((double)ny * pitch);
        for (int64_t kx = 0; kx < nx; ++kx) {
            double fx = signed_bin(kx, nx) / ((double)nx * pitch);
            double a = (1.0 / (lambda * lambda) - fx * fx) - fy * fy;
            if (a >= 0.0) {
                double ph = 2.0 * M_PI * z * sqrt(a);
                cplx H = cos(ph) + I * sin(ph);
                U[ky * nx + kx] *= conj_h ? conj(H) : H;
            } else {
                U[ky * nx + kx] = 0.0;
            }
        }
    }
}

/* the transfer function itself, for tests that want to look at it */
void oracle_transfer_function(int64_t ny, int64_t nx, cplx *H, double pitch, double lambda, double z)
{
    for (int64_t i = 0; i < ny * nx; ++i) H[i] = 1.0;
    oracle_transfer_multiply(ny, nx, H, pitch, lambda, z, 0);
}

/* O0 / O10 spectrum factor: Ghat[ky,kx] = exp(-2 pi^2 sigma^2 ((kx/Nx)^2 + (ky/Ny)^2)), signed bins */
void oracle_gaussian_multiply(int64_t ny, int64_t nx, cplx *U, double sigma_px)
{
#pragma omp parallel for schedule(static)
    for (int64_t ky = 0; ky < ny; ++ky) {
        double vy = signed_bin(ky, ny) / (double)ny;
        for (int64_t kx = 0; kx < nx; ++kx) {
            double vx = signed_bin(kx, nx) / (double)nx;
            U[ky * nx + kx] *= exp(-2.0 * M_PI * M_PI * sigma_px * sigma_px * (vx * vx + vy * vy));
        }
    }
}

/* O6 first half, Eq. (4): I = Re(u)^2 + Im(u)^2 */
void oracle_intensity(int64_t npts, const cplx *u, double *inten)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < npts; ++i)
        inten[i] = creal(u[i]) * creal(u[i]) + cimag(u[i]) * cimag(u[i]);
}

/* O6 second half: (1/N) sum (I - T)^2, Kahan-compensated, one fixed order */
double oracle_l2_loss(int64_t npts, const double *inten, const double *target)
{
    double s = 0.0, c = 0.0;
    for (int64_t i = 0; i < npts; ++i) {
        double d = inten[i] - target[i];
        double y = d * d - c, t = s + y;
        c = (t - s) - y;
        s = t;
    }
    return s / (double)npts;
}

/* O7: g_u = 2 gI u  (gradient w.r.t. (Re u, Im u) packed as a complex), gI = dL/dI */
void oracle_seed(int64_t npts, const cplx *u, const double *gI, cplx *gu)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < npts; ++i) gu[i] = 2.0 * gI[i] * u[i];
}

/* O9: grad += (2 pi (n-1)/lambda) Im( conj(u0) g_u0 ) */
void oracle_phase_adjoint(int64_t npts, const cplx *u0, const cplx *gu0, double lambda,
                          double n_refr, double *grad)
{
    const double c = 2.0 * M_PI * (n_refr - 1.0) / lambda;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < npts; ++i) grad[i] += c * cimag(conj(u0[i]) * gu0[i]);
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
