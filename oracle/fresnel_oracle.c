/*
 * fresnel_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct CPU restatement of the plane-to-plane Fresnel
 * propagation hot path that arXiv 1806.06467 (Douglas & Perrin) accelerates in POPPY.
 * It exists so that the CUDA library in paper_1806_06467_b200/csrc can be checked
 * against something independent.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may load this file's library.  It
 * shares no code, header, table or constant generator with the CUDA path.
 *
 * Arithmetic: double for the field, long double (x87 80-bit) for every phase.
 * No blocking, fusion or reordering beyond what the definitions below state:
 * the fftshift/ifftshift calls are literal array rotations, the chirps are evaluated
 * per pixel from r^2 = x^2 + y^2 (the non-separable route), the 2-D transform is a
 * textbook iterative radix-2 FFT applied to rows and then to columns.
 *
 * Passages followed (PAPER.md line numbers; DESIGN.md lists every reading g1..g20):
 *   - the three bottlenecks FFT / complex exponentials / fftshift:   PAPER.md:77-81 (sec. 2.1)
 *   - quadratic phase factor exp[i(x^2+y^2)/z], Eq. 2:
 *       read as exp(i*pi*(x^2+y^2)/(lambda*z))  (reading g1; thin lens f => z = -f, g2)
 *   - optic phasor A*exp[2*pi*i/lambda * phi], Eq. 3:
 *   - "plane-to-plane angular spectrum propagation ... thin lenses":
 *       transfer function exp(-i*pi*lambda*z*(fx^2+fy^2)) from BASELINE.json:north_star (g4)
 *   - "direct Fresnel" single-FFT propagation, pixelscale changes:
 *   - fftshift puts the origin in the centre of the array:
 *
 * Grid sizes: any N >= 2.  Powers of two go through the radix-2 FFT; every other N (the paper
 * ran N = 2800; App. B gives npix = 1025, :259) through the plain separable
 * O(N^3) DFT of item 2b -- no FFT cleverness for those.
 *
 * Parity pins: every function here is pinned in tests/test_oracle_pins.py (P0..P26 of
 * DESIGN.md) against closed forms / exact identities / brute force.  Nothing is
 * "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_OK 0
#define ORACLE_ERR_INVALID_ARG 1
#define ORACLE_ERR_UNSUPPORTED 2
#define ORACLE_ERR_ALLOC 3

static const long double PI_L = 3.14159265358979323846264338327950288419716939937510L;

static int g_threads = 0; /* 0 = OpenMP default */

void oracle_set_threads(int n) { g_threads = n > 0 ? n : 0; }

int oracle_get_threads(void)
{
#ifdef _OPENMP
    return g_threads > 0 ? g_threads : omp_get_max_threads();
#else
    return 1;
#endif
}

static int nthreads(void) { return oracle_get_threads(); }

static int is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

/* ------------------------------------------------------------------------------------------
 * 1. dft2_naive: the literal O(N^4) double sum  (DESIGN.md oracle item 1)
 *      out[p,q] = sum_j sum_k u[j,k] * exp(sign * 2*pi*i * (j*p + k*q) / N)
 *    sign = -1: unnormalised forward transform;  sign = +1: inverse, scaled by 1/N^2 (g6).
 *    The root exp(sign*2*pi*i*m/N) is taken from direct cosl/sinl of the reduced integer m.
 * ------------------------------------------------------------------------------------------ */
int oracle_dft2_naive(double *u, int N, int sign)
{
    if (!u || N <= 0 || (sign != 1 && sign != -1)) return ORACLE_ERR_INVALID_ARG;
    if (N > 64) return ORACLE_ERR_UNSUPPORTED;
    size_t n2 = (size_t)N * N;
    double *in = (double *)malloc(2 * n2 * sizeof(double));
    double *wr = (double *)malloc(N * sizeof(double));
    double *wi = (double *)malloc(N * sizeof(double));
    if (!in || !wr || !wi) { free(in); free(wr); free(wi); return ORACLE_ERR_ALLOC; }
    memcpy(in, u, 2 * n2 * sizeof(double));
    for (int m = 0; m < N; ++m) {
        long double a = (long double)sign * 2.0L * PI_L * (long double)m / (long double)N;
        wr[m] = (double)cosl(a);
        wi[m] = (double)sinl(a);
    }
#pragma omp parallel for num_threads(nthreads()) schedule(static)
    for (int p = 0; p < N; ++p) {
        for (int q = 0; q < N; ++q) {
            double sr = 0.0, si = 0.0;
            for (int j = 0; j < N; ++j) {
                for (int k = 0; k < N; ++k) {
                    int m = (int)(((long)j * p + (long)k * q) % N);
                    double ar = in[2 * ((size_t)j * N + k)], ai = in[2 * ((size_t)j * N + k) + 1];
                    sr += ar * wr[m] - ai * wi[m];
                    si += ar * wi[m] + ai * wr[m];
                }
            }
            if (sign > 0) { sr /= (double)N * (double)N; si /= (double)N * (double)N; }
            u[2 * ((size_t)p * N + q)] = sr;
            u[2 * ((size_t)p * N + q) + 1] = si;
        }
    }
    free(in); free(wr); free(wi);
    return ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------
 * 2. fft2: own iterative radix-2 (bit reversal + log2 N butterfly stages), rows then columns.
 *    Twiddles come from direct cosl/sinl per index, never from a recurrence.
 * ------------------------------------------------------------------------------------------ */
static void make_twiddles(double *tw, int n, int sign)
{
    for (int k = 0; k < n / 2; ++k) {
        long double a = (long double)sign * 2.0L * PI_L * (long double)k / (long double)n;
        tw[2 * k] = (double)cosl(a);
        tw[2 * k + 1] = (double)sinl(a);
    }
}

static void fft1d_radix2(double *x, int n, const double *tw)
{
    /* bit-reversal permutation */
    for (int i = 1, j = 0; i < n; ++i) {
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) {
            double tr = x[2 * i], ti = x[2 * i + 1];
            x[2 * i] = x[2 * j]; x[2 * i + 1] = x[2 * j + 1];
            x[2 * j] = tr; x[2 * j + 1] = ti;
        }
    }
    for (int len = 2; len <= n; len <<= 1) {
        int half = len >> 1, step = n / len;
        for (int i = 0; i < n; i += len) {
            for (int k = 0; k < half; ++k) {
                double wr = tw[2 * (k * step)], wi = tw[2 * (k * step) + 1];
                double *a = x + 2 * (i + k), *b = x + 2 * (i + k + half);
                double br = b[0] * wr - b[1] * wi;
                double bi = b[0] * wi + b[1] * wr;
                b[0] = a[0] - br; b[1] = a[1] - bi;
                a[0] = a[0] + br; a[1] = a[1] + bi;
            }
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * 2b. dft2_any: the separable DFT for ANY N, written out as its definition -- rows, then columns,
 *     each 1-D transform the plain O(N^2) sum
 *         out[p] = sum_k in[k] * w[(k*p) mod N],   w[m] = exp(sign*2*pi*i*m/N) from direct cosl/sinl,
 *     accumulated in double.  O(N^3) in total; used for every N that is not a power of two
 *     (SURVEY.md sec. 8(f) NEXT-2; PAPER.md:137, :172 N = 2800; :259 npix = 1025).
 * ------------------------------------------------------------------------------------------ */
static void dft1d_plain(const double *in, double *out, int n, int stride, const double *w)
{
    for (int p = 0; p < n; ++p) {
        double sr = 0.0, si = 0.0;
        long m = 0;                                /* (k*p) mod n, advanced by p per term */
        for (int k = 0; k < n; ++k) {
            const double ar = in[2 * (size_t)k * stride], ai = in[2 * (size_t)k * stride + 1];
            sr += ar * w[2 * m] - ai * w[2 * m + 1];
            si += ar * w[2 * m + 1] + ai * w[2 * m];
            m += p;
            if (m >= n) m -= n;
        }
        out[2 * p] = sr;
        out[2 * p + 1] = si;
    }
}

static int dft2_any_core(double *u, int N, int sign, int normalise)
{
    if (!u || N < 1 || (sign != 1 && sign != -1)) return ORACLE_ERR_INVALID_ARG;
    double *w = (double *)malloc(2 * (size_t)N * sizeof(double));
    if (!w) return ORACLE_ERR_ALLOC;
    for (int m = 0; m < N; ++m) {
        long double a = (long double)sign * 2.0L * PI_L * (long double)m / (long double)N;
        w[2 * m] = (double)cosl(a);
        w[2 * m + 1] = (double)sinl(a);
    }
    int fail = 0;
#pragma omp parallel num_threads(nthreads())
    {
        double *line = (double *)malloc(2 * (size_t)N * sizeof(double));
        if (!line) {
#pragma omp atomic write
            fail = 1;
        }
#pragma omp barrier
        if (!fail) {
#pragma omp for schedule(static)
            for (int j = 0; j < N; ++j) {                       /* rows */
                dft1d_plain(u + 2 * (size_t)j * N, line, N, 1, w);
                memcpy(u + 2 * (size_t)j * N, line, 2 * (size_t)N * sizeof(double));
            }
#pragma omp for schedule(static)
            for (int k = 0; k < N; ++k) {                       /* columns */
                dft1d_plain(u + 2 * (size_t)k, line, N, N, w);
                for (int j = 0; j < N; ++j) {
                    u[2 * ((size_t)j * N + k)] = line[2 * j];
                    u[2 * ((size_t)j * N + k) + 1] = line[2 * j + 1];
                }
            }
            if (normalise) {
                double sc = 1.0 / ((double)N * (double)N);
#pragma omp for schedule(static)
                for (int j = 0; j < N; ++j)
                    for (int k = 0; k < 2 * N; ++k) u[2 * (size_t)j * N + k] *= sc;
            }
        }
        free(line);
    }
    free(w);
    return fail ? ORACLE_ERR_ALLOC : ORACLE_OK;
}

/* forward (sign=-1) unnormalised; inverse (sign=+1) scaled by 1/N^2; any N >= 1. */
int oracle_dft2_any(double *u, int N, int sign) { return dft2_any_core(u, N, sign, sign > 0); }

/* normalise != 0: multiply by 1/N^2 (only meaningful with sign = +1). */
static int fft2_core(double *u, int N, int sign, int normalise)
{
    if (!u || (sign != 1 && sign != -1)) return ORACLE_ERR_INVALID_ARG;
    if (N < 2) return ORACLE_ERR_UNSUPPORTED;
    if (!is_pow2(N)) return dft2_any_core(u, N, sign, normalise);
    double *tw = (double *)malloc((size_t)N * sizeof(double));
    if (!tw) return ORACLE_ERR_ALLOC;
    make_twiddles(tw, N, sign);
    int fail = 0;
#pragma omp parallel num_threads(nthreads())
    {
        double *col = (double *)malloc(2 * (size_t)N * sizeof(double));
        if (!col) {
#pragma omp atomic write
            fail = 1;
        }
#pragma omp barrier
        if (!fail) {
#pragma omp for schedule(static)
            for (int j = 0; j < N; ++j) fft1d_radix2(u + 2 * (size_t)j * N, N, tw);
#pragma omp for schedule(static)
            for (int k = 0; k < N; ++k) {
                for (int j = 0; j < N; ++j) {
                    col[2 * j] = u[2 * ((size_t)j * N + k)];
                    col[2 * j + 1] = u[2 * ((size_t)j * N + k) + 1];
                }
                fft1d_radix2(col, N, tw);
                for (int j = 0; j < N; ++j) {
                    u[2 * ((size_t)j * N + k)] = col[2 * j];
                    u[2 * ((size_t)j * N + k) + 1] = col[2 * j + 1];
                }
            }
            if (normalise) {
                double s = 1.0 / ((double)N * (double)N);
#pragma omp for schedule(static)
                for (int j = 0; j < N; ++j)
                    for (int k = 0; k < 2 * N; ++k) u[2 * (size_t)j * N + k] *= s;
            }
        }
        free(col);
    }
    free(tw);
    return fail ? ORACLE_ERR_ALLOC : ORACLE_OK;
}

/* forward (sign=-1) unnormalised; inverse (sign=+1) scaled by 1/N^2 (reading g6). */
int oracle_fft2(double *u, int N, int sign) { return fft2_core(u, N, sign, sign > 0); }

/* ------------------------------------------------------------------------------------------
 * literal shifts: fftshift(x)[i] = x[(i - N/2) mod N], ifftshift(x)[i] = x[(i + N/2) mod N]
 * ------------------------------------------------------------------------------------------ */
static int roll2d(double *u, int N, int s)
{
    size_t n2 = (size_t)N * N;
    double *t = (double *)malloc(2 * n2 * sizeof(double));
    if (!t) return ORACLE_ERR_ALLOC;
    memcpy(t, u, 2 * n2 * sizeof(double));
    s = ((s % N) + N) % N;
#pragma omp parallel for num_threads(nthreads()) schedule(static)
    for (int j = 0; j < N; ++j) {
        int jj = (j + s) % N;
        for (int k = 0; k < N; ++k) {
            int kk = (k + s) % N;
            u[2 * ((size_t)jj * N + kk)] = t[2 * ((size_t)j * N + k)];
            u[2 * ((size_t)jj * N + kk) + 1] = t[2 * ((size_t)j * N + k) + 1];
        }
    }
    free(t);
    return ORACLE_OK;
}

int oracle_fftshift(double *u, int N) { return (!u || N <= 0) ? ORACLE_ERR_INVALID_ARG : roll2d(u, N, N / 2); }
int oracle_ifftshift(double *u, int N) { return (!u || N <= 0) ? ORACLE_ERR_INVALID_ARG : roll2d(u, N, -(N / 2)); }

/* fft2d as the ABI exposes it: forward unnormalised, inverse x 1/N^2;
 * centered != 0  =>  fftshift o fft2 o ifftshift  (origin on pixel N/2, reading g8). */
int oracle_fft2d(double *u, int N, int direction, int centered)
{
    int sign = direction > 0 ? -1 : +1; /* FRESNEL_FORWARD=+1 uses kernel exp(-...), INVERSE=-1 uses exp(+...) */
    if (direction != 1 && direction != -1) return ORACLE_ERR_INVALID_ARG;
    int rc;
    if (centered && (rc = oracle_ifftshift(u, N)) != ORACLE_OK) return rc;
    if ((rc = oracle_fft2(u, N, sign)) != ORACLE_OK) return rc;
    if (centered && (rc = oracle_fftshift(u, N)) != ORACLE_OK) return rc;
    return ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------
 * 3. apply_qpf (Eq. 2, reading g1):
 *      u[j,k] *= exp(i*pi*(x_k^2 + y_j^2)/(lambda*z)),  x_k = (k-N/2)*dx, y_j = (j-N/2)*dx
 *    per pixel, r^2 and the phase in long double.  A thin lens of focal length f is z = -f (g2).
 * ------------------------------------------------------------------------------------------ */
int oracle_apply_qpf(double *u, int N, double dx, double lambda, double z)
{
    if (!u || N <= 0 || !(dx > 0) || !(lambda > 0) || !isfinite(z) || z == 0.0) return ORACLE_ERR_INVALID_ARG;
    long double ldx = dx, ll = lambda, lz = z;
#pragma omp parallel for num_threads(nthreads()) schedule(static)
    for (int j = 0; j < N; ++j) {
        long double y = (long double)(j - N / 2) * ldx;
        for (int k = 0; k < N; ++k) {
            long double x = (long double)(k - N / 2) * ldx;
            long double r2 = x * x + y * y;
            long double th = PI_L * r2 / (ll * lz);
            double c = (double)cosl(th), s = (double)sinl(th);
            double *p = u + 2 * ((size_t)j * N + k);
            double re = p[0] * c - p[1] * s, im = p[0] * s + p[1] * c;
            p[0] = re; p[1] = im;
        }
    }
    return ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------
 * 4. apply_mask (Eq. 3, reading g3):  u *= A * exp(i*2*pi*OPD/lambda)
 *    amp and/or opd may be NULL (A = 1, OPD = 0).
 * ------------------------------------------------------------------------------------------ */
int oracle_apply_mask(double *u, int N, const double *amp, const double *opd, double lambda)
{
    if (!u || N <= 0 || !(lambda > 0)) return ORACLE_ERR_INVALID_ARG;
    long double ll = lambda;
#pragma omp parallel for num_threads(nthreads()) schedule(static)
    for (int j = 0; j < N; ++j) {
        for (int k = 0; k < N; ++k) {
            size_t i = (size_t)j * N + k;
            double a = amp ? amp[i] : 1.0;
            double c = 1.0, s = 0.0;
            if (opd) {
                long double th = 2.0L * PI_L * (long double)opd[i] / ll;
                c = (double)cosl(th); s = (double)sinl(th);
            }
            double re = u[2 * i] * c - u[2 * i + 1] * s, im = u[2 * i] * s + u[2 * i + 1] * c;
            u[2 * i] = a * re; u[2 * i + 1] = a * im;
        }
    }
    return ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------
 * 5. propagate_as: the literal sequence  ifftshift -> fft2(-) -> x H -> fft2(+) -> fftshift
 *      H[p,q] = exp(-i*pi*lambda*z*(f_q^2 + f_p^2)),  f in FFT order: f_q = q/(N dx) for q < (N+1)/2
 *      (= N/2 for even N), (q-N)/(N dx) otherwise.  No piston exp(ikz) (g5).  z = 0 is the identity (g11).
 *    ("plane-to-plane angular spectrum propagation"; BASELINE.json:north_star)
 * ------------------------------------------------------------------------------------------ */
int oracle_propagate_as(double *u, int N, double dx, double lambda, double z)
{
    if (!u || N <= 0 || !(dx > 0) || !(lambda > 0) || !isfinite(z)) return ORACLE_ERR_INVALID_ARG;
    int rc;
    if ((rc = oracle_ifftshift(u, N)) != ORACLE_OK) return rc;
    if ((rc = oracle_fft2(u, N, -1)) != ORACLE_OK) return rc;
    long double ldx = dx, ll = lambda, lz = z;
#pragma omp parallel for num_threads(nthreads()) schedule(static)
    for (int p = 0; p < N; ++p) {
        long double fp = (long double)(p < (N + 1) / 2 ? p : p - N) / ((long double)N * ldx);
        for (int q = 0; q < N; ++q) {
            long double fq = (long double)(q < (N + 1) / 2 ? q : q - N) / ((long double)N * ldx);
            long double th = -PI_L * ll * lz * (fq * fq + fp * fp);
            double c = (double)cosl(th), s = (double)sinl(th);
            double *e = u + 2 * ((size_t)p * N + q);
            double re = e[0] * c - e[1] * s, im = e[0] * s + e[1] * c;
            e[0] = re; e[1] = im;
        }
    }
    if ((rc = oracle_fft2(u, N, +1)) != ORACLE_OK) return rc;
    if ((rc = oracle_fftshift(u, N)) != ORACLE_OK) return rc;
    return ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------
 * 6. propagate_direct (single-FFT Fresnel; readings g7, g10):
 *      u *= Q_dx(z);  centred transform by literal ifftshift / fft2 / fftshift
 *      (forward kernel if z > 0, unnormalised inverse kernel, i.e. N^2 * ifft2, if z < 0);
 *      u *= dx^2/(i*lambda*z);   dx' = lambda*|z|/(N*dx);   u *= Q_dx'(z).
 * ------------------------------------------------------------------------------------------ */
int oracle_propagate_direct(double *u, int N, double *dx_inout, double lambda, double z)
{
    if (!u || !dx_inout || N <= 0 || !(*dx_inout > 0) || !(lambda > 0) || !isfinite(z) || z == 0.0)
        return ORACLE_ERR_INVALID_ARG;
    double dx = *dx_inout;
    int rc;
    if ((rc = oracle_apply_qpf(u, N, dx, lambda, z)) != ORACLE_OK) return rc;
    if ((rc = oracle_ifftshift(u, N)) != ORACLE_OK) return rc;
    if ((rc = fft2_core(u, N, z > 0 ? -1 : +1, 0)) != ORACLE_OK) return rc;
    if ((rc = oracle_fftshift(u, N)) != ORACLE_OK) return rc;
    /* dx^2/(i lambda z) = -i * dx^2/(lambda z) */
    long double g = (long double)dx * (long double)dx / ((long double)lambda * (long double)z);
    double gd = (double)g;
#pragma omp parallel for num_threads(nthreads()) schedule(static)
    for (int j = 0; j < N; ++j) {
        for (int k = 0; k < N; ++k) {
            double *e = u + 2 * ((size_t)j * N + k);
            double re = e[1] * gd, im = -e[0] * gd; /* (re + i im) * (-i g) = im*g - i re*g */
            e[0] = re; e[1] = im;
        }
    }
    long double dxo = (long double)lambda * fabsl((long double)z) / ((long double)N * (long double)dx);
    double dx_out = (double)dxo;
    if ((rc = oracle_apply_qpf(u, N, dx_out, lambda, z)) != ORACLE_OK) return rc;
    *dx_inout = dx_out;
    return ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------
 * fused surface = thin lens f  (QPF with z = -f; f = +-INFINITY => no lens), then the optic
 * phasor, then angular-spectrum propagation by z; applied literally one after the other
 * ("add_optic(lens, distance=...)").
 * ------------------------------------------------------------------------------------------ */
int oracle_surface_as(double *u, int N, double dx, double lambda, double f,
                      const double *amp, const double *opd, double z)
{
    int rc;
    if (isnan(f) || f == 0.0) return ORACLE_ERR_INVALID_ARG;
    if (isfinite(f) && (rc = oracle_apply_qpf(u, N, dx, lambda, -f)) != ORACLE_OK) return rc;
    if ((amp || opd) && (rc = oracle_apply_mask(u, N, amp, opd, lambda)) != ORACLE_OK) return rc;
    return oracle_propagate_as(u, N, dx, lambda, z);
}

/* ---- broadband (polychromatic) image: incoherent sum over wavelengths ------------------------------
 * "calculations must be repeated for all of the wavelengths" (one process per wavelength,
 * PAPER.md:63): a broadband image is the weighted sum of the monochromatic intensities,
 *     image[j][k] += w * |u[j][k]|^2        (one call per wavelength).
 * u: N x N interleaved complex, image: N x N real, both host. */
int oracle_accumulate_intensity(const double *u, int N, double w, double *image)
{
    if (!u || !image || N <= 0) return ORACLE_ERR_INVALID_ARG;
    for (long i = 0; i < (long)N * N; ++i) {
        const double re = u[2 * i], im = u[2 * i + 1];
        image[i] += w * (re * re + im * im);
    }
    return ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------
 * train of surfaces with a per-surface choice of propagator (reduced).
 * The paper's system is "add_optic(optic, distance=...)" repeated and POPPY picks
 * plane-to-plane or single-FFT propagation from a Gaussian pilot beam (Lawrence Eq. 82-89),
 * which the paper does not print.  Reading g13b: with method AUTO the choice is the sampling
 * criterion of the two discrete operators -- the angular-spectrum chirp exp(-i pi lambda z f^2) is
 * sampled without aliasing up to z_c = N dx^2 / lambda, the direct-Fresnel input chirp from z_c on --
 * so |z| < z_c takes the angular spectrum (pixel pitch kept), |z| >= z_c the direct transform
 * (pixel pitch becomes lambda |z| / (N dx)); z == 0 propagates nothing.
 * One wavefront; surfaces applied literally one after the other.
 *   f[s], z[s], method[s] (0 = angular spectrum, 1 = direct, 2 = auto); amp[s], opd[s] may be NULL.
 *   used[s] (optional) receives 0 / 1 / -1 (no propagation).  *dx_inout is the running pixel pitch.
 * ------------------------------------------------------------------------------------------ */
int oracle_system_run(double *u, int N, double *dx_inout, double lambda, int nsurf, const double *f,
                      const double *const *amp, const double *const *opd, const double *z,
                      const int *method, int *used)
{
    if (!u || !dx_inout || !f || !z || !method || nsurf < 0) return ORACLE_ERR_INVALID_ARG;
    int rc;
    for (int s = 0; s < nsurf; ++s) {
        const double dx = *dx_inout;
        if (isnan(f[s]) || f[s] == 0.0 || !isfinite(z[s])) return ORACLE_ERR_INVALID_ARG;
        if (isfinite(f[s]) && (rc = oracle_apply_qpf(u, N, dx, lambda, -f[s])) != ORACLE_OK) return rc;
        const double *a = amp ? amp[s] : NULL, *o = opd ? opd[s] : NULL;
        if ((a || o) && (rc = oracle_apply_mask(u, N, a, o, lambda)) != ORACLE_OK) return rc;
        int m = method[s];
        if (m < 0 || m > 2) return ORACLE_ERR_INVALID_ARG;
        if (z[s] == 0.0) { if (used) used[s] = -1; continue; }
        if (m == 2) {
            const long double zc = (long double)N * (long double)dx * (long double)dx / (long double)lambda;
            m = (fabsl((long double)z[s]) < zc) ? 0 : 1;
        }
        if (m == 0) rc = oracle_propagate_as(u, N, dx, lambda, z[s]);
        else        rc = oracle_propagate_direct(u, N, dx_inout, lambda, z[s]);
        if (rc != ORACLE_OK) return rc;
        if (used) used[s] = m;
    }
    return ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------
 * Gaussian pilot-beam propagation ("following the methods in Ref. [6,
 * Equation 82-89]" -- Lawrence 1992, which the paper does not print; the conventions below are DESIGN.md's
 * reading g21, restated from textbook Gaussian-beam optics).
 *
 * A Gaussian "pilot" beam rides along with the wavefront: waist radius w0 at position zw (so zR = pi w0^2/lambda),
 * current position z; complex beam parameter q = (z - zw) + i zR, 1/q = 1/R - i lambda/(pi w^2).  It decides on what
 * REFERENCE SURFACE the array is kept: within rf*zR of the pilot waist a plane, outside it a sphere centred on the
 * pilot waist, radius Rref = z - zw.  The stored array is the true field with the reference curvature removed,
 *     U_true = U_stored * exp(i pi r^2 / (lambda Rref))          (planar: 1/Rref = 0),
 * so the quadratic phases that are hard to sample far from focus are never put on the grid.  Propagators:
 *   PTP(dz)  plane -> plane: angular spectrum (item 5), pixel pitch kept;
 *   WTS(dz)  waist (plane) -> sphere of radius dz: direct Fresnel (item 6) WITHOUT its output chirp,
 *                U_stored' = dx^2/(i lambda dz) * CFT(Q_dx(dz) U),   dx' = lambda |dz| / (N dx);
 *   STW(dz)  sphere of radius -dz -> waist (plane): direct Fresnel WITHOUT its input chirp (it cancels the
 *                reference curvature exactly),  U' = dx^2/(i lambda dz) * Q_dx'(dz) * CFT(U_stored).
 * A propagation from z1 to z2 = z1 + dz:  inside->inside PTP(dz);  inside->outside PTP(zw - z1) then WTS(z2 - zw);
 * outside->inside STW(zw - z1) then PTP(z2 - zw);  outside->outside STW(zw - z1) then WTS(z2 - zw)   (a leg of zero
 * length is skipped).  "inside" means |z - zw| < rf * zR.
 * A thin lens f at z multiplies the TRUE field by exp(-i pi r^2/(lambda f)) (g2) and maps the pilot beam by the ABCD
 * rule 1/q' = 1/q - 1/f:  zw' = z - Re q', zR' = Im q', w0' = sqrt(lambda zR'/pi); the new reference is planar if
 * |z - zw'| < rf zR', else the sphere Rref' = z - zw'.  The stored array takes the residual chirp
 *     U_stored' = U_stored * exp(i pi r^2/lambda * (1/Rref - 1/f - 1/Rref')).
 * Masks multiply the stored array (they do not touch the reference).
 *
 * state[0..4] = {w0, zw, z, Rref (INFINITY when planar), unused}; dx_inout as elsewhere.  One wavefront.
 * legs_used (optional, 2 ints per surface): 0 none, 1 PTP, 2 WTS, 3 STW for the two legs of each propagation.
 * ------------------------------------------------------------------------------------------ */
static int centred_transform(double *u, int N, int forward_kernel)
{
    int rc;
    if ((rc = oracle_ifftshift(u, N)) != ORACLE_OK) return rc;
    if ((rc = fft2_core(u, N, forward_kernel ? -1 : +1, 0)) != ORACLE_OK) return rc;
    return oracle_fftshift(u, N);
}

static void scale_minus_i_g(double *u, int N, double g)      /* u *= -i*g  =  dx^2/(i lambda dz) with g = dx^2/(lambda dz) */
{
#pragma omp parallel for num_threads(nthreads()) schedule(static)
    for (long i = 0; i < (long)N * N; ++i) {
        double re = u[2 * i + 1] * g, im = -u[2 * i] * g;
        u[2 * i] = re; u[2 * i + 1] = im;
    }
}

/* waist -> spherical: chirp, centred transform, scale; no output chirp */
int oracle_wts(double *u, int N, double *dx_inout, double lambda, double dz)
{
    if (!u || !dx_inout || N <= 0 || !(*dx_inout > 0) || !(lambda > 0) || !isfinite(dz) || dz == 0.0) return ORACLE_ERR_INVALID_ARG;
    const double dx = *dx_inout;
    int rc;
    if ((rc = oracle_apply_qpf(u, N, dx, lambda, dz)) != ORACLE_OK) return rc;
    if ((rc = centred_transform(u, N, dz > 0)) != ORACLE_OK) return rc;
    scale_minus_i_g(u, N, (double)((long double)dx * (long double)dx / ((long double)lambda * (long double)dz)));
    *dx_inout = (double)((long double)lambda * fabsl((long double)dz) / ((long double)N * (long double)dx));
    return ORACLE_OK;
}

/* spherical -> waist: centred transform, scale, output chirp at the new pitch; no input chirp */
int oracle_stw(double *u, int N, double *dx_inout, double lambda, double dz)
{
    if (!u || !dx_inout || N <= 0 || !(*dx_inout > 0) || !(lambda > 0) || !isfinite(dz) || dz == 0.0) return ORACLE_ERR_INVALID_ARG;
    const double dx = *dx_inout;
    int rc;
    if ((rc = centred_transform(u, N, dz > 0)) != ORACLE_OK) return rc;
    scale_minus_i_g(u, N, (double)((long double)dx * (long double)dx / ((long double)lambda * (long double)dz)));
    const double dx_out = (double)((long double)lambda * fabsl((long double)dz) / ((long double)N * (long double)dx));
    if ((rc = oracle_apply_qpf(u, N, dx_out, lambda, dz)) != ORACLE_OK) return rc;
    *dx_inout = dx_out;
    return ORACLE_OK;
}

/* u *= exp(i pi r^2 kappa / lambda), kappa in 1/m (a QPF with 1/z = kappa); kappa == 0: nothing */
static int apply_curvature(double *u, int N, double dx, double lambda, long double kappa)
{
    if (kappa == 0.0L) return ORACLE_OK;
    return oracle_apply_qpf(u, N, dx, lambda, (double)(1.0L / kappa));
}

int oracle_system_run_pilot(double *u, int N, double *dx_inout, double lambda, int nsurf, const double *f,
                            const double *const *amp, const double *const *opd, const double *z,
                            double rayleigh_factor, double *state, int *legs_used)
{
    if (!u || !dx_inout || !state || nsurf < 0 || (nsurf > 0 && (!f || !z))) return ORACLE_ERR_INVALID_ARG;
    if (!(state[0] > 0) || !(rayleigh_factor > 0) || !(lambda > 0) || !(*dx_inout > 0)) return ORACLE_ERR_INVALID_ARG;
    long double w0 = state[0], zw = state[1], zc = state[2];
    long double inv_rref = isfinite(state[3]) ? 1.0L / (long double)state[3] : 0.0L;
    const long double rf = rayleigh_factor, lam = lambda;
    int rc;
    for (int s = 0; s < nsurf; ++s) {
        if (isnan(f[s]) || f[s] == 0.0 || !isfinite(z[s])) return ORACLE_ERR_INVALID_ARG;
        /* (1) thin lens: ABCD on the pilot beam, residual chirp on the array */
        if (isfinite(f[s])) {
            const long double zR = PI_L * w0 * w0 / lam;
            const long double qr = zc - zw, qi = zR;                 /* q = qr + i qi */
            const long double den = qr * qr + qi * qi;
            const long double ir = qr / den - 1.0L / (long double)f[s], ii = -qi / den;   /* 1/q' */
            const long double d2 = ir * ir + ii * ii;
            const long double q2r = ir / d2, q2i = -ii / d2;          /* q' */
            const long double zw2 = zc - q2r, zR2 = q2i;
            const long double inv_rref2 = (fabsl(zc - zw2) < rf * zR2) ? 0.0L : 1.0L / (zc - zw2);
            const long double kappa = inv_rref - 1.0L / (long double)f[s] - inv_rref2;
            if ((rc = apply_curvature(u, N, *dx_inout, lambda, kappa)) != ORACLE_OK) return rc;
            zw = zw2;
            w0 = sqrtl(lam * zR2 / PI_L);
            inv_rref = inv_rref2;
        }
        /* (2) optic phasor on the stored array */
        const double *a = amp ? amp[s] : NULL, *o = opd ? opd[s] : NULL;
        if ((a || o) && (rc = oracle_apply_mask(u, N, a, o, lambda)) != ORACLE_OK) return rc;
        /* (3) propagation by z[s] */
        int leg[2] = {0, 0};
        if (z[s] != 0.0) {
            const long double zR = PI_L * w0 * w0 / lam;
            const long double z1 = zc, z2 = zc + (long double)z[s];
            const int in1 = inv_rref == 0.0L;                          /* the reference says where we are */
            const int in2 = fabsl(z2 - zw) < rf * zR;
            if (in1 && in2) {
                if ((rc = oracle_propagate_as(u, N, *dx_inout, lambda, z[s])) != ORACLE_OK) return rc;
                leg[0] = 1;
            } else {
                const double d1 = (double)(zw - z1), d2 = (double)(z2 - zw);
                if (d1 != 0.0) {
                    if (in1) { rc = oracle_propagate_as(u, N, *dx_inout, lambda, d1); leg[0] = 1; }
                    else     { rc = oracle_stw(u, N, dx_inout, lambda, d1); leg[0] = 3; }
                    if (rc != ORACLE_OK) return rc;
                }
                if (d2 != 0.0) {
                    if (in2) { rc = oracle_propagate_as(u, N, *dx_inout, lambda, d2); leg[1] = 1; }
                    else     { rc = oracle_wts(u, N, dx_inout, lambda, d2); leg[1] = 2; }
                    if (rc != ORACLE_OK) return rc;
                }
            }
            zc = z2;
            inv_rref = in2 ? 0.0L : 1.0L / (z2 - zw);
        }
        if (legs_used) { legs_used[2 * s] = leg[0]; legs_used[2 * s + 1] = leg[1]; }
    }
    state[0] = (double)w0; state[1] = (double)zw; state[2] = (double)zc;
    state[3] = inv_rref == 0.0L ? INFINITY : (double)(1.0L / inv_rref);
    return ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------
 * Fraunhofer propagation by a matrix Fourier transform ("discrete matrix
 * Fourier transforms of modest sized arrays", :119; reading g22).
 *
 * The field in the focal plane of a lens of focal length f, sampled on ANY output grid (nb x nb pixels of pitch
 * dx_out, origin on pixel nb/2), from an na x na input of pitch dx_in (origin on pixel na/2):
 *     V[p,q] = s * sum_j sum_k  U[j,k] * exp(-+ 2 pi i (x_k x'_q + y_j y'_p) / (lambda f)),    s = dx_in^2 / (+- i lambda f)
 * upper signs for direction = +1 (forward kernel), lower for -1 (the inverse pair: with dx_out = lambda f/(na dx_in)
 * and nb = na, inverse o forward = identity).  It is the Fourier core of the direct Fresnel transform (item 6) freed
 * from the FFT's sampling: at dx_out = lambda f/(na dx_in), nb = na, it equals s * fftshift(fft2(ifftshift(U))).
 * Written out as the definition: the two kernel matrices E_x[q,k], E_y[p,j] from per-entry long-double phases,
 * then the two plain matrix products  T = U E_x^T,  V = s E_y T  accumulated in double (O(na^2 nb + na nb^2)).
 * u: na x na interleaved complex, v: nb x nb interleaved complex (written), both host.
 * ------------------------------------------------------------------------------------------ */
int oracle_mft(const double *u, int na, double dx_in, double *v, int nb, double dx_out, double lambda, double f, int direction)
{
    if (!u || !v || na <= 0 || nb <= 0 || !(dx_in > 0) || !(dx_out > 0) || !(lambda > 0) || !isfinite(f) || f == 0.0) return ORACLE_ERR_INVALID_ARG;
    if (direction != 1 && direction != -1) return ORACLE_ERR_INVALID_ARG;
    double *e = (double *)malloc(2 * (size_t)nb * na * sizeof(double));      /* E[q,k] = exp(-+ 2 pi i x_k x'_q/(lambda f)) (same for x and y) */
    double *t = (double *)malloc(2 * (size_t)na * nb * sizeof(double));      /* T[j,q] */
    if (!e || !t) { free(e); free(t); return ORACLE_ERR_ALLOC; }
    const long double sgn = direction > 0 ? -1.0L : 1.0L;
#pragma omp parallel for num_threads(nthreads()) schedule(static)
    for (int q = 0; q < nb; ++q) {
        const long double xq = (long double)(q - nb / 2) * (long double)dx_out;
        for (int k = 0; k < na; ++k) {
            const long double xk = (long double)(k - na / 2) * (long double)dx_in;
            const long double th = sgn * 2.0L * PI_L * xk * xq / ((long double)lambda * (long double)f);
            e[2 * ((size_t)q * na + k)] = (double)cosl(th);
            e[2 * ((size_t)q * na + k) + 1] = (double)sinl(th);
        }
    }
#pragma omp parallel for num_threads(nthreads()) schedule(static)
    for (int j = 0; j < na; ++j)                                             /* T[j,q] = sum_k U[j,k] E[q,k] */
        for (int q = 0; q < nb; ++q) {
            double sr = 0.0, si = 0.0;
            for (int k = 0; k < na; ++k) {
                const double ar = u[2 * ((size_t)j * na + k)], ai = u[2 * ((size_t)j * na + k) + 1];
                const double br = e[2 * ((size_t)q * na + k)], bi = e[2 * ((size_t)q * na + k) + 1];
                sr += ar * br - ai * bi;
                si += ar * bi + ai * br;
            }
            t[2 * ((size_t)j * nb + q)] = sr;
            t[2 * ((size_t)j * nb + q) + 1] = si;
        }
    /* s = dx^2/(+- i lambda f) = -+ i g,  g = dx^2/(lambda f) */
    const double g = (double)((long double)dx_in * (long double)dx_in / ((long double)lambda * (long double)f));
#pragma omp parallel for num_threads(nthreads()) schedule(static)
    for (int p = 0; p < nb; ++p)                                             /* V[p,q] = s sum_j E[p,j] T[j,q] */
        for (int q = 0; q < nb; ++q) {
            double sr = 0.0, si = 0.0;
            for (int j = 0; j < na; ++j) {
                const double ar = e[2 * ((size_t)p * na + j)], ai = e[2 * ((size_t)p * na + j) + 1];
                const double br = t[2 * ((size_t)j * nb + q)], bi = t[2 * ((size_t)j * nb + q) + 1];
                sr += ar * br - ai * bi;
                si += ar * bi + ai * br;
            }
            if (direction > 0) { v[2 * ((size_t)p * nb + q)] = si * g;  v[2 * ((size_t)p * nb + q) + 1] = -sr * g; }   /* x (-i g) */
            else               { v[2 * ((size_t)p * nb + q)] = -si * g; v[2 * ((size_t)p * nb + q) + 1] = sr * g; }    /* x (+i g) */
        }
    free(e); free(t);
    return ORACLE_OK;
}
