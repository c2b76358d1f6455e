// tables.cuh -- the 1-D tables every pass multiplies by.
//
// (1) FFT twiddles W_{Ns*R}^{t*k}: built on the HOST in long double from direct cosl/sinl per entry,
//     rounded once to the plan's precision, uploaded at plan creation.
// (2) Chirp tables: the quadratic phase factor exp(i pi (x^2+y^2)/(lambda z)) (Eq. 2)
//     and the angular-spectrum transfer function exp(-i pi lambda z (fx^2+fy^2))
//     (BASELINE.json:north_star) are outer products of ONE 1-D chirp with itself, so a surface needs
//     2N sincos evaluations instead of N^2 -- this removes the paper's bottleneck #2 ("complex
//     exponentials") from the per-pixel path.  An entry is
//         tab[b][n] = amp_b * exp(2 pi i (c_b * m(n)^2 + phase0_b)) * ramp(n)
//     with ramp(n) = exp(+-2 pi i (N/2) n / N) when alt = +-1 (the shift bookkeeping of a centred transform:
//     (-1)^n for even N, a phase ramp with the exact rational (h n mod N)/N for odd N), else 1;
//     m(n) = n - N/2 (centred pixel index) or the FFT-order frequency index, and c_b given in
//     TURNS per index^2 as a double-double (hi, lo) computed on the host in long double.  The phase
//     m^2*c reaches 1e3..1e5 turns; it is evaluated with an error-free product (fma) and reduced
//     to [-1/2, 1/2] turns before sincospi, so the table is good to ~1e-16 whatever its size
//     (computing the phase in plain double would already cost ~1e-11).
#pragma once
#include <cuda_runtime.h>
#include "fft_core.cuh"

namespace fresnel {

constexpr int kBuildMaxBatch = 16;   // batch elements per builder launch (kernel-parameter budget: 4 KB)
constexpr int kBuildMaxTables = 6;   // tables per builder launch (a fused train builds all its tables up front)

struct ChirpSpec {
    double c_hi, c_lo;   // turns per index^2 (double-double)
    double amp;          // real amplitude
    double phase0;       // constant phase in turns
};

struct TableBuild {
    void *out;           // [batch][N] complex of the plan's dtype
    int index_mode;      // 0: m = n - N/2;  1: m = FFT-order index (n < (N+1)/2 ? n : n - N)
    int alt_sign;        // +-1: multiply by exp(+-2 pi i (N/2) n / N)  (= (-1)^n for even N)
    ChirpSpec spec[kBuildMaxBatch];
};

struct BuildArgs {
    int N, b0, nb, ntab, is_double;
    double *scal_out;               // [batch] per-batch scalar (1/lambda) or nullptr
    double scal[kBuildMaxBatch];
    TableBuild t[kBuildMaxTables];
};

__global__ void build_tables_kernel(const __grid_constant__ BuildArgs a)
{
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    const int bl = blockIdx.y;            // batch index within this launch
    const int ti = blockIdx.z;
    if (ti == 0 && n == 0 && a.scal_out != nullptr) a.scal_out[a.b0 + bl] = a.scal[bl];
    if (n >= a.N || ti >= a.ntab) return;
    const TableBuild &t = a.t[ti];
    const ChirpSpec sp = t.spec[bl];
    const int m = t.index_mode == 0 ? n - a.N / 2 : (n < (a.N + 1) / 2 ? n : n - a.N);
    const double p = (double)m * (double)m;             // exact (|m| <= 8192)
    const double hi = p * sp.c_hi;
    const double err = fma(p, sp.c_hi, -hi);            // exact error of the product
    const double lo = fma(p, sp.c_lo, err);
    const double k = rint(hi);
    double r = (hi - k) + lo;                           // hi - k is exact
    r += sp.phase0;
    const bool odd_grid = (a.N & 1) != 0;
    if (t.alt_sign != 0 && odd_grid) {                  // phase ramp of an odd grid: (h n mod N) / N turns, exact rational
        const long long q = ((long long)(a.N / 2) * n) % a.N;
        const double fr = (double)q / (double)a.N;
        r += t.alt_sign > 0 ? fr : -fr;
    }
    double s, c;
    sincospi(2.0 * r, &s, &c);
    double re = sp.amp * c, im = sp.amp * s;
    if (t.alt_sign != 0 && !odd_grid && (n & 1)) { re = -re; im = -im; }
    const size_t o = (size_t)(a.b0 + bl) * a.N + n;
    if (a.is_double) reinterpret_cast<double2 *>(t.out)[o] = make_double2(re, im);
    else             reinterpret_cast<float2 *>(t.out)[o] = make_float2((float)re, (float)im);
}

} // namespace fresnel
