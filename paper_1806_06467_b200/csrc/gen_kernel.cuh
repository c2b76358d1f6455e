// gen_kernel.cuh -- the pass kernel for grids that are NOT a power of two.
//
// The paper ran N = 2800 and found it faster than 4096; its App. B uses npix = 1025 (:259).
// A line of N points (any N) lives in shared memory and is transformed there:
//   * N = 2^a 3^b 5^c 7^d 11^e 13^f [x one prime P, 17 <= P <= 61]: mixed-radix Stockham stages (radix 16/8/4/2 from
//     fft_core.cuh, odd radices in their symmetric form), ping-ponging between two line buffers; twiddles W_N^m come
//     exactly rounded from one table of N entries (never by recurrence).  The larger prime (1025 = 5^2 41, and the
//     paper's App. B grid npix = 1025 at beam ratio 0.25, N = 4100 = 2^2 5^2 41) is the FIRST stage
//     -- no twiddles -- as a direct P-point DFT, a warp taking a block of outputs with the roots in constant memory
//     (gen_stage_prime);
//   * any other N (1025 = 5^2 41): Bluestein -- a length-N DFT is  chirp x circular convolution x chirp,
//         X[k] = w[k] sum_n (x[n] w[n]) conj(w)[k-n],   w[n] = exp(-i pi n^2 / N),
//     the convolution of length M >= 2N-1 (the next 7-smooth size) done by the same mixed-radix stages on the
//     zero-padded line, entirely on chip; w (n^2 mod 2N in integers, so exact) and the transformed chirp filter
//     are built once per plan.
// An inverse transform is conj o forward o conj.  The pass itself does what pass_kernel.cuh does -- optic phasor
// and chirp table on load, transform, transfer function / output chirp, inverse transform for the convolution
// modes, scale and per-row factor -- for W lines per CTA; column tiles move by TMA exactly as in col_tma.cuh
// (rows of W complex numbers; a partial last box is clipped / zero-filled by the hardware).
// This path is built for coverage, not for the roofline: every stage costs a shared-memory round trip.
#pragma once
#include <cuda.h>
#include <cstdint>
#include "col_tma.cuh"

namespace fresnel {

constexpr int kGenMaxStages = 14;
constexpr int kGenThreads = 256;          // CTA size where two CTAs fit an SM; 2 * kGenThreads where only one does
constexpr int kGenMaxSmem = 226 * 1024;   // dynamic shared memory the generic pass may ask for (227 KB minus its static part)

// bytes of one line buffer (M x W complex), rounded up to the 128-byte alignment TMA wants of a shared-memory box
// (with room for the padded layout of the intermediate stages: one spare element every 16, see gen_stage)
__host__ __device__ constexpr size_t gen_buffer_bytes(int M, int W, int es) { return ((size_t)(M + M / 16 + 1) * W * es + 127) / 128 * 128; }

template <typename T> struct GenArgs {
    using C = typename cplx_of<T>::type;
    C *wf;                    // [batch][N][N]
    int N;                    // grid size
    int M;                    // transform length: N (mixed radix) or the Bluestein convolution length
    int W;                    // lines per CTA
    int mode;                 // PassMode (MODE_FWD / MODE_INV / MODE_CONV)
    int col;                  // 0: row pass; 1: column pass with TMA tiles; 2: column pass with per-thread loads
    int box_rows;             // rows per TMA box (min(256, N))
    int nstages;
    int radix[kGenMaxStages]; // of the length-M transform, in order
    const C *tw;              // [M] forward roots W_M^m = exp(-2 pi i m / M)
    const double2 *prime_roots; // [P] (cos, sin)(2 pi m / P) of the first stage's prime radix P > 16, or nullptr
    const C *blu_w;           // [N] Bluestein chirp exp(-i pi n^2 / N) or nullptr (mixed radix)
    const C *blu_b;           // [M] transform of the chirp filter, scaled by 1/M
    const C *pre, *mid, *rowfac;      // [batch][N] tables as in PassArgs
    const T *amp, *opd;       // [N][N] maps (row pass only)
    const double *inv_lambda;
    T scale;
    int pdl;
};

// ---- one prime factor 17 <= P <= 61 as a direct DFT (gen_stage_prime) ---------------------------------------------
constexpr int kGenMaxPrime = 61;
__host__ __device__ constexpr bool gen_is_stage_prime(int P)
{
    if (P < 17 || P > kGenMaxPrime) return false;
    for (int d = 2; d * d <= P; ++d)
        if (P % d == 0) return false;
    return true;
}
constexpr size_t kGenPrimeTableBytes = 1024;   // shared-memory copy of the roots behind the two line buffers (61 x 16 bytes)

// ---- odd-radix butterflies, symmetric form:  X[q], X[P-q] = (a0 + sum_t c_{tq} (a_t + a_{P-t})) -+ i (sum_t s_{tq} (a_t - a_{P-t}))
// cos / sin of 2 pi i / P, i = 1 .. (P-1)/2, to 30 digits
template <int P> struct OddRoots {
    __host__ __device__ static constexpr double c(int i)
    {
        if constexpr (P == 3) { constexpr double t[1] = {-0.5}; return t[i]; }
        else if constexpr (P == 5) { constexpr double t[2] = {0.309016994374947424102293417183, -0.809016994374947424102293417183}; return t[i]; }
        else if constexpr (P == 7) {
            constexpr double t[3] = {0.623489801858733530525004884004, -0.222520933956314404288902564497, -0.900968867902419126236102319507};
            return t[i];
        } else if constexpr (P == 11) {
            constexpr double t[5] = {0.841253532831181168861811648919, 0.41541501300188642552927414923, -0.142314838273285140443792668616,
                                     -0.654860733945285064056925072466, -0.959492973614497389890368057066};
            return t[i];
        } else {
            constexpr double t[6] = {0.885456025653209895900375522015, 0.568064746731155802511807559128, 0.120536680255323053349067687453,
                                     -0.3546048870425356259696378926, -0.748510748171101098634630599701, -0.970941817426052027156982276294};
            return t[i];
        }
    }
    __host__ __device__ static constexpr double s(int i)
    {
        if constexpr (P == 3) { constexpr double t[1] = {0.866025403784438646763723170753}; return t[i]; }
        else if constexpr (P == 5) { constexpr double t[2] = {0.951056516295153572116439333379, 0.587785252292473129168705954639}; return t[i]; }
        else if constexpr (P == 7) {
            constexpr double t[3] = {0.781831482468029808708444526674, 0.974927912181823607018131682994, 0.433883739117558120475768332849};
            return t[i];
        } else if constexpr (P == 11) {
            constexpr double t[5] = {0.540640817455597582107635954319, 0.909631995354518371411715383079, 0.989821441880932732376092037777,
                                     0.755749574354258283774035843972, 0.281732556841429697711417915347};
            return t[i];
        } else {
            constexpr double t[6] = {0.464723172043768545656015335133, 0.822983865893656394579617423439, 0.992708874098053992800751649493,
                                     0.935016242685414823439784599838, 0.663122658240795202376785492667, 0.23931566428755776714875372626};
            return t[i];
        }
    }
};

// forward DFT of odd prime length P (kernel exp(-2 pi i t q / P)), natural order in and out
template <int P, typename C> FR_DEV void dft_odd(C (&v)[P])
{
    using T = decltype(v[0].x);
    constexpr int H = (P - 1) / 2;
    C sp[H], sm[H];
#pragma unroll
    for (int t = 1; t <= H; ++t) {
        sp[t - 1] = cadd(v[t], v[P - t]);
        sm[t - 1] = csub(v[t], v[P - t]);
    }
    C out0 = v[0];
#pragma unroll
    for (int t = 0; t < H; ++t) out0 = cadd(out0, sp[t]);
    C res[P];
    res[0] = out0;
#pragma unroll
    for (int q = 1; q <= H; ++q) {
        C re = v[0];
        C im;
        im.x = (T)0; im.y = (T)0;
#pragma unroll
        for (int t = 1; t <= H; ++t) {
            const int m = (t * q) % P;                       // cos(2 pi m/P) = c[min(m,P-m)-1]; sin changes sign above P/2
            const int mi = (m <= H ? m : P - m) - 1;
            const T cc = (T)OddRoots<P>::c(mi);
            const T ss = (T)((m <= H ? 1.0 : -1.0) * OddRoots<P>::s(mi));
            re.x += cc * sp[t - 1].x; re.y += cc * sp[t - 1].y;
            im.x += ss * sm[t - 1].x; im.y += ss * sm[t - 1].y;
        }
        // X[q] = re - i*im ;  X[P-q] = re + i*im        (-i*(x+iy) = y - i x)
        res[q].x = re.x + im.y;      res[q].y = re.y - im.x;
        res[P - q].x = re.x - im.y;  res[P - q].y = re.y + im.x;
    }
#pragma unroll
    for (int q = 0; q < P; ++q) v[q] = res[q];
}

// one Stockham stage of radix R over W interleaved lines of length `len`: src -> dst, layout element (n, g) at [n*W + g].
// PIN / POUT: the input / output buffer uses the padded layout n -> n + n/16 (the stride-R scatter of the first stage
// would otherwise hit the same banks 8 times over); the first stage of a transform reads, and the last one writes, the
// dense layout that TMA and the pointwise steps use.
template <bool PADDED> FR_DEV int gen_pos(int n) { return PADDED ? n + (n >> 4) : n; }

template <typename T, int R, bool PIN, bool POUT>
FR_DEV void gen_stage(const typename cplx_of<T>::type *__restrict__ src, typename cplx_of<T>::type *__restrict__ dst, int len, int W, int Ns,
                      const typename cplx_of<T>::type *__restrict__ tw, int tid)
{
    using C = typename cplx_of<T>::type;
    const int nb = len / R;                    // butterflies per line
    const int tstep = len / (Ns * R);          // W_{Ns R}^{t k} = W_len^{t k tstep}
    for (int idx = tid; idx < nb * W; idx += (int)blockDim.x) {
        const int b = idx / W, g = idx - b * W;
        const int k = b % Ns;
        C v[R];
#pragma unroll
        for (int t = 0; t < R; ++t) v[t] = src[(size_t)gen_pos<PIN>(b + t * nb) * W + g];
        if (Ns > 1) {
            // W_{Ns R}^{t k} = w^t with w = W_len^{k tstep}: ONE table load, the powers by a product tree (w^t = w^(t/2) *
            // w^(t - t/2): at most four chained multiplies for t <= 15, so a power is good to a few ulp)
            C pw[R];
            pw[1] = ldg_c(tw + k * tstep);         // k * tstep < len
            v[1] = cmul(v[1], pw[1]);
#pragma unroll
            for (int t = 2; t < R; ++t) {
                pw[t] = (t & 1) ? cmul(pw[t / 2], pw[t - t / 2]) : csq(pw[t / 2]);
                v[t] = cmul(v[t], pw[t]);
            }
        }
        if constexpr (R == 16) dft16<-1>(v);
        else if constexpr (R == 8) dft8<-1>(v[0], v[1], v[2], v[3], v[4], v[5], v[6], v[7]);
        else if constexpr (R == 4) dft4<-1>(v[0], v[1], v[2], v[3]);
        else if constexpr (R == 2) dft2<-1>(v[0], v[1]);
        else dft_odd<R>(v);
        const int o = (b - k) * R + k;
#pragma unroll
        for (int q = 0; q < R; ++q) dst[(size_t)gen_pos<POUT>(o + q * Ns) * W + g] = v[q];
    }
}

// First stage (Ns = 1: no twiddles) of prime radix P > 16, dense src -> dst.  Symmetric form as in dft_odd, but the P
// points do not fit the registers of one thread: a task is (block of QC output pairs, 32 butterflies); the warp that
// takes it streams the input pairs x[t], x[P-t] from shared memory once and keeps 2 QC complex accumulators per lane; the
// roots (cos, sin)(2 pi m / P) sit in shared memory and every read of them is one address per warp.  X[q], X[P-q] = (x0 + sum_t c_{tq} (x_t + x_{P-t})) -+ i (sum_t
// s_{tq} (x_t - x_{P-t})).
template <typename T, bool POUT>
FR_DEV void gen_stage_prime(const typename cplx_of<T>::type *__restrict__ src, typename cplx_of<T>::type *__restrict__ dst, int len, int W,
                            int P, const double2 *roots, int tid)
{
    using C = typename cplx_of<T>::type;
    constexpr int QC = 5;                                           // P = 41: 4 blocks of 5 output pairs
    const int nb = len / P, H = (P - 1) / 2;
    const int items = nb * W, nblk = (items + 31) / 32, nchunk = (H + QC - 1) / QC;
    const int warp = tid >> 5, lane = tid & 31;
    for (int task = warp; task < nchunk * nblk; task += (int)blockDim.x / 32) {
        const int c = task / nblk, blk = task - c * nblk;
        const int item = blk * 32 + lane;
        if (item >= items) continue;
        const int b = item / W, g = item - b * W;
        const int q0 = c * QC + 1;                                  // this task's outputs: q0 .. q0 + QC - 1 (<= H) and P - q
        const C x0 = src[(size_t)b * W + g];
        C re[QC], im[QC], sum = x0;
        int m[QC];
#pragma unroll
        for (int i = 0; i < QC; ++i) { re[i] = x0; im[i].x = (T)0; im[i].y = (T)0; m[i] = 0; }
        for (int t = 1; t <= H; ++t) {
            const C xa = src[(size_t)(b + t * nb) * W + g], xb = src[(size_t)(b + (P - t) * nb) * W + g];
            const C sp = cadd(xa, xb), sm = csub(xa, xb);
            sum = cadd(sum, sp);
#pragma unroll
            for (int i = 0; i < QC; ++i) {
                m[i] += q0 + i;                                     // t q mod P
                if (m[i] >= P) m[i] -= P;
                const double2 r = roots[m[i]];                      // shared memory, one address per warp: a broadcast
                const T cc = (T)r.x, ss = (T)r.y;
                re[i].x += cc * sp.x; re[i].y += cc * sp.y;
                im[i].x += ss * sm.x; im[i].y += ss * sm.y;
            }
        }
        C *o = dst + g;
        const int p0 = b * P;
        if (c == 0) o[(size_t)gen_pos<POUT>(p0) * W] = sum;
#pragma unroll
        for (int i = 0; i < QC; ++i) {
            const int q = q0 + i;
            if (q <= H) {
                C a, z;                                              // X[q] = re - i im ; X[P-q] = re + i im
                a.x = re[i].x + im[i].y; a.y = re[i].y - im[i].x;
                z.x = re[i].x - im[i].y; z.y = re[i].y + im[i].x;
                o[(size_t)gen_pos<POUT>(p0 + q) * W] = a;
                o[(size_t)gen_pos<POUT>(p0 + P - q) * W] = z;
            }
        }
    }
}

template <typename T, int R>
FR_DEV void gen_stage_any(const typename cplx_of<T>::type *src, typename cplx_of<T>::type *dst, int len, int W, int Ns,
                          const typename cplx_of<T>::type *__restrict__ tw, int tid, bool pin, bool pout)
{
    if (pin) { if (pout) gen_stage<T, R, true, true>(src, dst, len, W, Ns, tw, tid); else gen_stage<T, R, true, false>(src, dst, len, W, Ns, tw, tid); }
    else     { if (pout) gen_stage<T, R, false, true>(src, dst, len, W, Ns, tw, tid); else gen_stage<T, R, false, false>(src, dst, len, W, Ns, tw, tid); }
}

// forward transform of length len = a.M on the W lines in *src; on return *src holds the result (buffers swapped as needed)
template <typename T>
FR_DEV void gen_fft(typename cplx_of<T>::type *&src, typename cplx_of<T>::type *&dst, const GenArgs<T> &a, const double2 *roots, int tid)
{
    using C = typename cplx_of<T>::type;
    int Ns = 1;
    for (int s = 0; s < a.nstages; ++s) {
        const int R = a.radix[s];
        const bool pin = s > 0, pout = s + 1 < a.nstages;
        switch (R) {
        case 16: gen_stage_any<T, 16>(src, dst, a.M, a.W, Ns, a.tw, tid, pin, pout); break;
        case 8:  gen_stage_any<T, 8>(src, dst, a.M, a.W, Ns, a.tw, tid, pin, pout); break;
        case 4:  gen_stage_any<T, 4>(src, dst, a.M, a.W, Ns, a.tw, tid, pin, pout); break;
        case 2:  gen_stage_any<T, 2>(src, dst, a.M, a.W, Ns, a.tw, tid, pin, pout); break;
        case 3:  gen_stage_any<T, 3>(src, dst, a.M, a.W, Ns, a.tw, tid, pin, pout); break;
        case 5:  gen_stage_any<T, 5>(src, dst, a.M, a.W, Ns, a.tw, tid, pin, pout); break;
        case 7:  gen_stage_any<T, 7>(src, dst, a.M, a.W, Ns, a.tw, tid, pin, pout); break;
        case 11: gen_stage_any<T, 11>(src, dst, a.M, a.W, Ns, a.tw, tid, pin, pout); break;
        case 13: gen_stage_any<T, 13>(src, dst, a.M, a.W, Ns, a.tw, tid, pin, pout); break;
        default:                                                    // one prime 17 .. 61, always the first stage
            if (pout) gen_stage_prime<T, true>(src, dst, a.M, a.W, R, roots, tid);
            else gen_stage_prime<T, false>(src, dst, a.M, a.W, R, roots, tid);
            break;
        }
        Ns *= R;
        __syncthreads();
        C *t = src; src = dst; dst = t;
    }
}

// length-N forward DFT of the W lines in *src (first N entries of each line valid; the rest is scratch).
//   conj_in (Bluestein only): the input is conjugated on the way in (first half of an inverse transform) -- folded into
//   the chirp multiply; in the mixed-radix case the CALLER conjugates inside its neighbouring pointwise step.
// Mixed radix: the transform itself.  Bluestein: chirp, zero-pad, FFT_M, x filter, inverse FFT_M, chirp.
template <typename T>
FR_DEV void gen_dft(typename cplx_of<T>::type *&src, typename cplx_of<T>::type *&dst, const GenArgs<T> &a, const double2 *roots, int tid, bool conj_in)
{
    using C = typename cplx_of<T>::type;
    const int N = a.N, M = a.M, W = a.W;
    if (a.blu_w == nullptr) {            // mixed radix: the caller has folded the conjugation into its own pointwise step
        gen_fft<T>(src, dst, a, roots, tid);
        return;
    }
    for (int e = tid; e < M * W; e += (int)blockDim.x) {
        const int n = e / W;
        C x;
        x.x = (T)0; x.y = (T)0;
        if (n < N) {
            x = src[e];
            if (conj_in) x.y = -x.y;
            x = cmul(x, ldg_c(a.blu_w + n));
        }
        src[e] = x;
    }
    __syncthreads();
    gen_fft<T>(src, dst, a, roots, tid);
    for (int e = tid; e < M * W; e += (int)blockDim.x) {          // x filter, conjugate: inverse FFT_M = conj o FFT_M o conj
        const C t = cmul(src[e], ldg_c(a.blu_b + e / W));
        src[e].x = t.x; src[e].y = -t.y;
    }
    __syncthreads();
    gen_fft<T>(src, dst, a, roots, tid);
    for (int e = tid; e < N * W; e += (int)blockDim.x) {
        C t = src[e];
        t.y = -t.y;
        src[e] = cmul(t, ldg_c(a.blu_w + e / W));
    }
    __syncthreads();
}

template <typename T, int NT>
__global__ void __launch_bounds__(NT, NT == kGenThreads ? 2 : 1) gen_pass_kernel(GenArgs<T> a, const __grid_constant__ CUtensorMap tmap)
{
    using C = typename cplx_of<T>::type;
    constexpr int ES = (int)sizeof(C);
    extern __shared__ __align__(1024) unsigned char fr_smem[];
    __shared__ __align__(8) uint64_t full_bar;
    unsigned char *base = fr_smem + ((1024u - (smem_u32(fr_smem) & 1023u)) & 1023u);
    const int N = a.N, M = a.M, W = a.W;
    C *src = reinterpret_cast<C *>(base);
    C *dst = reinterpret_cast<C *>(base + gen_buffer_bytes(M, W, ES));     // 128-byte aligned: either buffer may feed the TMA store
    const double2 *roots = reinterpret_cast<const double2 *>(base + 2 * gen_buffer_bytes(M, W, ES));
    if (a.prime_roots != nullptr)                           // visible after the barriers that follow the load
        for (int m = threadIdx.x; m < a.radix[0]; m += (int)blockDim.x) const_cast<double2 *>(roots)[m] = a.prime_roots[m];
    const int tid = threadIdx.x;
    const int b = blockIdx.y;
    const int line0 = blockIdx.x * W;                       // first row / column of this CTA
    const int nl = (N - line0 < W) ? N - line0 : W;         // lines that exist (row pass: the last CTA may be partial)

    if (tid == 0) mbar_init(&full_bar, 1);
    pdl_launch_dependents();
    __syncthreads();
    pdl_wait();
    // ---- load: element (n, g) of the tile -> src[n*W + g] ----
    if (a.col == 1) {
        // whole boxes are written (rows / columns beyond the grid arrive as zeros); the spill past row N lands in
        // the second line buffer, which is scratch at this point
        if (tid == 0) {
            const int nbox = (N + a.box_rows - 1) / a.box_rows;
            mbar_expect_tx(&full_bar, (uint32_t)((size_t)nbox * a.box_rows * W * ES));
            for (int r0 = 0; r0 < N; r0 += a.box_rows) tma_load_3d(base + (size_t)r0 * W * ES, &tmap, &full_bar, line0 * 2, r0, b);
        }
        mbar_wait(&full_bar, 0);
    } else if (a.col == 2) {
        const C *g0 = a.wf + (size_t)b * N * N + line0;
        for (int e = tid; e < N * W; e += (int)blockDim.x) {
            const int n = e / W, g = e - n * W;
            C x;
            x.x = (T)0; x.y = (T)0;
            if (g < nl) x = g0[(size_t)n * N + g];
            src[e] = x;
        }
    } else {
        for (int g = 0; g < W; ++g) {
            const C *row = a.wf + (size_t)b * N * N + (size_t)(line0 + g) * N;
            for (int n = tid; n < N; n += (int)blockDim.x) {
                C x;
                x.x = (T)0; x.y = (T)0;
                if (g < nl) {
                    x = row[n];
                    const size_t o = (size_t)(line0 + g) * N + n;
                    if (a.opd != nullptr) x = cmul(x, phasor_turns<T>(a.opd[o] * (T)a.inv_lambda[b]));
                    if (a.amp != nullptr) { const T s = a.amp[o]; x.x *= s; x.y *= s; }
                }
                src[(size_t)n * W + g] = x;
            }
        }
    }
    // pre table (along the line) and, for MODE_INV, the conjugation that opens an inverse transform
    const bool inv = a.mode == MODE_INV, conv = a.mode == MODE_CONV, blu = a.blu_w != nullptr;
    if (a.pre != nullptr || (inv && !blu)) {
        const C *p = a.pre != nullptr ? a.pre + (size_t)b * N : nullptr;
        for (int e = tid; e < N * W; e += (int)blockDim.x) {
            C x = src[e];
            if (p != nullptr) x = cmul(x, ldg_c(p + e / W));
            if (inv && !blu) x.y = -x.y;
            src[e] = x;
        }
    }
    __syncthreads();

    gen_dft<T>(src, dst, a, roots, tid, inv && blu);                // F (or conj . F . with the closing conj below)
    {
        const C *m = a.mid != nullptr ? a.mid + (size_t)b * N : nullptr;
        if (inv || m != nullptr || (conv && !blu)) {
            for (int e = tid; e < N * W; e += (int)blockDim.x) {
                C x = src[e];
                if (inv) x.y = -x.y;                         // closes the inverse transform
                if (m != nullptr) x = cmul(x, ldg_c(m + e / W));
                if (conv && !blu) x.y = -x.y;                // opens the inverse transform of the convolution
                src[e] = x;
            }
            __syncthreads();
        }
        if (conv) gen_dft<T>(src, dst, a, roots, tid, blu);         // inverse transform = conj . F . conj (closing conj: on the store)
    }
    // ---- scale, per-row factor, store ----
    const T sx = a.scale, sy = conv ? -a.scale : a.scale;   // scale, and the closing conjugation of the convolution
    if (a.col == 1) {
        if (a.scale != (T)1 || conv)
            for (int e = tid; e < N * W; e += (int)blockDim.x) { src[e].x *= sx; src[e].y *= sy; }
        fence_async_proxy();
        __syncthreads();
        if (tid == 0) {
            for (int r0 = 0; r0 < N; r0 += a.box_rows) tma_store_3d(&tmap, reinterpret_cast<unsigned char *>(src) + (size_t)r0 * W * ES, line0 * 2, r0, b);
            tma_store_commit_and_wait();
        }
    } else if (a.col == 2) {
        C *g0 = a.wf + (size_t)b * N * N + line0;
        for (int e = tid; e < N * W; e += (int)blockDim.x) {
            const int n = e / W, g = e - n * W;
            if (g < nl) { C x = src[e]; x.x *= sx; x.y *= sy; g0[(size_t)n * N + g] = x; }
        }
    } else {
        for (int g = 0; g < nl; ++g) {
            C *row = a.wf + (size_t)b * N * N + (size_t)(line0 + g) * N;
            C rf;
            rf.x = a.scale; rf.y = (T)0;
            if (a.rowfac != nullptr) {
                const C c = ldg_c(a.rowfac + (size_t)b * N + line0 + g);
                rf.x = c.x * a.scale; rf.y = c.y * a.scale;
            }
            for (int n = tid; n < N; n += (int)blockDim.x) {
                C x = src[(size_t)n * W + g];
                if (conv) x.y = -x.y;
                row[n] = cmul(x, rf);
            }
        }
    }
}

// One (precision, CTA size) of the generic kernel: instantiated in gen_inst.cu, one object each (the kernel is ~75 k SASS
// instructions per instantiation; four objects compile in parallel).
template <typename T, int NT>
cudaError_t launch_gen_pass_nt(const GenArgs<T> &a, const CUtensorMap &tmap, int batch, size_t smem, cudaStream_t stream)
{
    auto kern = gen_pass_kernel<T, NT>;
    static std::atomic<unsigned long long> configured{0};
    if (fr_needs_configuring(configured)) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kGenMaxSmem);
        if (e != cudaSuccess) return e;
        fr_mark_configured(configured);
    }
    dim3 grid((a.N + a.W - 1) / a.W, batch, 1);
    return launch_pdl(kern, grid, dim3(NT), smem, stream, a.pdl != 0, a, tmap);
}

} // namespace fresnel
