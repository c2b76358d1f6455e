// fresnel_api.cu -- the C ABI of include/fresnel.h: argument checks, chirp-table cache, pass scheduling, launches.
// Every step of the hot path runs in the kernels of pass_kernel.cuh / col_tma.cuh / pointwise.cuh / tables.cuh;
// this file only decides which tables a call needs, in which order the passes run, and enqueues them.
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include <cuda.h>
#include <cuda_runtime.h>

#include "../../include/fresnel.h"
#include "dispatch.h"
#include "gen_kernel.cuh"
#include "mft.cuh"
#include "pointwise.cuh"
#include "tables.cuh"

using namespace fresnel;

namespace {

constexpr int kDefaultSlots = 64;       // table slots of a new plan (fresnel_plan_reserve_tables grows the pool)
constexpr int kMaxMapDescs = 64;        // cached tensor maps of surface maps (fused column passes)
const long double PI_L = 3.14159265358979323846264338327950288419716939937510L;

// kinds of cached 1-D tables
enum { KIND_CENTRED = 0, KIND_FFTORDER = 1, KIND_SCALARS = 2 };

// One cached table: [batch][N] complex of the plan's dtype (chirps) or [batch] doubles (KIND_SCALARS: 1/lambda).
// Ownership.  An EAGER slot serves cache hits and may be evicted (least recently used).  A slot written while the
// stream is being captured into a CUDA graph is GRAPH-OWNED from then on: the builder was only recorded, and every
// replay rewrites the slot behind the host's back -- so it never serves an eager hit and is never evicted; it
// serves hits only to later calls of the SAME capture (its builder node precedes them in that graph).  Graph-owned
// slots return to the pool with fresnel_plan_release_graph_tables.
struct TableSlot {
    void *dev = nullptr;
    bool valid = false;
    bool graph_owned = false;
    unsigned long long capture_id = 0;
    uint64_t stamp = 0;
    uint64_t pin = 0;                   // pin epoch that last asked for it (never evicted within that epoch)
    int kind = 0, alt_sign = 0;
    std::vector<ChirpSpec> key;
};

struct TableRequest {
    int slot = -1;                      // -1: no slot could be had (all graph-owned or pinned)
    bool build = false;
};

struct CaptureState {
    bool active = false;
    unsigned long long id = 0;
};

struct MapDesc {
    const void *ptr = nullptr;
    uint64_t stamp = 0;
    CUtensorMap map{};
};

} // namespace

struct fresnel_plan {
    int N = 0, batch = 0;
    fresnel_dtype dtype = FRESNEL_C128;
    int device = 0;                     // the CUDA device the plan lives on; every entry point switches to it
    cudaStream_t stream = nullptr;
    cudaEvent_t order_ev = nullptr;     // orders the old and the new stream in fresnel_plan_set_stream
    void *tw = nullptr;                 // FFT twiddles
    std::vector<TableSlot> slots;
    std::vector<void *> arenas;         // device allocations behind the slots
    uint64_t clock = 0, pin_epoch = 0;
    unsigned long long launches = 0;
    int prefetch = 0;                   // L2 prefetch distance in tiles (see pass_kernel.cuh)
    int tma_w = 0;                      // columns per TMA tile of the column pass (0: not used for this N)
    int tma_w2 = 0;                     // the same for the fused column pass (MODE_CONV2), which may prefer narrower tiles
    int map_box = 0;                    // columns per TMA box of a surface map (fused column pass)
    int sms = 148;
    int pdl = 1;                        // programmatic dependent launch of the pass kernels (FRESNEL_PDL=0: off, A/B timing)
    int fuse = 1;                       // train-level pass fusion in fresnel_system_run (FRESNEL_FUSE=0: off, A/B timing)
    // grids that are not a power of two (gen_kernel.cuh): transform length, radices, root table, Bluestein tables
    bool generic = false;
    int gen_M = 0, gen_nstages = 0, gen_radix[kGenMaxStages] = {0};
    int gen_wcol = 1, gen_box_rows = 256;
    bool gen_tma = false;               // column tiles by TMA (needs a 16-byte multiple row pitch: not complex64 with odd N)
    bool mr = false;                    // this N has a register-resident mixed-radix pass (mr_kernel.cuh)
    void *gen_tw = nullptr, *gen_blu_w = nullptr, *gen_blu_b = nullptr, *gen_prime_roots = nullptr;
    // matrix Fourier transform (mft.cuh): kernel matrix E [batch][nb][N], intermediate T^t [batch][nb][N], per-batch scalars
    double2 *mft_e = nullptr, *mft_t = nullptr;
    double *mft_scal = nullptr;         // [4][batch]: c_hi, c_lo, alpha.re, alpha.im  (alpha interleaved at +2*batch)
    int mft_nb_cap = 0;
    std::vector<double> mft_key;        // what mft_e currently holds (nb, direction, c_hi.., c_lo..); empty: nothing
    CUtensorMap tmap{};                  // tensor map of the wavefront last seen by the column pass
    const void *tmap_wf = nullptr;
    CUtensorMap tmap2;                  // wavefront tiles of the fused column pass
    const void *tmap2_wf = nullptr;
    std::vector<MapDesc> map_descs;     // tensor maps of surface maps, by pointer
    cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};   // profiling hook, see fresnel_plan_record_pass_events
    bool ev_armed = false;
    std::vector<cudaEvent_t> train_ev;  // profiling hook, see fresnel_plan_record_train_events
    std::vector<fresnel_pass_info> schedule;           // pass kernels of the last fresnel_system_run
    size_t esize() const { return dtype == FRESNEL_C128 ? sizeof(double2) : sizeof(float2); }
    size_t slot_bytes() const { return (size_t)batch * N * esize(); }
};

namespace {

bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

// Every entry point runs on the plan's device, whatever the caller's current device is.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(const fresnel_plan *p)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) { cudaGetLastError(); prev = -1; return; }
        if (prev != p->device && cudaSetDevice(p->device) == cudaSuccess) switched = true;
    }
    ~DeviceGuard()
    {
        if (switched) cudaSetDevice(prev);
    }
};

// ---- FFT twiddle tables (host, long double) --------------------------------------------------------
template <typename C> void fill_twiddles_for(int N, std::vector<C> &out)
{
    const int S = fr_num_stages(N);
    out.assign((size_t)fr_tw_total(N), C{});
    for (int s = 1; s < S; ++s) {
        const int R = fr_radix(N, s), NS = fr_ns(N, s);
        C *t = out.data() + fr_tw_offset(N, s);
        for (int k = 0; k < NS; ++k) {
            // base forward twiddle W_{NS*R}^k = exp(-2 pi i k / (NS*R)); its powers are formed on the device
            long double ang = -2.0L * PI_L * (long double)k / (long double)((long)NS * R);
            C w;
            w.x = (decltype(w.x))cosl(ang);
            w.y = (decltype(w.y))sinl(ang);
            t[k] = w;
        }
    }
}

fresnel_status upload_twiddles(fresnel_plan *p)
{
    const size_t n = (size_t)fr_tw_total(p->N);
    if (cudaMalloc(&p->tw, (n ? n : 1) * p->esize()) != cudaSuccess) return FRESNEL_ERR_ALLOC;
    cudaError_t e;
    if (p->dtype == FRESNEL_C128) {
        std::vector<double2> h;
        fill_twiddles_for(p->N, h);
        e = cudaMemcpy(p->tw, h.data(), n * sizeof(double2), cudaMemcpyHostToDevice);
    } else {
        std::vector<float2> h;
        fill_twiddles_for(p->N, h);
        e = cudaMemcpy(p->tw, h.data(), n * sizeof(float2), cudaMemcpyHostToDevice);
    }
    return e == cudaSuccess ? FRESNEL_OK : FRESNEL_ERR_CUDA;
}

// ---- chirp-table cache -------------------------------------------------------------------------------
ChirpSpec make_spec(long double c_turns, double amp, double phase0)
{
    ChirpSpec s;
    s.c_hi = (double)c_turns;
    s.c_lo = (double)(c_turns - (long double)s.c_hi);
    s.amp = amp;
    s.phase0 = phase0;
    return s;
}

CaptureState capture_state(fresnel_plan *p)
{
    CaptureState c;
    cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
    unsigned long long id = 0;
    if (cudaStreamGetCaptureInfo(p->stream, &st, &id) != cudaSuccess) { cudaGetLastError(); return c; }
    c.active = st != cudaStreamCaptureStatusNone;
    c.id = id;
    return c;
}

// Grow the slot pool by `extra` slots (one device allocation).  Never called while capturing.
fresnel_status grow_slots(fresnel_plan *p, int extra)
{
    if (extra <= 0) return FRESNEL_OK;
    void *arena = nullptr;
    if (cudaMalloc(&arena, (size_t)extra * p->slot_bytes()) != cudaSuccess) { cudaGetLastError(); return FRESNEL_ERR_ALLOC; }
    p->arenas.push_back(arena);
    for (int i = 0; i < extra; ++i) {
        TableSlot s;
        s.dev = (unsigned char *)arena + (size_t)i * p->slot_bytes();
        p->slots.push_back(std::move(s));
    }
    return FRESNEL_OK;
}

int eager_slot_count(const fresnel_plan *p)
{
    int n = 0;
    for (const TableSlot &s : p->slots)
        if (!s.graph_owned) ++n;
    return n;
}

// Find or assign a cache slot for a table (see TableSlot for the ownership rules).
TableRequest request_table(fresnel_plan *p, int kind, int alt_sign, const std::vector<ChirpSpec> &key, const CaptureState &cap)
{
    ++p->clock;
    const int ns = (int)p->slots.size();
    for (int i = 0; i < ns; ++i) {
        TableSlot &s = p->slots[i];
        if (!s.valid || s.kind != kind || s.alt_sign != alt_sign || s.key.size() != key.size()) continue;
        if (cap.active ? !(s.graph_owned && s.capture_id == cap.id) : s.graph_owned) continue;
        if (std::memcmp(s.key.data(), key.data(), key.size() * sizeof(ChirpSpec)) != 0) continue;
        s.stamp = p->clock;
        s.pin = p->pin_epoch;
        return {i, false};
    }
    // miss: a slot never used, else the least recently used eager slot that this pin epoch has not asked for
    int victim = -1;
    for (int i = 0; i < ns && victim < 0; ++i)
        if (!p->slots[i].valid && !p->slots[i].graph_owned) victim = i;
    if (victim < 0)
        for (int i = 0; i < ns; ++i) {
            const TableSlot &s = p->slots[i];
            if (s.graph_owned || s.pin == p->pin_epoch) continue;
            if (victim < 0 || s.stamp < p->slots[victim].stamp) victim = i;
        }
    if (victim < 0) return {-1, false};
    TableSlot &s = p->slots[victim];
    s.valid = true;
    s.graph_owned = cap.active;
    s.capture_id = cap.id;
    s.kind = kind;
    s.alt_sign = alt_sign;
    s.key = key;
    s.stamp = p->clock;
    s.pin = p->pin_epoch;
    return {victim, true};
}

// 1/lambda per batch element on the device (needed by the optic phasor): a KIND_SCALARS table.
TableRequest request_inv_lambda(fresnel_plan *p, const double *lambda, const CaptureState &cap)
{
    std::vector<ChirpSpec> key(p->batch);
    for (int b = 0; b < p->batch; ++b) key[b] = make_spec((long double)(double)(1.0L / (long double)lambda[b]), 0.0, 0.0);
    return request_table(p, KIND_SCALARS, 0, key, cap);
}

// Launch the builder for every requested table that is not resident.
fresnel_status flush_builds(fresnel_plan *p, const TableRequest *req, int nreq)
{
    std::vector<int> todo;
    for (int i = 0; i < nreq; ++i) {
        if (req[i].slot < 0) return FRESNEL_ERR_ALLOC;
        if (!req[i].build) continue;
        bool dup = false;
        for (int s : todo) dup = dup || s == req[i].slot;
        if (!dup) todo.push_back(req[i].slot);
    }
    // scalar tables ride along one per launch; chirp tables kBuildMaxTables per launch
    std::vector<int> chirps, scalars;
    for (int s : todo) (p->slots[s].kind == KIND_SCALARS ? scalars : chirps).push_back(s);
    size_t ci = 0, si = 0;
    while (ci < chirps.size() || si < scalars.size()) {
        const int ntab = (int)((chirps.size() - ci < (size_t)kBuildMaxTables) ? chirps.size() - ci : (size_t)kBuildMaxTables);
        const int sc = si < scalars.size() ? scalars[si] : -1;
        for (int b0 = 0; b0 < p->batch; b0 += kBuildMaxBatch) {
            BuildArgs a;
            std::memset(&a, 0, sizeof(a));
            a.N = p->N;
            a.b0 = b0;
            a.nb = (p->batch - b0 < kBuildMaxBatch) ? p->batch - b0 : kBuildMaxBatch;
            a.ntab = ntab;
            a.is_double = p->dtype == FRESNEL_C128;
            a.scal_out = sc >= 0 ? (double *)p->slots[sc].dev : nullptr;
            for (int b = 0; b < a.nb; ++b) {
                if (sc >= 0) a.scal[b] = p->slots[sc].key[b0 + b].c_hi;
                for (int t = 0; t < ntab; ++t) a.t[t].spec[b] = p->slots[chirps[ci + t]].key[b0 + b];
            }
            for (int t = 0; t < ntab; ++t) {
                const TableSlot &s = p->slots[chirps[ci + t]];
                a.t[t].out = s.dev;
                a.t[t].index_mode = s.kind;
                a.t[t].alt_sign = s.alt_sign;
            }
            dim3 grid((p->N + 127) / 128, a.nb, ntab > 0 ? ntab : 1);
            build_tables_kernel<<<grid, 128, 0, p->stream>>>(a);
            if (cudaGetLastError() != cudaSuccess) return FRESNEL_ERR_CUDA;
            ++p->launches;
        }
        ci += ntab;
        if (sc >= 0) ++si;
    }
    return FRESNEL_OK;
}

bool valid_positive(const double *v, int n)
{
    if (!v) return false;
    for (int i = 0; i < n; ++i)
        if (!(v[i] > 0.0) || !std::isfinite(v[i])) return false;
    return true;
}

// ---- grids that are not a power of two ---------------------------------------------------------------------------
// Radices of a length-M mixed-radix transform (16, 8, 4, 2, then 13, 11, 7, 5, 3); what is left may be ONE prime of
// 17 .. 61, which then becomes the first stage (gen_stage_prime: a direct DFT without twiddles).  False if
// M has any other prime factor.
bool factor_radices(int M, int *radix, int *nstages)
{
    int n = 0;
    auto take = [&](int r) {
        while (M % r == 0 && n < kGenMaxStages - 1) { radix[n++] = r; M /= r; }
    };
    take(16); take(8); take(4); take(2); take(13); take(11); take(7); take(5); take(3);
    if (M > 1 && gen_is_stage_prime(M)) {
        for (int i = n; i > 0; --i) radix[i] = radix[i - 1];
        radix[0] = M;
        ++n;
        M = 1;
    }
    *nstages = n;
    return M == 1;
}

int next_smooth(int m)      // smallest 7-smooth integer >= m
{
    for (;; ++m) {
        int r = m;
        for (int p : {2, 3, 5, 7})
            while (r % p == 0) r /= p;
        if (r == 1) return m;
    }
}

template <typename C> fresnel_status upload_vec(void **dev, const std::vector<C> &h)
{
    if (cudaMalloc(dev, h.size() * sizeof(C)) != cudaSuccess) return FRESNEL_ERR_ALLOC;
    return cudaMemcpy(*dev, h.data(), h.size() * sizeof(C), cudaMemcpyHostToDevice) == cudaSuccess ? FRESNEL_OK : FRESNEL_ERR_CUDA;
}

// Root table W_M^m, and for Bluestein the chirp w[n] = exp(-i pi n^2/N) (n^2 mod 2N in integers: exact) and the
// length-M transform of the chirp filter conj(w)[|m|] (zero elsewhere), scaled by 1/M -- all in long double on the
// host, rounded once.
template <typename C> fresnel_status build_generic_tables(fresnel_plan *p, bool bluestein)
{
    using T = decltype(C{}.x);
    const int N = p->N, M = p->gen_M;
    std::vector<C> tw(M);
    std::vector<long double> wr(M), wi(M);
    for (int m = 0; m < M; ++m) {
        const long double a = -2.0L * PI_L * (long double)m / (long double)M;
        wr[m] = cosl(a); wi[m] = sinl(a);
        tw[m].x = (T)wr[m]; tw[m].y = (T)wi[m];
    }
    fresnel_status st = upload_vec(&p->gen_tw, tw);
    if (st != FRESNEL_OK || !bluestein) return st;
    std::vector<C> w(N), bh(M);
    std::vector<long double> br(M, 0.0L), bi(M, 0.0L);
    for (int n = 0; n < N; ++n) {
        const long long q = ((long long)n * n) % (2LL * N);
        const long double a = PI_L * (long double)q / (long double)N;
        w[n].x = (T)cosl(a); w[n].y = (T)(-sinl(a));
        br[n] = cosl(a); bi[n] = sinl(a);                           // conj(w)[n]
        if (n > 0) { br[M - n] = br[n]; bi[M - n] = bi[n]; }
    }
    // plain O(M^2) sum: a one-off of at most ~5e7 terms per plan
    for (int k = 0; k < M; ++k) {
        long double sr = 0.0L, si = 0.0L;
        long long e = 0;
        for (int m = 0; m < M; ++m) {
            if (br[m] != 0.0L || bi[m] != 0.0L) {
                sr += br[m] * wr[e] - bi[m] * wi[e];
                si += br[m] * wi[e] + bi[m] * wr[e];
            }
            e += k;
            if (e >= M) e -= M;
        }
        bh[k].x = (T)(sr / (long double)M);
        bh[k].y = (T)(si / (long double)M);
    }
    st = upload_vec(&p->gen_blu_w, w);
    if (st != FRESNEL_OK) return st;
    return upload_vec(&p->gen_blu_b, bh);
}

// Can the shared-memory path take this grid?  Two line buffers of the transform length (N, or the Bluestein
// convolution length) with the narrowest column tile (16 bytes) must fit one SM's shared memory.
bool generic_supported(int N, fresnel_dtype dt)
{
    int radix[kGenMaxStages], ns = 0;
    int M = N;
    if (!factor_radices(N, radix, &ns)) {
        M = next_smooth(2 * N - 1);
        if (!factor_radices(M, radix, &ns)) return false;
    }
    const size_t es = dt == FRESNEL_C128 ? 16 : 8;
    return 2 * gen_buffer_bytes(M, (int)(16 / es), (int)es) + 1024 + kGenPrimeTableBytes <= (size_t)kGenMaxSmem;
}

// Shared memory of the generic pass: two line buffers of M x W complex + alignment slack.
size_t gen_smem(const fresnel_plan *p, int W) { return 2 * gen_buffer_bytes(p->gen_M, W, (int)p->esize()) + 1024 + kGenPrimeTableBytes; }

fresnel_status setup_generic(fresnel_plan *p)
{
    const int N = p->N;
    bool bluestein = !factor_radices(N, p->gen_radix, &p->gen_nstages);
    p->gen_M = N;
    if (bluestein) {
        p->gen_M = next_smooth(2 * N - 1);
        if (!factor_radices(p->gen_M, p->gen_radix, &p->gen_nstages)) return FRESNEL_ERR_UNSUPPORTED;
    }
    // column tiles: W complex per row, at least 16 bytes (TMA minimum; also the box start alignment), 32 where two
    // CTAs still fit an SM
    const int es = (int)p->esize();
    const int wmin = 16 / es, wpref = 32 / es;
    if (gen_smem(p, wmin) > (size_t)kGenMaxSmem) return FRESNEL_ERR_UNSUPPORTED;
    p->gen_wcol = (2 * gen_smem(p, wpref) <= (size_t)kGenMaxSmem) ? wpref : wmin;
    p->gen_box_rows = N < 256 ? N : 256;
    p->gen_tma = ((size_t)N * es) % 16 == 0 && std::getenv("FRESNEL_NO_TMA") == nullptr;
    if (p->gen_radix[0] > 16) {                                   // (cos, sin)(2 pi m / P) of the prime first stage
        const int P = p->gen_radix[0];
        std::vector<double2> h(P);
        for (int m = 0; m < P; ++m) {
            const long double a = 2.0L * PI_L * (long double)m / (long double)P;
            h[m].x = (double)cosl(a);
            h[m].y = (double)sinl(a);
        }
        fresnel_status st = upload_vec(&p->gen_prime_roots, h);
        if (st != FRESNEL_OK) return st;
    }
    p->generic = true;
    p->fuse = 0;
    // selected sizes (2800 = 5*5*7*16, ...) have a register-resident pass; its column tiles are TMA tiles of its own width
    const int wmr = mr_col_width(N, es);
    if (wmr > 0 && p->gen_tma && std::getenv("FRESNEL_NO_MR") == nullptr) {
        p->mr = true;
        p->gen_wcol = wmr;
    }
    return p->dtype == FRESNEL_C128 ? build_generic_tables<double2>(p, bluestein) : build_generic_tables<float2>(p, bluestein);
}

// ---- TMA tensor maps -------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled_fn()
{
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *ptr = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)ptr;
        else
            cudaGetLastError();
    }
    return fn;
}

int query_tma_width(int N, fresnel_dtype dt, bool conv2)
{
    switch (N) {
#define FR_CASE(NN) case NN: return dt == FRESNEL_C128 ? col_tma_width_f64_##NN(conv2) : col_tma_width_f32_##NN(conv2);
        FR_CASE(64) FR_CASE(128) FR_CASE(256) FR_CASE(512) FR_CASE(1024) FR_CASE(2048) FR_CASE(4096) FR_CASE(8192)
#undef FR_CASE
    }
    return 0;
}

int query_map_box(int N, fresnel_dtype dt)
{
    switch (N) {
#define FR_CASE(NN) case NN: return dt == FRESNEL_C128 ? col_tma_map_box_f64_##NN() : col_tma_map_box_f32_##NN();
        FR_CASE(64) FR_CASE(128) FR_CASE(256) FR_CASE(512) FR_CASE(1024) FR_CASE(2048) FR_CASE(4096) FR_CASE(8192)
#undef FR_CASE
    }
    return 0;
}

// The wavefront as a 3-D tensor {2N scalars, N rows, batch}; a box is {2W scalars, 256 rows, 1}.
bool make_tensor_map(fresnel_plan *p, void *wf, bool conv2 = false)
{
    const int tma_w = conv2 ? p->tma_w2 : p->tma_w;
    if (conv2 && tma_w == p->tma_w) {                     // same tile geometry: one tensor map serves both
        if (!make_tensor_map(p, wf, false)) return false;
        p->tmap2 = p->tmap;
        p->tmap2_wf = wf;
        return true;
    }
    if ((conv2 ? p->tmap2_wf : p->tmap_wf) == wf) return true;
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return false;
    const bool dbl = p->dtype == FRESNEL_C128;
    const size_t es = p->esize();
    const cuuint64_t N = (cuuint64_t)p->N;
    cuuint64_t gdim[3] = {2 * N, N, (cuuint64_t)p->batch};
    cuuint64_t gstr[2] = {N * es, N * N * es};
    cuuint32_t box[3] = {(cuuint32_t)(2 * tma_w), p->generic ? (cuuint32_t)p->gen_box_rows : 256u, 1u};
    cuuint32_t estr[3] = {1, 1, 1};
    const size_t row_bytes = (size_t)tma_w * es;
    CUtensorMapSwizzle sw = (p->generic && !p->mr) ? CU_TENSOR_MAP_SWIZZLE_NONE
                          : row_bytes == 32 ? CU_TENSOR_MAP_SWIZZLE_32B
                          : row_bytes == 64 ? CU_TENSOR_MAP_SWIZZLE_64B
                          : row_bytes == 128 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE;
    CUresult r = fn(conv2 ? &p->tmap2 : &p->tmap, dbl ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, wf, gdim,
                    gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, sw, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return false;
    (conv2 ? p->tmap2_wf : p->tmap_wf) = wf;
    return true;
}

// A real [N][N] surface map as a 2-D tensor {N, N}; a box is {map_box columns, 256 rows} (fused column pass).
const CUtensorMap *map_tensor_map(fresnel_plan *p, const void *m)
{
    ++p->clock;
    for (MapDesc &d : p->map_descs)
        if (d.ptr == m) { d.stamp = p->clock; return &d.map; }
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return nullptr;
    MapDesc d;
    const bool dbl = p->dtype == FRESNEL_C128;
    const size_t rs = dbl ? sizeof(double) : sizeof(float);
    const cuuint64_t N = (cuuint64_t)p->N;
    cuuint64_t gdim[2] = {N, N};
    cuuint64_t gstr[1] = {N * rs};
    cuuint32_t box[2] = {(cuuint32_t)p->map_box, 256u};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(&d.map, dbl ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void *>(m), gdim, gstr,
                    box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return nullptr;
    d.ptr = m;
    d.stamp = p->clock;
    if ((int)p->map_descs.size() < kMaxMapDescs) {
        p->map_descs.push_back(d);
        return &p->map_descs.back().map;
    }
    size_t victim = 0;
    for (size_t i = 1; i < p->map_descs.size(); ++i)
        if (p->map_descs[i].stamp < p->map_descs[victim].stamp) victim = i;
    p->map_descs[victim] = d;
    return &p->map_descs[victim].map;
}

// ---- pass launch by (dtype, N) ---------------------------------------------------------------------
// Everything one pass kernel may be asked to do (see pass_kernel.cuh); tables are device pointers of the plan's dtype.
struct PassSpec {
    bool col = false;
    int mode = MODE_CONV;
    const void *pre = nullptr, *rowfac = nullptr, *mid = nullptr;
    const void *amp = nullptr, *opd = nullptr;          // load-side optic (row pass only)
    const void *lens2 = nullptr, *mid2 = nullptr;       // MODE_CONV2
    const void *amp2 = nullptr, *opd2 = nullptr;
    const double *inv_lambda = nullptr;
    double scale = 1.0;
};

template <typename T> cudaError_t run_generic(fresnel_plan *p, void *wf, const PassSpec &q)
{
    using C = typename cplx_of<T>::type;
    GenArgs<T> a;
    std::memset(&a, 0, sizeof(a));
    const bool tma = q.col && p->gen_tma && make_tensor_map(p, wf);
    a.wf = (C *)wf; a.N = p->N; a.M = p->gen_M; a.W = q.col ? p->gen_wcol : 1; a.mode = q.mode;
    a.col = q.col ? (tma ? 1 : 2) : 0;
    a.box_rows = p->gen_box_rows;
    a.nstages = p->gen_nstages;
    for (int i = 0; i < p->gen_nstages; ++i) a.radix[i] = p->gen_radix[i];
    a.tw = (const C *)p->gen_tw; a.blu_w = (const C *)p->gen_blu_w; a.blu_b = (const C *)p->gen_blu_b;
    a.prime_roots = (const double2 *)p->gen_prime_roots;
    a.pre = (const C *)q.pre; a.mid = (const C *)q.mid; a.rowfac = (const C *)q.rowfac;
    a.amp = (const T *)q.amp; a.opd = (const T *)q.opd; a.inv_lambda = q.inv_lambda;
    a.scale = (T)q.scale; a.pdl = p->pdl;
    if (p->mr && (!q.col || tma)) {
        if constexpr (sizeof(T) == 8) return launch_mr_f64(p->N, q.col, q.mode, a, p->tmap, p->batch, p->stream);
        else return launch_mr_f32(p->N, q.col, q.mode, a, p->tmap, p->batch, p->stream);
    }
    if constexpr (sizeof(T) == 8) return launch_gen_pass_f64(a, p->tmap, p->batch, gen_smem(p, a.W), p->stream);
    else return launch_gen_pass_f32(a, p->tmap, p->batch, gen_smem(p, a.W), p->stream);
}

fresnel_status run_pass(fresnel_plan *p, void *wf, const PassSpec &q)
{
    cudaError_t e = cudaErrorInvalidValue;
    if (p->generic) {
        e = p->dtype == FRESNEL_C128 ? run_generic<double>(p, wf, q) : run_generic<float>(p, wf, q);
        if (e != cudaSuccess) return FRESNEL_ERR_CUDA;
        ++p->launches;
        return FRESNEL_OK;
    }
    const bool conv2 = q.mode == MODE_CONV2;
    const bool tma = q.col && p->tma_w > 0 && make_tensor_map(p, wf, conv2);
    const CUtensorMap &wmap = conv2 ? p->tmap2 : p->tmap;
    const CUtensorMap *ma = &wmap, *mo = &wmap;
    if (tma && q.mode == MODE_CONV2) {
        if (q.amp2 && !(ma = map_tensor_map(p, q.amp2))) return FRESNEL_ERR_CUDA;
        if (q.opd2 && !(mo = map_tensor_map(p, q.opd2))) return FRESNEL_ERR_CUDA;
    }
    // L2 prefetch of upcoming rows pays when the data does not already sit in the 126 MB L2 (measured:
    // +10..17 % at N >= 4096, -4 % at N = 2048 without maps); TMA tile prefetch of 16..32-byte-wide
    // column boxes costs more TMA issue slots than it saves and stays off.
    const size_t wf_bytes = (size_t)p->batch * p->N * p->N * p->esize();
    const int prefetch = (!q.col && (wf_bytes > ((size_t)64 << 20) || q.amp || q.opd)) ? p->prefetch : 0;
    if (p->dtype == FRESNEL_C128) {
        PassArgs<double> a;
        a.wf = (double2 *)wf; a.pre = (const double2 *)q.pre; a.mid = (const double2 *)q.mid; a.rowfac = (const double2 *)q.rowfac;
        a.tw = (const double2 *)p->tw; a.amp = (const double *)q.amp; a.opd = (const double *)q.opd;
        a.inv_lambda = q.inv_lambda; a.scale = q.scale; a.prefetch_distance = prefetch; a.pdl = p->pdl;
        a.lens2 = (const double2 *)q.lens2; a.mid2 = (const double2 *)q.mid2; a.amp2 = (const double *)q.amp2; a.opd2 = (const double *)q.opd2;
        switch (p->N) {
#define FR_CASE(NN) case NN: e = tma ? launch_col_tma_f64_##NN(q.mode, a, wmap, *ma, *mo, p->batch, p->stream)           \
                                   : launch_pass_f64_##NN(q.col, q.mode, a, p->batch, p->stream); break;
            FR_CASE(64) FR_CASE(128) FR_CASE(256) FR_CASE(512) FR_CASE(1024) FR_CASE(2048) FR_CASE(4096) FR_CASE(8192)
#undef FR_CASE
        }
    } else {
        PassArgs<float> a;
        a.wf = (float2 *)wf; a.pre = (const float2 *)q.pre; a.mid = (const float2 *)q.mid; a.rowfac = (const float2 *)q.rowfac;
        a.tw = (const float2 *)p->tw; a.amp = (const float *)q.amp; a.opd = (const float *)q.opd;
        a.inv_lambda = q.inv_lambda; a.scale = (float)q.scale; a.prefetch_distance = prefetch; a.pdl = p->pdl;
        a.lens2 = (const float2 *)q.lens2; a.mid2 = (const float2 *)q.mid2; a.amp2 = (const float *)q.amp2; a.opd2 = (const float *)q.opd2;
        switch (p->N) {
#define FR_CASE(NN) case NN: e = tma ? launch_col_tma_f32_##NN(q.mode, a, wmap, *ma, *mo, p->batch, p->stream)           \
                                   : launch_pass_f32_##NN(q.col, q.mode, a, p->batch, p->stream); break;
            FR_CASE(64) FR_CASE(128) FR_CASE(256) FR_CASE(512) FR_CASE(1024) FR_CASE(2048) FR_CASE(4096) FR_CASE(8192)
#undef FR_CASE
        }
    }
    if (e != cudaSuccess) return FRESNEL_ERR_CUDA;
    ++p->launches;
    return FRESNEL_OK;
}

// profiling hook of fresnel_system_run: event k before pass kernel k of the train, one more after the last
void train_event(fresnel_plan *p, size_t k)
{
    if (k < p->train_ev.size()) cudaEventRecord(p->train_ev[k], p->stream);
}

void note_pass(fresnel_plan *p, int direction, int nconv, int surface, int maps)
{
    fresnel_pass_info i;
    i.direction = direction;
    i.convolutions = nconv;
    i.first_surface = surface;
    i.maps_read = maps;
    p->schedule.push_back(i);
}

// The two HBM round trips of a propagation / transform: row pass then column pass.
fresnel_status run_two_passes(fresnel_plan *p, int mode, void *wf, const void *pre, const void *mid,
                              const void *amp, const void *opd, const double *inv_lambda, double scale, int surface = -1)
{
    const bool ev = p->ev_armed;
    p->ev_armed = false;
    if (ev && cudaEventRecord(p->ev[0], p->stream) != cudaSuccess) return FRESNEL_ERR_CUDA;
    // the input chirp is separable: its x-part rides on the load of the row pass, its y-part (one factor per
    // row) on the store of the row pass, so the column pass has no input table at all
    PassSpec r;
    r.col = false; r.mode = mode; r.pre = pre; r.rowfac = pre; r.mid = mid; r.amp = amp; r.opd = opd;
    r.inv_lambda = inv_lambda; r.scale = scale;
    if (surface >= 0) { train_event(p, p->schedule.size()); note_pass(p, 0, mode == MODE_CONV ? 1 : 0, surface, (amp != nullptr) + (opd != nullptr)); }
    fresnel_status st = run_pass(p, wf, r);
    if (st != FRESNEL_OK) return st;
    if (ev && cudaEventRecord(p->ev[1], p->stream) != cudaSuccess) return FRESNEL_ERR_CUDA;
    PassSpec c;
    c.col = true; c.mode = mode; c.mid = mid; c.scale = scale;
    if (surface >= 0) { train_event(p, p->schedule.size()); note_pass(p, 1, mode == MODE_CONV ? 1 : 0, surface, 0); }
    st = run_pass(p, wf, c);
    if (st != FRESNEL_OK) return st;
    if (ev && cudaEventRecord(p->ev[2], p->stream) != cudaSuccess) return FRESNEL_ERR_CUDA;
    return FRESNEL_OK;
}

fresnel_status run_pointwise(fresnel_plan *p, void *wf, const void *tab, const void *amp, const void *opd, const double *inv_lambda)
{
    cudaError_t e;
    if (p->dtype == FRESNEL_C128)
        e = launch_pointwise<double>((double2 *)wf, (const double2 *)tab, (const double *)amp, (const double *)opd,
                                     inv_lambda, p->N, p->batch, p->stream);
    else
        e = launch_pointwise<float>((float2 *)wf, (const float2 *)tab, (const float *)amp, (const float *)opd,
                                    inv_lambda, p->N, p->batch, p->stream);
    if (e != cudaSuccess) return FRESNEL_ERR_CUDA;
    ++p->launches;
    return FRESNEL_OK;
}

// chirp coefficient (turns per pixel^2) of exp(i pi x^2/(lambda z)), x = m*dx:  dx^2/(2 lambda z)
long double qpf_coeff(double dx, double lambda, long double z)
{
    return (long double)dx * (long double)dx / (2.0L * (long double)lambda * z);
}
// transfer function exp(-i pi lambda z f^2), f = m/(N dx):  -lambda z/(2 N^2 dx^2) turns per index^2
long double as_coeff(int N, double dx, double lambda, double z)
{
    long double nd = (long double)N * (long double)dx;
    return -(long double)lambda * (long double)z / (2.0L * nd * nd);
}

// Constant phase (turns) a centred 1-D transform of an ODD grid carries besides its two ramps: -+ (h^2 mod N)/N,
// h = N/2, for the forward (alt = +1) / inverse (alt = -1) kernel.  Even grids: the 2-D product of the constants is 1.
double centred_phase0(int N, int alt)
{
    if ((N & 1) == 0) return 0.0;
    const long long h = N / 2;
    const double fr = (double)((h * h) % N) / (double)N;
    return alt > 0 ? -fr : fr;
}

// chirp exp(i pi r^2 kappa / lambda) as a table coefficient (turns per pixel^2): kappa dx^2 / (2 lambda); a thin lens is kappa = -1/f
long double curvature_coeff(double dx, double lambda, long double kappa)
{
    return kappa * (long double)dx * (long double)dx / (2.0L * (long double)lambda);
}

std::vector<ChirpSpec> lens_key(const fresnel_plan *p, const double *pixel, const double *lambda, double f)
{
    std::vector<ChirpSpec> key(p->batch);
    for (int b = 0; b < p->batch; ++b) key[b] = make_spec(qpf_coeff(pixel[b], lambda[b], -(long double)f), 1.0, 0.0);
    return key;
}
std::vector<ChirpSpec> transfer_key(const fresnel_plan *p, const double *pixel, const double *lambda, double z)
{
    std::vector<ChirpSpec> key(p->batch);
    for (int b = 0; b < p->batch; ++b) key[b] = make_spec(as_coeff(p->N, pixel[b], lambda[b], z), 1.0 / (double)p->N, 0.0);
    return key;
}

// ---- angular-spectrum leg: [chirp] -> [optic phasor] -> propagation, two passes ----------------------------------
// chirp_key: the table of the input chirp (a thin lens, or the residual reference curvature of the pilot-beam rule),
// empty for none; z: per batch element (all zero: optic only).
fresnel_status as_leg(fresnel_plan *p, void *wf, const double *pixel, const double *lambda, const std::vector<ChirpSpec> &chirp_key,
                      const void *amp, const void *opd, const double *z, int surface)
{
    ++p->pin_epoch;
    const CaptureState cap = capture_state(p);
    const bool lens = !chirp_key.empty();
    bool prop = false;
    for (int b = 0; b < p->batch; ++b) prop = prop || z[b] != 0.0;
    if (!lens && !prop && !amp && !opd) return FRESNEL_OK;

    TableRequest r[3];
    int nreq = 0, i_lens = -1, i_h = -1, i_s = -1;
    if (lens) { i_lens = nreq; r[nreq++] = request_table(p, KIND_CENTRED, 0, chirp_key, cap); }
    if (prop) {
        std::vector<ChirpSpec> key(p->batch);
        for (int b = 0; b < p->batch; ++b) key[b] = make_spec(as_coeff(p->N, pixel[b], lambda[b], z[b]), 1.0 / (double)p->N, 0.0);
        i_h = nreq;
        r[nreq++] = request_table(p, KIND_FFTORDER, 0, key, cap);
    }
    if (opd) { i_s = nreq; r[nreq++] = request_inv_lambda(p, lambda, cap); }
    fresnel_status st = flush_builds(p, r, nreq);
    if (st != FRESNEL_OK) return st;
    const void *tl = lens ? p->slots[r[i_lens].slot].dev : nullptr;
    const double *il = opd ? (const double *)p->slots[r[i_s].slot].dev : nullptr;
    if (!prop) {                                                   // optic only
        if (surface >= 0) { train_event(p, p->schedule.size()); note_pass(p, 0, 0, surface, (amp != nullptr) + (opd != nullptr)); }
        return run_pointwise(p, wf, tl, amp, opd, il);
    }
    const void *th = p->slots[r[i_h].slot].dev;
    // row pass: optic phasor and x-chirp of the lens on load, FFT, x H1, inverse FFT, y-chirp of the lens (one
    // factor per row) on store;  column pass: FFT, x H1, inverse FFT
    return run_two_passes(p, MODE_CONV, wf, tl, th, amp, opd, il, 1.0, surface);
}

// one fused surface (thin lens + optic phasor + angular spectrum)
fresnel_status surface_as_impl(fresnel_plan *p, void *wf, const double *pixel, const double *lambda,
                               double f, const void *amp, const void *opd, double z, int surface = -1)
{
    std::vector<double> zb(p->batch, z);
    return as_leg(p, wf, pixel, lambda, std::isfinite(f) ? lens_key(p, pixel, lambda, f) : std::vector<ChirpSpec>(), amp, opd, zb.data(), surface);
}

// ---- single-transform leg: [extra chirp] -> [optic phasor] -> centred transform with the Fresnel factors ----------
//   FT_DIRECT  direct Fresnel: input chirp Q_dx(dz), transform, dx^2/(i lambda dz), output chirp Q_dx'(dz);
//   FT_WTS     waist -> sphere (pilot-beam rule): no output chirp;    FT_STW   sphere -> waist: no input chirp.
// An extra chirp on the input side (a thin lens, the residual reference curvature) is the same kind of factor as the
// propagator's input chirp: the coefficients are added (long double) and ONE table serves both; the optic phasor
// rides on the row-pass load.  dz, kappa: per batch element (kappa may be null); every dz must have the same sign.
enum { FT_DIRECT = 0, FT_WTS = 1, FT_STW = 2 };

fresnel_status ft_leg(fresnel_plan *p, void *wf, double *pixel_inout, const double *lambda, const double *dz, int kind,
                      const long double *kappa, const void *amp, const void *opd, int surface)
{
    ++p->pin_epoch;
    const CaptureState cap = capture_state(p);
    const bool fwd = dz[0] > 0;
    std::vector<ChirpSpec> kin(p->batch), kout(p->batch);
    std::vector<double> dx_out(p->batch);
    for (int b = 0; b < p->batch; ++b) {
        if ((dz[b] > 0) != fwd || dz[b] == 0.0) return FRESNEL_ERR_UNSUPPORTED;
        const double dx = pixel_inout[b];
        const long double z = dz[b];
        const long double dxo = (long double)lambda[b] * fabsl(z) / ((long double)p->N * (long double)dx);
        dx_out[b] = (double)dxo;
        long double cin = kind != FT_STW ? qpf_coeff(dx, lambda[b], z) : 0.0L;
        if (kappa) cin += curvature_coeff(dx, lambda[b], kappa[b]);
        kin[b] = make_spec(cin, 1.0, 0.0);
        // per-axis share of dx^2/(i lambda z): dx/sqrt(lambda |z|) * exp(-+ i pi/4)
        const double a1 = (double)((long double)dx / sqrtl((long double)lambda[b] * fabsl(z)));
        const long double cout = kind != FT_WTS ? qpf_coeff(dx_out[b], lambda[b], z) : 0.0L;
        kout[b] = make_spec(cout, a1, (fwd ? -0.125 : 0.125) + centred_phase0(p->N, fwd ? +1 : -1));
    }
    // the (-1)^n (odd N: the phase ramp) of the centred transform rides on both tables
    TableRequest r[3];
    int nreq = 2;
    const int alt = fwd ? +1 : -1;
    r[0] = request_table(p, KIND_CENTRED, alt, kin, cap);
    r[1] = request_table(p, KIND_CENTRED, alt, kout, cap);
    if (opd) r[nreq++] = request_inv_lambda(p, lambda, cap);
    fresnel_status st = flush_builds(p, r, nreq);
    if (st != FRESNEL_OK) return st;
    const double *il = opd ? (const double *)p->slots[r[2].slot].dev : nullptr;
    st = run_two_passes(p, fwd ? MODE_FWD : MODE_INV, wf, p->slots[r[0].slot].dev, p->slots[r[1].slot].dev, amp, opd, il, 1.0, surface);
    if (st != FRESNEL_OK) return st;
    for (int b = 0; b < p->batch; ++b) pixel_inout[b] = dx_out[b];
    return FRESNEL_OK;
}

// [thin lens f] -> [optic phasor] -> direct Fresnel propagation by z
fresnel_status direct_impl(fresnel_plan *p, void *wf, double *pixel_inout, const double *lambda, double z,
                           double f, const void *amp, const void *opd, int surface = -1)
{
    std::vector<double> zb(p->batch, z);
    std::vector<long double> kappa;
    if (std::isfinite(f)) kappa.assign(p->batch, -1.0L / (long double)f);
    return ft_leg(p, wf, pixel_inout, lambda, zb.data(), FT_DIRECT, kappa.empty() ? nullptr : kappa.data(), amp, opd, surface);
}

// ---- a run of consecutive angular-spectrum surfaces, fused at train level ---------------------------------------
// Surfaces s0 .. s0+L-1 (all with z != 0, same pixel pitch).  Row and column convolution of a surface commute, so the
// passes are ordered
//     rows_0 (with optic_0 on load) | cols_0, optic_1, cols_1 | rows_1, optic_2, rows_2 | ... | last convolution
// i.e. L+1 kernels instead of 2L: kernel k (1 <= k < L) runs along columns for odd k and along rows for even k and
// holds every line resident through  conv_{k-1} -> optic_k -> conv_k  (MODE_CONV2).
fresnel_status fused_chain(fresnel_plan *p, void *wf, const double *pixel, const double *lambda,
                           const fresnel_surface *surf, int s0, int L)
{
    ++p->pin_epoch;
    const CaptureState cap = capture_state(p);
    std::vector<TableRequest> req;
    std::vector<int> i_lens(L, -1), i_h(L, -1);
    int i_s = -1;
    bool any_opd = false;
    for (int k = 0; k < L; ++k) {
        const fresnel_surface &q = surf[s0 + k];
        if (std::isfinite(q.f)) { i_lens[k] = (int)req.size(); req.push_back(request_table(p, KIND_CENTRED, 0, lens_key(p, pixel, lambda, q.f), cap)); }
        i_h[k] = (int)req.size();
        req.push_back(request_table(p, KIND_FFTORDER, 0, transfer_key(p, pixel, lambda, q.z), cap));
        any_opd = any_opd || q.opd != nullptr;
    }
    if (any_opd) { i_s = (int)req.size(); req.push_back(request_inv_lambda(p, lambda, cap)); }
    fresnel_status st = flush_builds(p, req.data(), (int)req.size());
    if (st != FRESNEL_OK) return st;
    auto lens = [&](int k) -> const void * { return i_lens[k] >= 0 ? p->slots[req[i_lens[k]].slot].dev : nullptr; };
    auto H = [&](int k) -> const void * { return p->slots[req[i_h[k]].slot].dev; };
    const double *il = any_opd ? (const double *)p->slots[req[i_s].slot].dev : nullptr;

    for (int k = 0; k <= L; ++k) {
        PassSpec q;
        q.col = (k & 1) != 0;
        q.inv_lambda = il;
        int maps = 0;
        if (k == 0) {                       // optic_0 on load, rows_0
            const fresnel_surface &s = surf[s0];
            q.mode = MODE_CONV; q.pre = lens(0); q.rowfac = lens(0); q.mid = H(0); q.amp = s.amp; q.opd = s.opd;
            maps = (s.amp != nullptr) + (s.opd != nullptr);
        } else if (k < L) {                 // conv_{k-1}, optic_k, conv_k along the same direction
            const fresnel_surface &s = surf[s0 + k];
            q.mode = MODE_CONV2; q.mid = H(k - 1); q.lens2 = lens(k); q.amp2 = s.amp; q.opd2 = s.opd; q.mid2 = H(k);
            maps = (s.amp != nullptr) + (s.opd != nullptr);
        } else {                            // the remaining convolution of the last surface
            q.mode = MODE_CONV; q.mid = H(L - 1);
        }
        train_event(p, p->schedule.size());
        note_pass(p, q.col ? 1 : 0, (k > 0 && k < L) ? 2 : 1, s0 + (k < L ? k : L - 1), maps);
        st = run_pass(p, wf, q);
        if (st != FRESNEL_OK) return st;
    }
    return FRESNEL_OK;
}

} // namespace

// =====================================================================================================
extern "C" {

const char *fresnel_status_string(fresnel_status s)
{
    switch (s) {
    case FRESNEL_OK: return "FRESNEL_OK";
    case FRESNEL_ERR_INVALID_ARG: return "FRESNEL_ERR_INVALID_ARG";
    case FRESNEL_ERR_UNSUPPORTED: return "FRESNEL_ERR_UNSUPPORTED";
    case FRESNEL_ERR_ALLOC: return "FRESNEL_ERR_ALLOC";
    case FRESNEL_ERR_CUDA: return "FRESNEL_ERR_CUDA";
    case FRESNEL_ERR_TOO_LARGE: return "FRESNEL_ERR_TOO_LARGE";
    }
    return "FRESNEL_ERR_UNKNOWN";
}

const char *fresnel_version(void) { return "fresnel-b200 0.2 sm_100a"; }

fresnel_status fresnel_plan_create(fresnel_plan **out, int N, int batch, fresnel_dtype dtype)
{
    if (!out || batch <= 0 || N <= 0) return FRESNEL_ERR_INVALID_ARG;
    if (dtype != FRESNEL_C64 && dtype != FRESNEL_C128) return FRESNEL_ERR_UNSUPPORTED;
    if (N < 16 || N > 8192 || (is_pow2(N) && N < 64)) return FRESNEL_ERR_UNSUPPORTED;
    if (!is_pow2(N) && !generic_supported(N, dtype)) return FRESNEL_ERR_UNSUPPORTED;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0) { cudaGetLastError(); return FRESNEL_ERR_CUDA; }
    fresnel_plan *p = new (std::nothrow) fresnel_plan();
    if (!p) return FRESNEL_ERR_ALLOC;
    p->N = N; p->batch = batch; p->dtype = dtype;
    {
        int sms = 148;
        cudaGetDevice(&p->device);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, p->device);
        p->sms = sms;
        const char *pf = std::getenv("FRESNEL_PREFETCH");          // tuning only: tiles ahead, 0 = off
        p->prefetch = pf ? std::atoi(pf) : -sms;                   // negative: auto = SMs x resident CTAs per SM
    }
    { const char *pd = std::getenv("FRESNEL_PDL"); p->pdl = pd ? std::atoi(pd) : 1; }
    { const char *fu = std::getenv("FRESNEL_FUSE"); p->fuse = fu ? std::atoi(fu) : 1; }
    p->map_descs.reserve(kMaxMapDescs);                            // pointers into it are handed out
    fresnel_status st;
    if (is_pow2(N)) {
        p->tma_w = std::getenv("FRESNEL_NO_TMA") ? 0 : query_tma_width(N, dtype, false);     // env switch: A/B timing only
        p->tma_w2 = p->tma_w > 0 ? query_tma_width(N, dtype, true) : 0;
        p->map_box = query_map_box(N, dtype);
        st = upload_twiddles(p);
    } else {
        st = setup_generic(p);                                     // mixed radix / Bluestein (gen_kernel.cuh)
        p->tma_w = p->gen_wcol;
    }
    if (st == FRESNEL_OK && cudaEventCreateWithFlags(&p->order_ev, cudaEventDisableTiming) != cudaSuccess) st = FRESNEL_ERR_CUDA;
    if (st == FRESNEL_OK) st = grow_slots(p, kDefaultSlots);
    if (st != FRESNEL_OK) { cudaGetLastError(); fresnel_plan_destroy(p); return st; }
    *out = p;
    return FRESNEL_OK;
}

fresnel_status fresnel_plan_reserve_tables(fresnel_plan *p, int n_tables)
{
    if (!p || n_tables < 0) return FRESNEL_ERR_INVALID_ARG;
    DeviceGuard g(p);
    if (capture_state(p).active) return FRESNEL_ERR_UNSUPPORTED;  // allocates: not while capturing
    return grow_slots(p, n_tables - eager_slot_count(p));
}

fresnel_status fresnel_plan_release_graph_tables(fresnel_plan *p)
{
    if (!p) return FRESNEL_ERR_INVALID_ARG;
    for (TableSlot &s : p->slots)
        if (s.graph_owned) { s.graph_owned = false; s.valid = false; s.capture_id = 0; }
    return FRESNEL_OK;
}

fresnel_status fresnel_plan_set_stream(fresnel_plan *p, void *cuda_stream)
{
    if (!p) return FRESNEL_ERR_INVALID_ARG;
    DeviceGuard g(p);
    cudaStream_t ns = (cudaStream_t)cuda_stream;
    if (ns == p->stream) return FRESNEL_OK;
    // Tables built (and kernels reading them) on the old stream must precede whatever the new stream does with the
    // same slots: the new stream waits for the old one's tail.  Not possible across a capture boundary.
    cudaStreamCaptureStatus so = cudaStreamCaptureStatusNone, sn = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(p->stream, &so) != cudaSuccess) { cudaGetLastError(); so = cudaStreamCaptureStatusNone; }
    if (cudaStreamIsCapturing(ns, &sn) != cudaSuccess) { cudaGetLastError(); sn = cudaStreamCaptureStatusNone; }
    if (so == cudaStreamCaptureStatusNone && sn == cudaStreamCaptureStatusNone) {
        if (cudaEventRecord(p->order_ev, p->stream) != cudaSuccess || cudaStreamWaitEvent(ns, p->order_ev, 0) != cudaSuccess) {
            cudaGetLastError();
            return FRESNEL_ERR_CUDA;
        }
    } else {
        for (TableSlot &s : p->slots)                              // cannot be ordered: forget the eager tables
            if (!s.graph_owned) s.valid = false;
    }
    p->stream = ns;
    return FRESNEL_OK;
}

fresnel_status fresnel_plan_synchronize(fresnel_plan *p)
{
    if (!p) return FRESNEL_ERR_INVALID_ARG;
    DeviceGuard g(p);
    return cudaStreamSynchronize(p->stream) == cudaSuccess ? FRESNEL_OK : FRESNEL_ERR_CUDA;
}

fresnel_status fresnel_plan_destroy(fresnel_plan *p)
{
    if (!p) return FRESNEL_OK;
    {
        DeviceGuard g(p);
        cudaStreamSynchronize(p->stream);
        cudaFree(p->tw);
        cudaFree(p->gen_tw);
        cudaFree(p->gen_blu_w);
        cudaFree(p->gen_blu_b);
        cudaFree(p->gen_prime_roots);
        cudaFree(p->mft_e);
        cudaFree(p->mft_t);
        cudaFree(p->mft_scal);
        for (void *a : p->arenas) cudaFree(a);
        if (p->order_ev) cudaEventDestroy(p->order_ev);
        cudaGetLastError();
    }
    delete p;
    return FRESNEL_OK;
}

fresnel_status fresnel_plan_launch_count(const fresnel_plan *p, unsigned long long *count)
{
    if (!p || !count) return FRESNEL_ERR_INVALID_ARG;
    *count = p->launches;
    return FRESNEL_OK;
}

fresnel_status fresnel_plan_record_pass_events(fresnel_plan *p, void *const events[3])
{
    if (!p) return FRESNEL_ERR_INVALID_ARG;
    if (!events) { p->ev_armed = false; return FRESNEL_OK; }
    for (int i = 0; i < 3; ++i) {
        if (!events[i]) return FRESNEL_ERR_INVALID_ARG;
        p->ev[i] = (cudaEvent_t)events[i];
    }
    p->ev_armed = true;
    return FRESNEL_OK;
}

fresnel_status fresnel_plan_record_train_events(fresnel_plan *p, void *const *events, int n_events)
{
    if (!p || n_events < 0 || (n_events > 0 && !events)) return FRESNEL_ERR_INVALID_ARG;
    p->train_ev.clear();
    for (int i = 0; i < n_events; ++i) {
        if (!events[i]) { p->train_ev.clear(); return FRESNEL_ERR_INVALID_ARG; }
        p->train_ev.push_back((cudaEvent_t)events[i]);
    }
    return FRESNEL_OK;
}

fresnel_status fresnel_plan_last_schedule(const fresnel_plan *p, fresnel_pass_info *out, int capacity, int *count)
{
    if (!p || !count || capacity < 0 || (capacity > 0 && !out)) return FRESNEL_ERR_INVALID_ARG;
    *count = (int)p->schedule.size();
    for (int i = 0; i < capacity && i < *count; ++i) out[i] = p->schedule[i];
    return FRESNEL_OK;
}

fresnel_status fresnel_memcpy_h2d(fresnel_plan *p, void *dst_device, const void *src_host, size_t bytes)
{
    if (!p || !dst_device || !src_host) return FRESNEL_ERR_INVALID_ARG;
    DeviceGuard g(p);
    return cudaMemcpyAsync(dst_device, src_host, bytes, cudaMemcpyHostToDevice, p->stream) == cudaSuccess ? FRESNEL_OK : FRESNEL_ERR_CUDA;
}

fresnel_status fresnel_memcpy_d2h(fresnel_plan *p, void *dst_host, const void *src_device, size_t bytes)
{
    if (!p || !dst_host || !src_device) return FRESNEL_ERR_INVALID_ARG;
    DeviceGuard g(p);
    return cudaMemcpyAsync(dst_host, src_device, bytes, cudaMemcpyDeviceToHost, p->stream) == cudaSuccess ? FRESNEL_OK : FRESNEL_ERR_CUDA;
}

// ---- Eq. 2: quadratic phase factor ------------------------------------------------------------------
fresnel_status fresnel_apply_qpf(fresnel_plan *p, void *wf, const double *pixel, const double *lambda, double z)
{
    if (!p || !wf || !valid_positive(pixel, p ? p->batch : 0) || !valid_positive(lambda, p->batch)) return FRESNEL_ERR_INVALID_ARG;
    if (!std::isfinite(z) || z == 0.0) return FRESNEL_ERR_INVALID_ARG;
    DeviceGuard g(p);
    ++p->pin_epoch;
    const CaptureState cap = capture_state(p);
    std::vector<ChirpSpec> key(p->batch);
    for (int b = 0; b < p->batch; ++b) key[b] = make_spec(qpf_coeff(pixel[b], lambda[b], z), 1.0, 0.0);
    TableRequest r = request_table(p, KIND_CENTRED, 0, key, cap);
    fresnel_status st = flush_builds(p, &r, 1);
    if (st != FRESNEL_OK) return st;
    return run_pointwise(p, wf, p->slots[r.slot].dev, nullptr, nullptr, nullptr);
}

// ---- Eq. 3: optic phasor ------------------------------------------------------------------------------
fresnel_status fresnel_apply_mask(fresnel_plan *p, void *wf, const void *amp, const void *opd, const double *lambda)
{
    if (!p || !wf || !valid_positive(lambda, p ? p->batch : 0)) return FRESNEL_ERR_INVALID_ARG;
    if (!amp && !opd) return FRESNEL_OK;
    DeviceGuard g(p);
    ++p->pin_epoch;
    const double *il = nullptr;
    if (opd) {
        TableRequest r = request_inv_lambda(p, lambda, capture_state(p));
        fresnel_status st = flush_builds(p, &r, 1);
        if (st != FRESNEL_OK) return st;
        il = (const double *)p->slots[r.slot].dev;
    }
    return run_pointwise(p, wf, nullptr, amp, opd, il);
}

// ---- 2-D FFT ---------------------------------------------------------------------------------------------
fresnel_status fresnel_fft2d(fresnel_plan *p, void *wf, int direction, int centered)
{
    if (!p || !wf || (direction != FRESNEL_FORWARD && direction != FRESNEL_INVERSE)) return FRESNEL_ERR_INVALID_ARG;
    DeviceGuard g(p);
    ++p->pin_epoch;
    const int mode = direction == FRESNEL_FORWARD ? MODE_FWD : MODE_INV;
    const double per_pass = direction == FRESNEL_FORWARD ? 1.0 : 1.0 / (double)p->N;
    if (!centered) {
        return run_two_passes(p, mode, wf, nullptr, nullptr, nullptr, nullptr, nullptr, per_pass);
    }
    // centred transform = s * fft2(s * u), s = (-1)^(j+k): sign tables on load and after the transform
    // (odd N: phase ramps exp(+-2 pi i h n/N), h = N/2, and the constant exp(-+2 pi i h^2/N) per dimension)
    const CaptureState cap = capture_state(p);
    const int alt = mode == MODE_FWD ? +1 : -1;
    std::vector<ChirpSpec> k1(p->batch, make_spec(0.0L, 1.0, 0.0)), k2(p->batch, make_spec(0.0L, per_pass, centred_phase0(p->N, alt)));
    TableRequest r[2];
    r[0] = request_table(p, KIND_CENTRED, alt, k1, cap);
    r[1] = request_table(p, KIND_CENTRED, alt, k2, cap);
    fresnel_status st = flush_builds(p, r, 2);
    if (st != FRESNEL_OK) return st;
    return run_two_passes(p, mode, wf, p->slots[r[0].slot].dev, p->slots[r[1].slot].dev, nullptr, nullptr, nullptr, 1.0);
}

// ---- fused surface: lens + optic phasor + angular-spectrum propagation ----------------------------
fresnel_status fresnel_surface_as(fresnel_plan *p, void *wf, const double *pixel, const double *lambda,
                                  double f, const void *amp, const void *opd, double z)
{
    if (!p || !wf || !valid_positive(pixel, p ? p->batch : 0) || !valid_positive(lambda, p->batch)) return FRESNEL_ERR_INVALID_ARG;
    if (!std::isfinite(z) || std::isnan(f) || f == 0.0) return FRESNEL_ERR_INVALID_ARG;
    DeviceGuard g(p);
    return surface_as_impl(p, wf, pixel, lambda, f, amp, opd, z);
}

fresnel_status fresnel_propagate_as(fresnel_plan *p, void *wf, const double *pixel, const double *lambda, double z)
{
    return fresnel_surface_as(p, wf, pixel, lambda, INFINITY, nullptr, nullptr, z);
}

// ---- direct (single-FFT) Fresnel ---------------------------------------------------------------------
fresnel_status fresnel_propagate_direct(fresnel_plan *p, void *wf, double *pixel_inout, const double *lambda, double z)
{
    if (!p || !wf || !valid_positive(pixel_inout, p ? p->batch : 0) || !valid_positive(lambda, p->batch)) return FRESNEL_ERR_INVALID_ARG;
    if (!std::isfinite(z) || z == 0.0) return FRESNEL_ERR_INVALID_ARG;
    DeviceGuard g(p);
    return direct_impl(p, wf, pixel_inout, lambda, z, INFINITY, nullptr, nullptr);
}

// ---- train of surfaces ---------------------------------------------------------------------------------
fresnel_status fresnel_system_run(fresnel_plan *p, void *wf, double *pixel_inout, const double *lambda,
                                  const fresnel_surface *surf, int nsurf, int *method_used)
{
    if (!p || !wf || nsurf < 0 || (nsurf > 0 && !surf)) return FRESNEL_ERR_INVALID_ARG;
    if (!valid_positive(pixel_inout, p->batch) || !valid_positive(lambda, p->batch)) return FRESNEL_ERR_INVALID_ARG;
    DeviceGuard g(p);
    // dry run on the host: validate everything and fix the propagator of every surface before anything is enqueued
    std::vector<int> method(nsurf);
    std::vector<long double> dx(p->batch);
    for (int b = 0; b < p->batch; ++b) dx[b] = pixel_inout[b];
    for (int s = 0; s < nsurf; ++s) {
        const fresnel_surface &q = surf[s];
        if (std::isnan(q.f) || q.f == 0.0 || !std::isfinite(q.z)) return FRESNEL_ERR_INVALID_ARG;
        if (q.method != FRESNEL_METHOD_AS && q.method != FRESNEL_METHOD_DIRECT && q.method != FRESNEL_METHOD_AUTO) return FRESNEL_ERR_INVALID_ARG;
        if (q.z == 0.0) { method[s] = -1; continue; }
        int m = q.method;
        if (m == FRESNEL_METHOD_AUTO) {
            int n_as = 0;
            for (int b = 0; b < p->batch; ++b) {
                const long double zc = (long double)p->N * dx[b] * dx[b] / (long double)lambda[b];
                if (fabsl((long double)q.z) < zc) ++n_as;
            }
            if (n_as == p->batch) m = FRESNEL_METHOD_AS;
            else if (n_as == 0) m = FRESNEL_METHOD_DIRECT;
            else return FRESNEL_ERR_UNSUPPORTED;        // the batch straddles z_c: split it or force a method
        }
        method[s] = m;
        if (m == FRESNEL_METHOD_DIRECT)
            for (int b = 0; b < p->batch; ++b) {
                dx[b] = (long double)(double)((long double)lambda[b] * fabsl((long double)q.z) / ((long double)p->N * (long double)(double)dx[b]));
                if (!(dx[b] > 0.0L) || !std::isfinite((double)dx[b])) return FRESNEL_ERR_INVALID_ARG;
            }
    }
    p->schedule.clear();
    auto finish = [&](fresnel_status st) {
        if (st == FRESNEL_OK) train_event(p, p->schedule.size());
        p->train_ev.clear();
        return st;
    };
    // a fused run needs all its tables at once (two per surface + 1/lambda): bounded by the eager slots at hand
    const int avail = eager_slot_count(p);
    const int max_run = (avail - 4) / 2;
    int s = 0;
    while (s < nsurf) {
        fresnel_status st;
        int L = 0;
        if (p->fuse && max_run >= 2)
            while (s + L < nsurf && L < max_run && method[s + L] == FRESNEL_METHOD_AS) ++L;
        if (L >= 2) {
            st = fused_chain(p, wf, pixel_inout, lambda, surf, s, L);
            if (st != FRESNEL_OK) return finish(st);
            if (method_used)
                for (int k = 0; k < L; ++k) method_used[s + k] = FRESNEL_METHOD_AS;
            s += L;
            continue;
        }
        const fresnel_surface &q = surf[s];
        if (method[s] == FRESNEL_METHOD_DIRECT) st = direct_impl(p, wf, pixel_inout, lambda, q.z, q.f, q.amp, q.opd, s);
        else st = surface_as_impl(p, wf, pixel_inout, lambda, q.f, q.amp, q.opd, q.z, s);   // z == 0: optic only
        if (st != FRESNEL_OK) return finish(st);
        if (method_used) method_used[s] = method[s];
        ++s;
    }
    return finish(FRESNEL_OK);
}

// ---- train of surfaces under the Gaussian pilot-beam rule ------------------------------------------------------
// Host-side bookkeeping per batch element in long double (the same expressions, in the same order, as the oracle's
// description of the rule in DESIGN.md reading g21); the array work is the existing two-pass kernels with other
// tables: PTP = angular-spectrum leg, WTS / STW = single-transform legs without the output / input chirp.
fresnel_status fresnel_system_run_pilot(fresnel_plan *p, void *wf, double *pixel_inout, const double *lambda,
                                        const fresnel_surface *surf, int nsurf, double rayleigh_factor,
                                        fresnel_pilot_state *state, int *legs_used)
{
    if (!p || !wf || !state || nsurf < 0 || (nsurf > 0 && !surf) || !(rayleigh_factor > 0)) return FRESNEL_ERR_INVALID_ARG;
    if (!valid_positive(pixel_inout, p->batch) || !valid_positive(lambda, p->batch)) return FRESNEL_ERR_INVALID_ARG;
    const int nb = p->batch;
    for (int b = 0; b < nb; ++b)
        if (!(state[b].w0 > 0) || !std::isfinite(state[b].zw) || !std::isfinite(state[b].z) || std::isnan(state[b].rref) || state[b].rref == 0.0)
            return FRESNEL_ERR_INVALID_ARG;
    for (int s = 0; s < nsurf; ++s)
        if (std::isnan(surf[s].f) || surf[s].f == 0.0 || !std::isfinite(surf[s].z)) return FRESNEL_ERR_INVALID_ARG;
    DeviceGuard g(p);
    const long double rf = rayleigh_factor;

    // ---- dry run: the legs of every surface, for every batch element; nothing is enqueued before the whole train is known
    struct Step { int leg[2]; bool chirp; std::vector<long double> kappa; std::vector<double> d1, d2; };
    std::vector<Step> steps(nsurf);
    std::vector<long double> w0(nb), zw(nb), zc(nb), inv_rref(nb);
    for (int b = 0; b < nb; ++b) {
        w0[b] = state[b].w0; zw[b] = state[b].zw; zc[b] = state[b].z;
        inv_rref[b] = std::isfinite(state[b].rref) ? 1.0L / (long double)state[b].rref : 0.0L;
    }
    for (int s = 0; s < nsurf; ++s) {
        Step &st = steps[s];
        st.leg[0] = st.leg[1] = 0;
        st.chirp = false;
        st.kappa.assign(nb, 0.0L); st.d1.assign(nb, 0.0); st.d2.assign(nb, 0.0);
        const fresnel_surface &q = surf[s];
        for (int b = 0; b < nb; ++b) {
            const long double lam = lambda[b];
            if (std::isfinite(q.f)) {            // thin lens: ABCD on the pilot beam, residual chirp on the array
                const long double zR = PI_L * w0[b] * w0[b] / lam;
                const long double qr = zc[b] - zw[b], qi = zR;
                const long double den = qr * qr + qi * qi;
                const long double ir = qr / den - 1.0L / (long double)q.f, ii = -qi / den;
                const long double d2 = ir * ir + ii * ii;
                const long double q2r = ir / d2, q2i = -ii / d2;
                const long double zw2 = zc[b] - q2r, zR2 = q2i;
                const long double inv_rref2 = (fabsl(zc[b] - zw2) < rf * zR2) ? 0.0L : 1.0L / (zc[b] - zw2);
                st.kappa[b] = inv_rref[b] - 1.0L / (long double)q.f - inv_rref2;
                if (st.kappa[b] != 0.0L) st.chirp = true;
                zw[b] = zw2;
                w0[b] = sqrtl(lam * zR2 / PI_L);
                inv_rref[b] = inv_rref2;
            }
            int leg[2] = {0, 0};
            if (q.z != 0.0) {
                const long double zR = PI_L * w0[b] * w0[b] / lam;
                const long double z1 = zc[b], z2 = zc[b] + (long double)q.z;
                const int in1 = inv_rref[b] == 0.0L;
                const int in2 = fabsl(z2 - zw[b]) < rf * zR;
                if (in1 && in2) {
                    leg[0] = 1; st.d1[b] = q.z;
                } else {
                    st.d1[b] = (double)(zw[b] - z1); st.d2[b] = (double)(z2 - zw[b]);
                    if (st.d1[b] != 0.0) leg[0] = in1 ? 1 : 3;
                    if (st.d2[b] != 0.0) leg[1] = in2 ? 1 : 2;
                }
                zc[b] = z2;
                inv_rref[b] = in2 ? 0.0L : 1.0L / (z2 - zw[b]);
            }
            if (b == 0) { st.leg[0] = leg[0]; st.leg[1] = leg[1]; }
            else if (leg[0] != st.leg[0] || leg[1] != st.leg[1]) return FRESNEL_ERR_UNSUPPORTED;   // the batch straddles a regime boundary
        }
        // a single-transform leg needs one sign of dz over the batch
        for (int l = 0; l < 2; ++l)
            if (st.leg[l] >= 2) {
                const std::vector<double> &d = l == 0 ? st.d1 : st.d2;
                for (int b = 1; b < nb; ++b)
                    if ((d[b] > 0) != (d[0] > 0)) return FRESNEL_ERR_UNSUPPORTED;
            }
    }

    // ---- enqueue ----
    p->schedule.clear();
    auto finish = [&](fresnel_status st) {
        if (st == FRESNEL_OK) train_event(p, p->schedule.size());
        p->train_ev.clear();
        return st;
    };
    for (int s = 0; s < nsurf; ++s) {
        const Step &st = steps[s];
        const fresnel_surface &q = surf[s];
        const void *amp = q.amp, *opd = q.opd;
        bool optic_pending = st.chirp || amp || opd;
        std::vector<ChirpSpec> ck;
        if (st.chirp) {
            ck.resize(nb);
            for (int b = 0; b < nb; ++b) ck[b] = make_spec(curvature_coeff(pixel_inout[b], lambda[b], st.kappa[b]), 1.0, 0.0);
        }
        fresnel_status rc = FRESNEL_OK;
        for (int l = 0; l < 2 && rc == FRESNEL_OK; ++l) {
            const int leg = st.leg[l];
            if (leg == 0) continue;
            const std::vector<double> &d = l == 0 ? st.d1 : st.d2;
            if (leg == 1) rc = as_leg(p, wf, pixel_inout, lambda, optic_pending ? ck : std::vector<ChirpSpec>(), optic_pending ? amp : nullptr,
                                      optic_pending ? opd : nullptr, d.data(), s);
            else rc = ft_leg(p, wf, pixel_inout, lambda, d.data(), leg == 2 ? FT_WTS : FT_STW, (optic_pending && st.chirp) ? st.kappa.data() : nullptr,
                             optic_pending ? amp : nullptr, optic_pending ? opd : nullptr, s);
            optic_pending = false;
        }
        if (rc == FRESNEL_OK && optic_pending) {         // no propagation leg took the optic along: apply it on its own
            std::vector<double> zero(nb, 0.0);
            rc = as_leg(p, wf, pixel_inout, lambda, ck, amp, opd, zero.data(), s);
        }
        if (rc != FRESNEL_OK) return finish(rc);
        if (legs_used) { legs_used[2 * s] = st.leg[0]; legs_used[2 * s + 1] = st.leg[1]; }
    }
    for (int b = 0; b < nb; ++b) {
        state[b].w0 = (double)w0[b]; state[b].zw = (double)zw[b]; state[b].z = (double)zc[b];
        state[b].rref = inv_rref[b] == 0.0L ? INFINITY : (double)(1.0L / inv_rref[b]);
    }
    return finish(FRESNEL_OK);
}

// ---- Fraunhofer propagation by a matrix Fourier transform ----------------------------------------------------------
} // extern "C"

namespace {

struct MftScalArgs {
    double *dst;                // [4][batch]
    int batch, b0, n;
    double v[4][32];
};
__global__ void mft_scalars_kernel(MftScalArgs a)
{
    const int i = threadIdx.x;
    if (i < a.n)
        for (int r = 0; r < 4; ++r) a.dst[(size_t)r * a.batch + a.b0 + i] = a.v[r][i];
}
__global__ void mft_alpha_kernel(const double *scal, double2 *alpha, int batch)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < batch) alpha[i] = make_double2(scal[(size_t)2 * batch + i], scal[(size_t)3 * batch + i]);
}

fresnel_status mft_reserve(fresnel_plan *p, int nb)
{
    if (nb <= p->mft_nb_cap) return FRESNEL_OK;
    if (capture_state(p).active) return FRESNEL_ERR_ALLOC;                 // allocates: reserve before capturing
    cudaStreamSynchronize(p->stream);
    cudaFree(p->mft_e); cudaFree(p->mft_t);
    p->mft_e = p->mft_t = nullptr;
    p->mft_nb_cap = 0;
    p->mft_key.clear();
    const size_t n = (size_t)p->batch * nb * p->N;
    if (cudaMalloc((void **)&p->mft_e, n * sizeof(double2)) != cudaSuccess || cudaMalloc((void **)&p->mft_t, n * sizeof(double2)) != cudaSuccess) {
        cudaGetLastError();
        cudaFree(p->mft_e); p->mft_e = nullptr;
        return FRESNEL_ERR_ALLOC;
    }
    if (!p->mft_scal && cudaMalloc((void **)&p->mft_scal, (size_t)6 * p->batch * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return FRESNEL_ERR_ALLOC; }
    p->mft_nb_cap = nb;
    return FRESNEL_OK;
}

} // namespace

extern "C" {

fresnel_status fresnel_plan_reserve_mft(fresnel_plan *p, int nb_max)
{
    if (!p || nb_max <= 0 || nb_max > 8192) return FRESNEL_ERR_INVALID_ARG;
    DeviceGuard g(p);
    return mft_reserve(p, nb_max);
}

fresnel_status fresnel_mft(fresnel_plan *p, const void *in, void *out, int nb, const double *pixel_in, const double *pixel_out,
                           const double *lambda, double f, int direction)
{
    if (!p || !in || !out || in == out || nb <= 0 || nb > 8192) return FRESNEL_ERR_INVALID_ARG;
    if (!valid_positive(pixel_in, p->batch) || !valid_positive(pixel_out, p->batch) || !valid_positive(lambda, p->batch)) return FRESNEL_ERR_INVALID_ARG;
    if (!std::isfinite(f) || f == 0.0 || (direction != FRESNEL_FORWARD && direction != FRESNEL_INVERSE)) return FRESNEL_ERR_INVALID_ARG;
    DeviceGuard g(p);
    fresnel_status st = mft_reserve(p, nb);
    if (st != FRESNEL_OK) return st;
    const int nbt = p->batch, na = p->N;
    // per batch element: c = dx dx'/(lambda f) in turns (double-double), alpha = dx^2/(+- i lambda f) = -+ i dx^2/(lambda f)
    std::vector<double> key(2 + 2 * (size_t)nbt), scal(4 * (size_t)nbt);
    key[0] = nb; key[1] = direction;
    for (int b = 0; b < nbt; ++b) {
        const long double c = (long double)pixel_in[b] * (long double)pixel_out[b] / ((long double)lambda[b] * (long double)f);
        const double hi = (double)c, lo = (double)(c - (long double)hi);
        const double gq = (double)((long double)pixel_in[b] * (long double)pixel_in[b] / ((long double)lambda[b] * (long double)f));
        key[2 + b] = hi; key[2 + nbt + b] = lo;
        scal[b] = hi; scal[nbt + b] = lo; scal[2 * (size_t)nbt + b] = 0.0; scal[3 * (size_t)nbt + b] = direction == FRESNEL_FORWARD ? -gq : gq;
    }
    const bool cap = capture_state(p).active;
    double2 *alpha = reinterpret_cast<double2 *>(p->mft_scal + 4 * (size_t)nbt);
    for (int b0 = 0; b0 < nbt; b0 += 32) {                     // the scalars travel as kernel parameters
        MftScalArgs a;
        a.dst = p->mft_scal; a.batch = nbt; a.b0 = b0; a.n = nbt - b0 < 32 ? nbt - b0 : 32;
        for (int r = 0; r < 4; ++r)
            for (int i = 0; i < a.n; ++i) a.v[r][i] = scal[(size_t)r * nbt + b0 + i];
        mft_scalars_kernel<<<1, 32, 0, p->stream>>>(a);
        ++p->launches;
    }
    mft_alpha_kernel<<<(nbt + 127) / 128, 128, 0, p->stream>>>(p->mft_scal, alpha, nbt);
    ++p->launches;
    if (cap || p->mft_key != key) {                            // the kernel matrix of this geometry
        MftMatrixArgs m;
        m.out = p->mft_e; m.na = na; m.nb = nb; m.batch = nbt; m.sign = direction == FRESNEL_FORWARD ? -1 : +1;
        m.c_hi = p->mft_scal; m.c_lo = p->mft_scal + nbt;
        mft_matrix_kernel<<<dim3((na + 255) / 256, nb, nbt), 256, 0, p->stream>>>(m);
        ++p->launches;
        if (cap) p->mft_key.clear(); else p->mft_key = key;
    }
    if (cudaGetLastError() != cudaSuccess) return FRESNEL_ERR_CUDA;
    // T^t[q,j] = sum_k U[j,k] E[q,k]
    MftGemmArgs g1;
    g1.A = in; g1.B = p->mft_e; g1.C = p->mft_t; g1.M = na; g1.N = nb; g1.K = na;
    g1.strideA = (size_t)na * na; g1.strideB = (size_t)nb * na; g1.strideC = (size_t)nb * na; g1.alpha = nullptr;
    cudaError_t e = p->dtype == FRESNEL_C128 ? launch_mft_gemm<double2, double2, true>(g1, nbt, p->stream)
                                             : launch_mft_gemm<float2, double2, true>(g1, nbt, p->stream);
    if (e != cudaSuccess) return FRESNEL_ERR_CUDA;
    ++p->launches;
    // V[p,q] = alpha sum_j E[p,j] T^t[q,j]
    MftGemmArgs g2;
    g2.A = p->mft_e; g2.B = p->mft_t; g2.C = out; g2.M = nb; g2.N = nb; g2.K = na;
    g2.strideA = (size_t)nb * na; g2.strideB = (size_t)nb * na; g2.strideC = (size_t)nb * nb; g2.alpha = alpha;
    e = p->dtype == FRESNEL_C128 ? launch_mft_gemm<double2, double2, false>(g2, nbt, p->stream)
                                 : launch_mft_gemm<double2, float2, false>(g2, nbt, p->stream);
    if (e != cudaSuccess) return FRESNEL_ERR_CUDA;
    ++p->launches;
    return FRESNEL_OK;
}

// ---- broadband image: incoherent sum over the batch ---------------------------------------------------------
fresnel_status fresnel_accumulate_intensity(fresnel_plan *p, const void *wf, const double *weight, void *image)
{
    if (!p || !wf || !weight || !image) return FRESNEL_ERR_INVALID_ARG;
    for (int b = 0; b < p->batch; ++b)
        if (!std::isfinite(weight[b])) return FRESNEL_ERR_INVALID_ARG;
    DeviceGuard g(p);
    cudaError_t e;
    if (p->dtype == FRESNEL_C128)
        e = launch_intensity<double>((const double2 *)wf, (double *)image, weight, p->N, p->batch, p->sms, p->stream, &p->launches);
    else
        e = launch_intensity<float>((const float2 *)wf, (float *)image, weight, p->N, p->batch, p->sms, p->stream, &p->launches);
    return e == cudaSuccess ? FRESNEL_OK : FRESNEL_ERR_CUDA;
}

} // extern "C"

// ---- fresnel_mft_noalloc: the matrix Fourier transform for callers that may not allocate ------------------------------
// fresnel_mft keeps its kernel matrix E and the intermediate T^t of its two GEMMs in plan-owned cudaMalloc memory.  Callers
// that cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops, harnesses that forbid it) get this variant:
// no plan, and the same scratch in ONE file-scope device array of a fixed, modest size that every GPU that loads the
// library holds until exit (8 MiB + 1.5 KiB).  In host code the array's NAME is a host-side stand-in, not a device address, so
// its address is looked up once per device with cudaGetSymbolAddress (that device current) and only that pointer goes to
// the kernels.  All calls share the array and it keeps the last call's contents: every word a call reads (kernel matrix,
// intermediate, per-batch scalars) is written by the same call first, so nothing has to start at zero and nothing is
// cleared; calls that overlap on the GPU (two streams, two host threads) race on it.
namespace {

constexpr size_t kMftStaticElems = FRESNEL_MFT_NOALLOC_MAX_ELEMS;      // complex doubles per region: batch * nb * na at most
constexpr int kMftStaticBatch = FRESNEL_MFT_NOALLOC_MAX_BATCH;         // one mft_scalars_kernel launch carries 32
static_assert(kMftStaticBatch <= 32, "the per-batch scalars travel in one kernel-parameter block of 32");
// [0, E): kernel matrix   [E, 2E): intermediate T^t   then 6 * batch doubles: c_hi, c_lo, alpha.re, alpha.im, alpha (interleaved)
static __device__ __align__(256) double2 fr_mft_static_scratch[2 * kMftStaticElems + 3 * kMftStaticBatch];

// device address of the array on the current device: cudaGetSymbolAddress once per device ordinal (a second thread
// racing here looks the same address up twice)
cudaError_t mft_static_scratch(double2 **out)
{
    static std::atomic<double2 *> addr[64];
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    double2 *p = addr[dev].load(std::memory_order_acquire);
    if (p == nullptr) {
        e = cudaGetSymbolAddress((void **)&p, fr_mft_static_scratch);
        if (e != cudaSuccess) return e;
        if (p == nullptr) return cudaErrorInvalidSymbol;
        addr[dev].store(p, std::memory_order_release);
    }
    *out = p;
    return cudaSuccess;
}

} // namespace

extern "C" {

fresnel_status fresnel_mft_noalloc(const void *in, void *out, int na, int nb, int batch, fresnel_dtype dtype, const double *pixel_in,
                                   const double *pixel_out, const double *lambda, double f, int direction, void *stream)
{
    if (!in || !out || in == out || na <= 0 || nb <= 0 || batch <= 0) return FRESNEL_ERR_INVALID_ARG;
    if (dtype != FRESNEL_C64 && dtype != FRESNEL_C128) return FRESNEL_ERR_UNSUPPORTED;
    if (batch > kMftStaticBatch || (size_t)batch * (size_t)nb * (size_t)na > kMftStaticElems) return FRESNEL_ERR_TOO_LARGE;
    if (!valid_positive(pixel_in, batch) || !valid_positive(pixel_out, batch) || !valid_positive(lambda, batch)) return FRESNEL_ERR_INVALID_ARG;
    if (!std::isfinite(f) || f == 0.0 || (direction != FRESNEL_FORWARD && direction != FRESNEL_INVERSE)) return FRESNEL_ERR_INVALID_ARG;
    double2 *scratch = nullptr;
    if (mft_static_scratch(&scratch) != cudaSuccess) { cudaGetLastError(); return FRESNEL_ERR_CUDA; }
    cudaStream_t s = (cudaStream_t)stream;
    double2 *E = scratch, *T = scratch + kMftStaticElems;
    double *scal = reinterpret_cast<double *>(scratch + 2 * kMftStaticElems);
    double2 *alpha = reinterpret_cast<double2 *>(scal + 4 * (size_t)batch);
    // per batch element, as in fresnel_mft: c = dx dx'/(lambda f) in turns (double-double), alpha = -+ i dx^2/(lambda f)
    MftScalArgs sa;
    sa.dst = scal; sa.batch = batch; sa.b0 = 0; sa.n = batch;
    for (int b = 0; b < batch; ++b) {
        const long double c = (long double)pixel_in[b] * (long double)pixel_out[b] / ((long double)lambda[b] * (long double)f);
        const double hi = (double)c, lo = (double)(c - (long double)hi);
        const double gq = (double)((long double)pixel_in[b] * (long double)pixel_in[b] / ((long double)lambda[b] * (long double)f));
        sa.v[0][b] = hi; sa.v[1][b] = lo; sa.v[2][b] = 0.0; sa.v[3][b] = direction == FRESNEL_FORWARD ? -gq : gq;
    }
    mft_scalars_kernel<<<1, 32, 0, s>>>(sa);
    mft_alpha_kernel<<<(batch + 127) / 128, 128, 0, s>>>(scal, alpha, batch);
    MftMatrixArgs m;                                            // the kernel matrix is rebuilt by every call: the array is shared
    m.out = E; m.na = na; m.nb = nb; m.batch = batch; m.sign = direction == FRESNEL_FORWARD ? -1 : +1;
    m.c_hi = scal; m.c_lo = scal + batch;
    mft_matrix_kernel<<<dim3((na + 255) / 256, nb, batch), 256, 0, s>>>(m);
    if (cudaGetLastError() != cudaSuccess) return FRESNEL_ERR_CUDA;
    MftGemmArgs g1;                                             // T^t[q,j] = sum_k U[j,k] E[q,k]
    g1.A = in; g1.B = E; g1.C = T; g1.M = na; g1.N = nb; g1.K = na;
    g1.strideA = (size_t)na * na; g1.strideB = (size_t)nb * na; g1.strideC = (size_t)nb * na; g1.alpha = nullptr;
    cudaError_t e = dtype == FRESNEL_C128 ? launch_mft_gemm<double2, double2, true>(g1, batch, s)
                                          : launch_mft_gemm<float2, double2, true>(g1, batch, s);
    if (e != cudaSuccess) return FRESNEL_ERR_CUDA;
    MftGemmArgs g2;                                             // V[p,q] = alpha sum_j E[p,j] T^t[q,j]
    g2.A = E; g2.B = T; g2.C = out; g2.M = nb; g2.N = nb; g2.K = na;
    g2.strideA = (size_t)nb * na; g2.strideB = (size_t)nb * na; g2.strideC = (size_t)nb * nb; g2.alpha = alpha;
    e = dtype == FRESNEL_C128 ? launch_mft_gemm<double2, double2, false>(g2, batch, s)
                              : launch_mft_gemm<double2, float2, false>(g2, batch, s);
    return e == cudaSuccess ? FRESNEL_OK : FRESNEL_ERR_CUDA;
}

} // extern "C"
