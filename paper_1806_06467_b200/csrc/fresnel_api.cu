// fresnel_api.cu -- the C ABI of include/fresnel.h: argument checks, chirp-table cache, launches.
// Every step of the hot path runs in the kernels of pass_kernel.cuh / pointwise.cuh / tables.cuh;
// this file only decides which tables a call needs and enqueues the passes.
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
#include "pointwise.cuh"
#include "tables.cuh"

using namespace fresnel;

namespace {

constexpr int kSlots = 64;              // cached chirp tables per plan (a 20-surface train needs 40)
const long double PI_L = 3.14159265358979323846264338327950288419716939937510L;

struct TableSlot {
    void *dev = nullptr;
    bool valid = false;
    uint64_t stamp = 0;
    uint64_t pinned_call = 0;           // API call that last asked for it (never evicted within that call)
    int index_mode = 0, alt_sign = 0;
    std::vector<ChirpSpec> key;
};

struct TableRequest {
    int slot;
    bool build;
};

} // namespace

struct fresnel_plan {
    int N = 0, batch = 0;
    fresnel_dtype dtype = FRESNEL_C128;
    cudaStream_t stream = nullptr;
    void *tw = nullptr;                 // FFT twiddles
    double *scal_dev = nullptr;         // [batch] 1/lambda
    std::vector<double> scal_key;
    bool scal_valid = false;
    TableSlot slots[kSlots];
    uint64_t clock = 0, call_id = 0;
    unsigned long long launches = 0;
    int prefetch = 0;                   // L2 prefetch distance in tiles (see pass_kernel.cuh)
    int tma_w = 0;                      // columns per TMA tile of the column pass (0: not used for this N)
    int sms = 148;
    int pdl = 1;                        // programmatic dependent launch of the pass kernels (FRESNEL_PDL=0: off, A/B timing)
    CUtensorMap tmap{};                  // tensor map of the wavefront last seen by the column pass
    const void *tmap_wf = nullptr;
    cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};   // profiling hook, see fresnel_plan_record_pass_events
    bool ev_armed = false;
    size_t esize() const { return dtype == FRESNEL_C128 ? sizeof(double2) : sizeof(float2); }
};

namespace {

bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

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

bool capturing(fresnel_plan *p)
{
    cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(p->stream, &st) != cudaSuccess) { cudaGetLastError(); return false; }
    return st != cudaStreamCaptureStatusNone;
}

// Find or allocate a cache slot for a table.  While the stream is being captured into a CUDA graph
// the table is always rebuilt inside the graph, so that replays are self-contained.
TableRequest request_table(fresnel_plan *p, int index_mode, int alt_sign, const std::vector<ChirpSpec> &key, bool force)
{
    ++p->clock;
    for (int i = 0; i < kSlots; ++i) {
        TableSlot &s = p->slots[i];
        if (s.valid && s.index_mode == index_mode && s.alt_sign == alt_sign && s.key.size() == key.size() &&
            std::memcmp(s.key.data(), key.data(), key.size() * sizeof(ChirpSpec)) == 0) {
            s.stamp = p->clock;
            s.pinned_call = p->call_id;
            return {i, force};
        }
    }
    // miss: take a free slot, else the least recently used one that this call has not asked for
    int victim = -1;
    for (int i = 0; i < kSlots && victim < 0; ++i)
        if (!p->slots[i].valid) victim = i;
    if (victim < 0)
        for (int i = 0; i < kSlots; ++i) {
            if (p->slots[i].pinned_call == p->call_id) continue;
            if (victim < 0 || p->slots[i].stamp < p->slots[victim].stamp) victim = i;
        }
    TableSlot &s = p->slots[victim];
    s.valid = true;
    s.index_mode = index_mode;
    s.alt_sign = alt_sign;
    s.key = key;
    s.stamp = p->clock;
    s.pinned_call = p->call_id;
    return {victim, true};
}

// Launch the builder for every requested table that is not cached (and the per-batch scalars).
fresnel_status flush_builds(fresnel_plan *p, const TableRequest *req, int nreq, const double *scal /*or null*/)
{
    int build_idx[kBuildMaxTables];
    int nb_tab = 0;
    for (int i = 0; i < nreq; ++i)
        if (req[i].build) build_idx[nb_tab++] = req[i].slot;
    if (nb_tab == 0 && scal == nullptr) return FRESNEL_OK;
    for (int b0 = 0; b0 < p->batch; b0 += kBuildMaxBatch) {
        BuildArgs a;
        std::memset(&a, 0, sizeof(a));
        a.N = p->N;
        a.b0 = b0;
        a.nb = (p->batch - b0 < kBuildMaxBatch) ? p->batch - b0 : kBuildMaxBatch;
        a.ntab = nb_tab;
        a.is_double = p->dtype == FRESNEL_C128;
        a.scal_out = scal ? p->scal_dev : nullptr;
        for (int b = 0; b < a.nb; ++b) {
            if (scal) a.scal[b] = scal[b0 + b];
            for (int t = 0; t < nb_tab; ++t) a.t[t].spec[b] = p->slots[build_idx[t]].key[b0 + b];
        }
        for (int t = 0; t < nb_tab; ++t) {
            a.t[t].out = p->slots[build_idx[t]].dev;
            a.t[t].index_mode = p->slots[build_idx[t]].index_mode;
            a.t[t].alt_sign = p->slots[build_idx[t]].alt_sign;
        }
        dim3 grid((p->N + 127) / 128, a.nb, nb_tab > 0 ? nb_tab : 1);
        build_tables_kernel<<<grid, 128, 0, p->stream>>>(a);
        if (cudaGetLastError() != cudaSuccess) return FRESNEL_ERR_CUDA;
        ++p->launches;
    }
    return FRESNEL_OK;
}

// 1/lambda per batch element on the device (needed by the optic phasor); cached by value.
const double *need_inv_lambda(fresnel_plan *p, const double *lambda, std::vector<double> &tmp, bool force)
{
    tmp.resize(p->batch);
    for (int b = 0; b < p->batch; ++b) tmp[b] = (double)(1.0L / (long double)lambda[b]);
    if (!force && p->scal_valid && p->scal_key == tmp) return nullptr;      // already resident
    p->scal_key = tmp;
    p->scal_valid = true;
    return tmp.data();
}

bool valid_positive(const double *v, int n)
{
    if (!v) return false;
    for (int i = 0; i < n; ++i)
        if (!(v[i] > 0.0) || !std::isfinite(v[i])) return false;
    return true;
}

// ---- TMA tensor map of a wavefront for the column pass ------------------------------------------------
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

int query_tma_width(int N, fresnel_dtype dt)
{
    switch (N) {
#define FR_CASE(NN) case NN: return dt == FRESNEL_C128 ? col_tma_width_f64_##NN() : col_tma_width_f32_##NN();
        FR_CASE(64) FR_CASE(128) FR_CASE(256) FR_CASE(512) FR_CASE(1024) FR_CASE(2048) FR_CASE(4096) FR_CASE(8192)
#undef FR_CASE
    }
    return 0;
}

// The wavefront as a 3-D tensor {2N scalars, N rows, batch}; a box is {2W scalars, 256 rows, 1}.
bool make_tensor_map(fresnel_plan *p, void *wf)
{
    if (p->tmap_wf == wf) return true;
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return false;
    const bool dbl = p->dtype == FRESNEL_C128;
    const size_t es = p->esize();
    const cuuint64_t N = (cuuint64_t)p->N;
    cuuint64_t gdim[3] = {2 * N, N, (cuuint64_t)p->batch};
    cuuint64_t gstr[2] = {N * es, N * N * es};
    cuuint32_t box[3] = {(cuuint32_t)(2 * p->tma_w), 256u, 1u};
    cuuint32_t estr[3] = {1, 1, 1};
    const size_t row_bytes = (size_t)p->tma_w * es;
    CUtensorMapSwizzle sw = row_bytes == 32 ? CU_TENSOR_MAP_SWIZZLE_32B
                          : row_bytes == 64 ? CU_TENSOR_MAP_SWIZZLE_64B
                          : row_bytes == 128 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE;
    CUresult r = fn(&p->tmap, dbl ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, wf, gdim, gstr, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, sw, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return false;
    p->tmap_wf = wf;
    return true;
}

// ---- pass launch by (dtype, N) ---------------------------------------------------------------------
fresnel_status run_pass(fresnel_plan *p, bool col, int mode, void *wf, const void *pre, const void *rowfac, const void *mid,
                        const void *amp, const void *opd, double scale)
{
    cudaError_t e = cudaErrorInvalidValue;
    const bool tma = col && p->tma_w > 0 && make_tensor_map(p, wf);
    // L2 prefetch of upcoming rows pays when the data does not already sit in the 126 MB L2 (measured:
    // +10..17 % at N >= 4096, -4 % at N = 2048 without maps); TMA tile prefetch of 16..32-byte-wide
    // column boxes costs more TMA issue slots than it saves and stays off.
    const size_t wf_bytes = (size_t)p->batch * p->N * p->N * p->esize();
    const int prefetch = (!col && (wf_bytes > ((size_t)64 << 20) || amp || opd)) ? p->prefetch : 0;
    if (p->dtype == FRESNEL_C128) {
        PassArgs<double> a;
        a.wf = (double2 *)wf; a.pre = (const double2 *)pre; a.mid = (const double2 *)mid; a.rowfac = (const double2 *)rowfac;
        a.tw = (const double2 *)p->tw; a.amp = (const double *)amp; a.opd = (const double *)opd;
        a.inv_lambda = p->scal_dev; a.scale = scale; a.prefetch_distance = prefetch; a.pdl = p->pdl;
        switch (p->N) {
#define FR_CASE(NN) case NN: e = tma ? launch_col_tma_f64_##NN(mode, a, p->tmap, p->batch, p->stream)           \
                                   : launch_pass_f64_##NN(col, mode, a, p->batch, p->stream); break;
            FR_CASE(64) FR_CASE(128) FR_CASE(256) FR_CASE(512) FR_CASE(1024) FR_CASE(2048) FR_CASE(4096) FR_CASE(8192)
#undef FR_CASE
        }
    } else {
        PassArgs<float> a;
        a.wf = (float2 *)wf; a.pre = (const float2 *)pre; a.mid = (const float2 *)mid; a.rowfac = (const float2 *)rowfac;
        a.tw = (const float2 *)p->tw; a.amp = (const float *)amp; a.opd = (const float *)opd;
        a.inv_lambda = p->scal_dev; a.scale = (float)scale; a.prefetch_distance = prefetch; a.pdl = p->pdl;
        switch (p->N) {
#define FR_CASE(NN) case NN: e = tma ? launch_col_tma_f32_##NN(mode, a, p->tmap, p->batch, p->stream)           \
                                   : launch_pass_f32_##NN(col, mode, a, p->batch, p->stream); break;
            FR_CASE(64) FR_CASE(128) FR_CASE(256) FR_CASE(512) FR_CASE(1024) FR_CASE(2048) FR_CASE(4096) FR_CASE(8192)
#undef FR_CASE
        }
    }
    if (e != cudaSuccess) return FRESNEL_ERR_CUDA;
    ++p->launches;
    return FRESNEL_OK;
}

// The two HBM round trips of a propagation / transform: row pass then column pass.
fresnel_status run_two_passes(fresnel_plan *p, int mode, void *wf, const void *pre, const void *mid,
                              const void *amp, const void *opd, double scale)
{
    const bool ev = p->ev_armed;
    p->ev_armed = false;
    if (ev && cudaEventRecord(p->ev[0], p->stream) != cudaSuccess) return FRESNEL_ERR_CUDA;
    // the input chirp is separable: its x-part rides on the load of the row pass, its y-part (one factor per
    // row) on the store of the row pass, so the column pass has no input table at all
    fresnel_status st = run_pass(p, false, mode, wf, pre, pre, mid, amp, opd, scale);
    if (st != FRESNEL_OK) return st;
    if (ev && cudaEventRecord(p->ev[1], p->stream) != cudaSuccess) return FRESNEL_ERR_CUDA;
    st = run_pass(p, true, mode, wf, nullptr, nullptr, mid, nullptr, nullptr, scale);
    if (st != FRESNEL_OK) return st;
    if (ev && cudaEventRecord(p->ev[2], p->stream) != cudaSuccess) return FRESNEL_ERR_CUDA;
    return FRESNEL_OK;
}

fresnel_status run_pointwise(fresnel_plan *p, void *wf, const void *tab, const void *amp, const void *opd)
{
    cudaError_t e;
    if (p->dtype == FRESNEL_C128)
        e = launch_pointwise<double>((double2 *)wf, (const double2 *)tab, (const double *)amp, (const double *)opd,
                                     p->scal_dev, p->N, p->batch, p->stream);
    else
        e = launch_pointwise<float>((float2 *)wf, (const float2 *)tab, (const float *)amp, (const float *)opd,
                                    p->scal_dev, p->N, p->batch, p->stream);
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
    }
    return "FRESNEL_ERR_UNKNOWN";
}

const char *fresnel_version(void) { return "fresnel-b200 0.1 sm_100a"; }

fresnel_status fresnel_plan_create(fresnel_plan **out, int N, int batch, fresnel_dtype dtype)
{
    if (!out || batch <= 0 || N <= 0) return FRESNEL_ERR_INVALID_ARG;
    if (dtype != FRESNEL_C64 && dtype != FRESNEL_C128) return FRESNEL_ERR_UNSUPPORTED;
    if (!is_pow2(N) || N < 64 || N > 8192) return FRESNEL_ERR_UNSUPPORTED;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0) { cudaGetLastError(); return FRESNEL_ERR_CUDA; }
    fresnel_plan *p = new (std::nothrow) fresnel_plan();
    if (!p) return FRESNEL_ERR_ALLOC;
    p->N = N; p->batch = batch; p->dtype = dtype;
    {
        int sms = 148;
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        p->sms = sms;
        const char *pf = std::getenv("FRESNEL_PREFETCH");          // tuning only: tiles ahead, 0 = off
        p->prefetch = pf ? std::atoi(pf) : -sms;                   // negative: auto = SMs x resident CTAs per SM
    }
    { const char *pd = std::getenv("FRESNEL_PDL"); p->pdl = pd ? std::atoi(pd) : 1; }
    p->tma_w = std::getenv("FRESNEL_NO_TMA") ? 0 : query_tma_width(N, dtype);     // env switch: A/B timing only
    fresnel_status st = upload_twiddles(p);
    if (st == FRESNEL_OK && cudaMalloc((void **)&p->scal_dev, sizeof(double) * batch) != cudaSuccess) st = FRESNEL_ERR_ALLOC;
    for (int i = 0; i < kSlots && st == FRESNEL_OK; ++i)
        if (cudaMalloc(&p->slots[i].dev, (size_t)batch * N * p->esize()) != cudaSuccess) st = FRESNEL_ERR_ALLOC;
    if (st != FRESNEL_OK) { cudaGetLastError(); fresnel_plan_destroy(p); return st; }
    *out = p;
    return FRESNEL_OK;
}

fresnel_status fresnel_plan_set_stream(fresnel_plan *p, void *cuda_stream)
{
    if (!p) return FRESNEL_ERR_INVALID_ARG;
    p->stream = (cudaStream_t)cuda_stream;
    return FRESNEL_OK;
}

fresnel_status fresnel_plan_synchronize(fresnel_plan *p)
{
    if (!p) return FRESNEL_ERR_INVALID_ARG;
    return cudaStreamSynchronize(p->stream) == cudaSuccess ? FRESNEL_OK : FRESNEL_ERR_CUDA;
}

fresnel_status fresnel_plan_destroy(fresnel_plan *p)
{
    if (!p) return FRESNEL_OK;
    cudaStreamSynchronize(p->stream);
    cudaFree(p->tw);
    cudaFree(p->scal_dev);
    for (int i = 0; i < kSlots; ++i) cudaFree(p->slots[i].dev);
    cudaGetLastError();
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

fresnel_status fresnel_memcpy_h2d(fresnel_plan *p, void *dst_device, const void *src_host, size_t bytes)
{
    if (!p || !dst_device || !src_host) return FRESNEL_ERR_INVALID_ARG;
    return cudaMemcpyAsync(dst_device, src_host, bytes, cudaMemcpyHostToDevice, p->stream) == cudaSuccess ? FRESNEL_OK : FRESNEL_ERR_CUDA;
}

fresnel_status fresnel_memcpy_d2h(fresnel_plan *p, void *dst_host, const void *src_device, size_t bytes)
{
    if (!p || !dst_host || !src_device) return FRESNEL_ERR_INVALID_ARG;
    return cudaMemcpyAsync(dst_host, src_device, bytes, cudaMemcpyDeviceToHost, p->stream) == cudaSuccess ? FRESNEL_OK : FRESNEL_ERR_CUDA;
}

// ---- Eq. 2: quadratic phase factor ------------------------------------------------------------------
fresnel_status fresnel_apply_qpf(fresnel_plan *p, void *wf, const double *pixel, const double *lambda, double z)
{
    if (!p || !wf || !valid_positive(pixel, p ? p->batch : 0) || !valid_positive(lambda, p->batch)) return FRESNEL_ERR_INVALID_ARG;
    if (!std::isfinite(z) || z == 0.0) return FRESNEL_ERR_INVALID_ARG;
    ++p->call_id;
    const bool force = capturing(p);
    std::vector<ChirpSpec> key(p->batch);
    for (int b = 0; b < p->batch; ++b) key[b] = make_spec(qpf_coeff(pixel[b], lambda[b], z), 1.0, 0.0);
    TableRequest r = request_table(p, 0, 0, key, force);
    fresnel_status st = flush_builds(p, &r, 1, nullptr);
    if (st != FRESNEL_OK) return st;
    return run_pointwise(p, wf, p->slots[r.slot].dev, nullptr, nullptr);
}

// ---- Eq. 3: optic phasor ------------------------------------------------------------------------------
fresnel_status fresnel_apply_mask(fresnel_plan *p, void *wf, const void *amp, const void *opd, const double *lambda)
{
    if (!p || !wf || !valid_positive(lambda, p ? p->batch : 0)) return FRESNEL_ERR_INVALID_ARG;
    if (!amp && !opd) return FRESNEL_OK;
    ++p->call_id;
    std::vector<double> tmp;
    const double *scal = opd ? need_inv_lambda(p, lambda, tmp, capturing(p)) : nullptr;
    fresnel_status st = flush_builds(p, nullptr, 0, scal);
    if (st != FRESNEL_OK) return st;
    return run_pointwise(p, wf, nullptr, amp, opd);
}

// ---- 2-D FFT ---------------------------------------------------------------------------------------------
fresnel_status fresnel_fft2d(fresnel_plan *p, void *wf, int direction, int centered)
{
    if (!p || !wf || (direction != FRESNEL_FORWARD && direction != FRESNEL_INVERSE)) return FRESNEL_ERR_INVALID_ARG;
    ++p->call_id;
    const int mode = direction == FRESNEL_FORWARD ? MODE_FWD : MODE_INV;
    const double per_pass = direction == FRESNEL_FORWARD ? 1.0 : 1.0 / (double)p->N;
    if (!centered) {
        return run_two_passes(p, mode, wf, nullptr, nullptr, nullptr, nullptr, per_pass);
    }
    // centred transform = s * fft2(s * u), s = (-1)^(j+k): sign tables on load and after the transform
    const bool force = capturing(p);
    std::vector<ChirpSpec> k1(p->batch, make_spec(0.0L, 1.0, 0.0)), k2(p->batch, make_spec(0.0L, per_pass, 0.0));
    TableRequest r[2] = {request_table(p, 0, 1, k1, force), request_table(p, 0, 1, k2, force)};
    if (r[0].slot == r[1].slot) r[1].build = false;
    fresnel_status st = flush_builds(p, r, 2, nullptr);
    if (st != FRESNEL_OK) return st;
    return run_two_passes(p, mode, wf, p->slots[r[0].slot].dev, p->slots[r[1].slot].dev, nullptr, nullptr, 1.0);
}

// ---- fused surface: lens + optic phasor + angular-spectrum propagation ----------------------------
fresnel_status fresnel_surface_as(fresnel_plan *p, void *wf, const double *pixel, const double *lambda,
                                  double f, const void *amp, const void *opd, double z)
{
    if (!p || !wf || !valid_positive(pixel, p ? p->batch : 0) || !valid_positive(lambda, p->batch)) return FRESNEL_ERR_INVALID_ARG;
    if (!std::isfinite(z) || std::isnan(f) || f == 0.0) return FRESNEL_ERR_INVALID_ARG;
    ++p->call_id;
    const bool force = capturing(p);
    const bool lens = std::isfinite(f);
    const bool prop = z != 0.0;
    if (!lens && !prop && !amp && !opd) return FRESNEL_OK;

    TableRequest r[2];
    int nreq = 0, i_lens = -1, i_h = -1;
    std::vector<ChirpSpec> key(p->batch);
    if (lens) {
        for (int b = 0; b < p->batch; ++b) key[b] = make_spec(qpf_coeff(pixel[b], lambda[b], -(long double)f), 1.0, 0.0);
        i_lens = nreq;
        r[nreq++] = request_table(p, 0, 0, key, force);
    }
    if (prop) {
        for (int b = 0; b < p->batch; ++b) key[b] = make_spec(as_coeff(p->N, pixel[b], lambda[b], z), 1.0 / (double)p->N, 0.0);
        i_h = nreq;
        r[nreq++] = request_table(p, 1, 0, key, force);
    }
    std::vector<double> tmp;
    const double *scal = opd ? need_inv_lambda(p, lambda, tmp, force) : nullptr;
    fresnel_status st = flush_builds(p, r, nreq, scal);
    if (st != FRESNEL_OK) return st;
    const void *tl = lens ? p->slots[r[i_lens].slot].dev : nullptr;
    if (!prop) return run_pointwise(p, wf, tl, amp, opd);          // optic only
    const void *th = p->slots[r[i_h].slot].dev;
    // row pass: optic phasor and x-chirp of the lens on load, FFT, x H1, inverse FFT, y-chirp of the lens (one
    // factor per row) on store;  column pass: FFT, x H1, inverse FFT
    return run_two_passes(p, MODE_CONV, wf, tl, th, amp, opd, 1.0);
}

fresnel_status fresnel_propagate_as(fresnel_plan *p, void *wf, const double *pixel, const double *lambda, double z)
{
    return fresnel_surface_as(p, wf, pixel, lambda, INFINITY, nullptr, nullptr, z);
}

// ---- direct (single-FFT) Fresnel ---------------------------------------------------------------------
} // extern "C"

namespace {

// [thin lens f] -> [optic phasor] -> direct Fresnel propagation by z, in the two passes of the transform:
// the lens chirp and the input chirp of the propagator are the same kind of factor, so their
// coefficients are added (long double) and ONE table serves both; the optic phasor rides on the row-pass load.
fresnel_status direct_impl(fresnel_plan *p, void *wf, double *pixel_inout, const double *lambda, double z,
                           double f, const void *amp, const void *opd)
{
    ++p->call_id;
    const bool force = capturing(p);
    const bool lens = std::isfinite(f);
    std::vector<ChirpSpec> kin(p->batch), kout(p->batch);
    std::vector<double> dx_out(p->batch);
    for (int b = 0; b < p->batch; ++b) {
        const double dx = pixel_inout[b];
        const long double dxo = (long double)lambda[b] * fabsl((long double)z) / ((long double)p->N * (long double)dx);
        dx_out[b] = (double)dxo;
        long double cin = qpf_coeff(dx, lambda[b], z);
        if (lens) cin += qpf_coeff(dx, lambda[b], -(long double)f);
        kin[b] = make_spec(cin, 1.0, 0.0);
        // per-axis share of dx^2/(i lambda z): dx/sqrt(lambda |z|) * exp(-+ i pi/4)
        const double a1 = (double)((long double)dx / sqrtl((long double)lambda[b] * fabsl((long double)z)));
        kout[b] = make_spec(qpf_coeff(dx_out[b], lambda[b], z), a1, z > 0 ? -0.125 : 0.125);
    }
    // the (-1)^n of the centred transform rides on both tables
    TableRequest r[2] = {request_table(p, 0, 1, kin, force), request_table(p, 0, 1, kout, force)};
    std::vector<double> tmp;
    const double *scal = opd ? need_inv_lambda(p, lambda, tmp, force) : nullptr;
    fresnel_status st = flush_builds(p, r, 2, scal);
    if (st != FRESNEL_OK) return st;
    const int mode = z > 0 ? MODE_FWD : MODE_INV;
    st = run_two_passes(p, mode, wf, p->slots[r[0].slot].dev, p->slots[r[1].slot].dev, amp, opd, 1.0);
    if (st != FRESNEL_OK) return st;
    for (int b = 0; b < p->batch; ++b) pixel_inout[b] = dx_out[b];
    return FRESNEL_OK;
}

} // namespace

extern "C" {

fresnel_status fresnel_propagate_direct(fresnel_plan *p, void *wf, double *pixel_inout, const double *lambda, double z)
{
    if (!p || !wf || !valid_positive(pixel_inout, p ? p->batch : 0) || !valid_positive(lambda, p->batch)) return FRESNEL_ERR_INVALID_ARG;
    if (!std::isfinite(z) || z == 0.0) return FRESNEL_ERR_INVALID_ARG;
    return direct_impl(p, wf, pixel_inout, lambda, z, INFINITY, nullptr, nullptr);
}

// ---- train of surfaces ---------------------------------------------------------------------------------
fresnel_status fresnel_system_run(fresnel_plan *p, void *wf, double *pixel_inout, const double *lambda,
                                  const fresnel_surface *surf, int nsurf, int *method_used)
{
    if (!p || !wf || nsurf < 0 || (nsurf > 0 && !surf)) return FRESNEL_ERR_INVALID_ARG;
    if (!valid_positive(pixel_inout, p->batch) || !valid_positive(lambda, p->batch)) return FRESNEL_ERR_INVALID_ARG;
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
    for (int s = 0; s < nsurf; ++s) {
        const fresnel_surface &q = surf[s];
        fresnel_status st;
        if (method[s] == FRESNEL_METHOD_DIRECT) st = direct_impl(p, wf, pixel_inout, lambda, q.z, q.f, q.amp, q.opd);
        else st = fresnel_surface_as(p, wf, pixel_inout, lambda, q.f, q.amp, q.opd, q.z);   // z == 0: optic only
        if (st != FRESNEL_OK) return st;
        if (method_used) method_used[s] = method[s];
    }
    return FRESNEL_OK;
}

// ---- broadband image: incoherent sum over the batch ---------------------------------------------------------
fresnel_status fresnel_accumulate_intensity(fresnel_plan *p, const void *wf, const double *weight, void *image)
{
    if (!p || !wf || !weight || !image) return FRESNEL_ERR_INVALID_ARG;
    for (int b = 0; b < p->batch; ++b)
        if (!std::isfinite(weight[b])) return FRESNEL_ERR_INVALID_ARG;
    cudaError_t e;
    if (p->dtype == FRESNEL_C128)
        e = launch_intensity<double>((const double2 *)wf, (double *)image, weight, p->N, p->batch, p->sms, p->stream, &p->launches);
    else
        e = launch_intensity<float>((const float2 *)wf, (float *)image, weight, p->N, p->batch, p->sms, p->stream, &p->launches);
    return e == cudaSuccess ? FRESNEL_OK : FRESNEL_ERR_CUDA;
}

} // extern "C"
