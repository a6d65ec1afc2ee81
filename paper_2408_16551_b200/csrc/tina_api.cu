// tina_api.cu -- the C ABI of libtina (include/tina.h): argument validation, dispatch
// between the tcgen05 path and the generic CUDA-core path, host-buffer wrappers.
#include "tina_common.cuh"

#include <cstdlib>
#include <cstring>
#include <mutex>

namespace tina {

std::atomic<long long> g_launches{0};
std::atomic<int> g_last_path{kPathNone};
std::atomic<const char*> g_last_kernel{"none"};
std::atomic<double> g_last_issued_ratio{1.0};
static thread_local char t_err[512] = "";

void set_error(const char* fmt, ...)
{
    va_list ap; va_start(ap, fmt);
    vsnprintf(t_err, sizeof(t_err), fmt, ap);
    va_end(ap);
}

tina_status fail(tina_status s, const char* fmt, ...)
{
    va_list ap; va_start(ap, fmt);
    vsnprintf(t_err, sizeof(t_err), fmt, ap);
    va_end(ap);
    return s;
}

tina_status check_cuda(cudaError_t e, const char* what)
{
    if (e == cudaSuccess) return TINA_OK;
    set_error("%s: %s", what, cudaGetErrorString(e));
    return e == cudaErrorMemoryAllocation ? TINA_ERR_OUT_OF_MEMORY : TINA_ERR_CUDA;
}

// ---- options ------------------------------------------------------------------------------------
static std::mutex g_opt_mu;
static Options g_opt;
static std::atomic<bool> g_opt_loaded{false};

static void load_options_locked()
{
    Options o;
    auto on = [](const char* n) { const char* v = getenv(n); return v && *v && strcmp(v, "0") != 0; };
    o.nt256 = on("TINA_NT256");
    o.share = on("TINA_SHARE") && !on("TINA_NO_SHARE");
    o.no_out_tma = on("TINA_NO_OUT_TMA");
    o.fir_simt = on("TINA_FIR_SIMT");
    o.fir_v1 = on("TINA_FIR_V1");
    o.ct_no_ws = on("TINA_CT_NO_WS");
    o.ctr_ws = on("TINA_CTR_WS");
    o.no_sym = on("TINA_NO_SYM");
    o.sym_v1 = on("TINA_SYM_V1");
    o.fold = on("TINA_SYM_FOLD");
#ifdef TINA_DEV
    auto num = [](const char* n) { const char* v = getenv(n); return v ? atoi(v) : 0; };
    o.debug_skip = num("TINA_DEBUG_SKIP");
    o.ksplit = num("TINA_KSPLIT");
    o.a_slots = num("TINA_A_SLOTS");
    o.b_entries = num("TINA_B_ENTRIES");
    o.cl4 = num("TINA_CL4");
    o.prof = on("TINA_PROF");
#endif
    g_opt = o;
    g_opt_loaded.store(true, std::memory_order_release);
}

const Options& options()
{
    if (!g_opt_loaded.load(std::memory_order_acquire)) {
        std::lock_guard<std::mutex> lk(g_opt_mu);
        if (!g_opt_loaded.load(std::memory_order_relaxed)) load_options_locked();
    }
    return g_opt;
}

void reload_options()
{
    std::lock_guard<std::mutex> lk(g_opt_mu);
    load_options_locked();
}

// ---- per-device contexts ------------------------------------------------------------------------
static std::mutex g_ctx_mu;
static std::map<int, DevCtx*> g_ctx;

tina_status dev_ctx(DevCtx** out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return check_cuda(e, "cudaGetDevice");
    std::lock_guard<std::mutex> lk(g_ctx_mu);
    auto it = g_ctx.find(dev);
    if (it == g_ctx.end()) {
        int n_sm = 0;
        e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess || n_sm < 1) return check_cuda(e != cudaSuccess ? e : cudaErrorInvalidDevice, "cudaDeviceGetAttribute(SM count)");
        DevCtx* c = new DevCtx();
        c->dev = dev;
        c->n_sm = n_sm;
        it = g_ctx.emplace(dev, c).first;
    }
    *out = it->second;
    return TINA_OK;
}

tina_status ensure_smem(DevCtx* ctx, const void* func, int bytes, const char* what)
{
    std::lock_guard<std::mutex> lk(ctx->mu);
    auto it = ctx->smem_attr.find(func);
    if (it != ctx->smem_attr.end() && it->second >= bytes) return TINA_OK;
    cudaError_t e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e != cudaSuccess) return check_cuda(e, what);
    ctx->smem_attr[func] = bytes;
    return TINA_OK;
}

bool tmap_cache_get(DevCtx* ctx, const TmapKey& key, TmapSet* out)
{
    std::lock_guard<std::mutex> lk(ctx->mu);
    for (const auto& e : ctx->tmaps)
        if (e.first == key) { *out = e.second; return true; }
    return false;
}

void tmap_cache_put(DevCtx* ctx, const TmapKey& key, const TmapSet& set)
{
    constexpr size_t kMax = 16;
    std::lock_guard<std::mutex> lk(ctx->mu);
    if (ctx->tmaps.size() < kMax) ctx->tmaps.emplace_back(key, set);
    else ctx->tmaps[ctx->tmap_next++ % kMax] = std::make_pair(key, set);
}

void dev_ctx_release_all()
{
    std::lock_guard<std::mutex> lk(g_ctx_mu);
    int cur = 0;
    cudaGetDevice(&cur);
    for (auto& kv : g_ctx) {
        DevCtx* c = kv.second;
        std::lock_guard<std::mutex> l2(c->host_mu);
        std::lock_guard<std::mutex> l3(c->mu);
        cudaSetDevice(c->dev);
        for (int i = 0; i < 3; ++i) { if (c->stage_p[i]) cudaFree(c->stage_p[i]); c->stage_p[i] = nullptr; c->stage_n[i] = 0; }
        if (c->tz_ring) { cudaFree(c->tz_ring); c->tz_ring = nullptr; }
        c->tmaps.clear();
    }
    cudaSetDevice(cur);
}

// Device staging buffers for the *_host entry points (per device, grown on demand, freed by
// tina_clear_plan_cache).
static tina_status stage_reserve(DevCtx* c, int i, size_t bytes)
{
    if (c->stage_n[i] >= bytes) return TINA_OK;
    if (c->stage_p[i]) cudaFree(c->stage_p[i]);
    c->stage_p[i] = nullptr; c->stage_n[i] = 0;
    cudaError_t e = cudaMalloc(&c->stage_p[i], bytes);
    if (e != cudaSuccess) return check_cuda(e, "cudaMalloc(staging)");
    c->stage_n[i] = bytes;
    return TINA_OK;
}

static tina_status pfb_validate(const void* x, int S, long long n_samples, int P, int M,
                                const float* window, tina_kind kind, const void* out,
                                const char* who, long long* F_out)
{
    if (!x || !window) return fail(TINA_ERR_NULL_POINTER, "%s: null pointer", who);
    if (kind != TINA_COMPLEX && kind != TINA_REAL) return fail(TINA_ERR_BAD_SHAPE, "%s: bad kind", who);
    if (S < 1 || P < 2 || M < 1 || n_samples < 1) return fail(TINA_ERR_BAD_SHAPE, "%s: S, M >= 1 and P >= 2 required", who);
    if (kind == TINA_REAL && (P & 1)) return fail(TINA_ERR_BAD_SHAPE, "%s: P must be even for the real kind", who);
    if (P > kMaxP) return fail(TINA_ERR_UNSUPPORTED, "%s: P > %d", who, kMaxP);
    if (M > kMaxTapsPfb) return fail(TINA_ERR_UNSUPPORTED, "%s: M > %d", who, kMaxTapsPfb);
    const long long F = n_samples / P - M + 1;
    if (F < 1) return fail(TINA_ERR_BAD_SHAPE, "%s: n_samples too short (F = %lld)", who, F);
    if (!out) return fail(TINA_ERR_NULL_POINTER, "%s: null output pointer", who);
    if (x == out) return fail(TINA_ERR_BAD_SHAPE, "%s: in-place not supported", who);
    if (!aligned16(x) || !aligned16(out) || !aligned16(window))
        return fail(TINA_ERR_ALIGNMENT, "%s: x, window, out must be 16-byte aligned", who);
    if (S > 1) {
        const long long mod = (kind == TINA_REAL) ? 4 : 2;
        if (n_samples % mod) return fail(TINA_ERR_ALIGNMENT, "%s: n_samples must be a multiple of %lld when S > 1", who, mod);
    }
    *F_out = F;
    return TINA_OK;
}

}  // namespace tina

using namespace tina;

extern "C" {

tina_status tina_fir(const float* x, const float* taps, float* y, int C, long long L, int M, void* stream)
{
    if (!x || !taps || !y) return fail(TINA_ERR_NULL_POINTER, "tina_fir: null pointer");
    if (C < 1 || M < 1 || L < M) return fail(TINA_ERR_BAD_SHAPE, "tina_fir: need C >= 1, M >= 1, L >= M");
    if (M > kMaxTapsFir) return fail(TINA_ERR_UNSUPPORTED, "tina_fir: M > %d", kMaxTapsFir);
    if ((const void*)x == (const void*)y) return fail(TINA_ERR_BAD_SHAPE, "tina_fir: in-place not supported");
    if (!aligned16(x) || !aligned16(y)) return fail(TINA_ERR_ALIGNMENT, "tina_fir: x, y must be 16-byte aligned");
    tina_status fs = TINA_OK;
    if (firt_fir(x, taps, y, C, L, M, false, (cudaStream_t)stream, &fs)) return fs;
    if (umma_fir(x, taps, y, C, L, M, (cudaStream_t)stream, &fs)) return fs;
    return simt_fir(x, taps, y, C, L, M, (cudaStream_t)stream);
}

tina_status tina_fir_multi(const float* x, const float* taps, float* y, int C, long long L, int M, void* stream)
{
    if (!x || !taps || !y) return fail(TINA_ERR_NULL_POINTER, "tina_fir_multi: null pointer");
    if (C < 1 || M < 1 || L < M) return fail(TINA_ERR_BAD_SHAPE, "tina_fir_multi: need C >= 1, M >= 1, L >= M");
    if (M > kMaxTapsFir) return fail(TINA_ERR_UNSUPPORTED, "tina_fir_multi: M > %d", kMaxTapsFir);
    if ((const void*)x == (const void*)y) return fail(TINA_ERR_BAD_SHAPE, "tina_fir_multi: in-place not supported");
    if (!aligned16(x) || !aligned16(y)) return fail(TINA_ERR_ALIGNMENT, "tina_fir_multi: x, y must be 16-byte aligned");
    tina_status fs = TINA_OK;
    if (firt_fir(x, taps, y, C, L, M, true, (cudaStream_t)stream, &fs)) return fs;
    return simt_fir(x, taps, y, C, L, M, (cudaStream_t)stream, true);
}

tina_status tina_dft(const void* x, void* out, long long B, int N, int inverse,
                     tina_precision prec, void* stream)
{
    if (!x || !out) return fail(TINA_ERR_NULL_POINTER, "tina_dft: null pointer");
    if (B < 1 || N < 2) return fail(TINA_ERR_BAD_SHAPE, "tina_dft: need B >= 1, N >= 2");
    if (N > kMaxP) return fail(TINA_ERR_UNSUPPORTED, "tina_dft: N > %d", kMaxP);
    if (prec != TINA_PREC_FP32 && prec != TINA_PREC_BF16 && prec != TINA_PREC_FP16) return fail(TINA_ERR_BAD_SHAPE, "tina_dft: bad precision");
    if (x == out) return fail(TINA_ERR_BAD_SHAPE, "tina_dft: in-place not supported");
    if (!aligned16(x) || !aligned16(out)) return fail(TINA_ERR_ALIGNMENT, "tina_dft: x, out must be 16-byte aligned");
    // A DFT batch is a PFB with M = 1 and unit taps over one stream of B*N samples.
    if (umma_supported(N, false))
        return umma_pfb(x, 1, B * (long long)N, N, 1, nullptr, false, inverse != 0, prec, out, (cudaStream_t)stream);
    return simt_pfb(x, 1, B * (long long)N, N, 1, nullptr, false, inverse != 0, out, (cudaStream_t)stream);
}

tina_status tina_pfb_batched(const void* x, int S, long long n_samples, int P, int M,
                             const float* window, tina_kind kind, tina_precision prec,
                             void* out, void* stream)
{
    long long F;
    tina_status st = pfb_validate(x, S, n_samples, P, M, window, kind, out, "tina_pfb", &F);
    if (st != TINA_OK) return st;
    if (prec != TINA_PREC_FP32 && prec != TINA_PREC_BF16 && prec != TINA_PREC_FP16) return fail(TINA_ERR_BAD_SHAPE, "tina_pfb: bad precision");
    const bool real = kind == TINA_REAL;
    if (umma_supported(P, real))
        return umma_pfb(x, S, n_samples, P, M, window, real, false, prec, out, (cudaStream_t)stream);
    return simt_pfb(x, S, n_samples, P, M, window, real, false, out, (cudaStream_t)stream);
}

tina_status tina_pfb(const void* x, long long n_samples, int P, int M, const float* window,
                     tina_kind kind, tina_precision prec, void* out, void* stream)
{
    return tina_pfb_batched(x, 1, n_samples, P, M, window, kind, prec, out, stream);
}

tina_status tina_pfb_fft_batched(const void* x, int S, long long n_samples, int P, int M, const float* window,
                                 tina_kind kind, void* out, void* stream)
{
    long long F;
    tina_status st = pfb_validate(x, S, n_samples, P, M, window, kind, out, "tina_pfb_fft", &F);
    if (st != TINA_OK) return st;
    if (kind == TINA_COMPLEX && P == 1024 && M <= 16) return ct_pfb(x, S, n_samples, M, window, out, (cudaStream_t)stream);
    if (kind == TINA_REAL && P == 4096 && M <= 8) return ctr_pfb(x, S, n_samples, M, window, out, (cudaStream_t)stream);
    return fail(TINA_ERR_UNSUPPORTED, "tina_pfb_fft: this version covers COMPLEX P = 1024 M <= 16 and REAL P = 4096 M <= 8");
}

tina_status tina_pfb_fir_batched(const void* x, int S, long long n_samples, int P, int M,
                                 const float* window, tina_kind kind, void* y, void* stream)
{
    long long F;
    tina_status st = pfb_validate(x, S, n_samples, P, M, window, kind, y, "tina_pfb_fir", &F);
    if (st != TINA_OK) return st;
    tina_status fs = TINA_OK;
    if (umma_pfb_fir(x, S, n_samples, P, M, window, kind == TINA_REAL, y, (cudaStream_t)stream, &fs)) return fs;
    return simt_pfb_fir(x, S, n_samples, P, M, window, kind == TINA_REAL, y, (cudaStream_t)stream);
}

tina_status tina_pfb_batched_host(const void* x_host, int S, long long n_samples, int P, int M,
                                  const float* window_host, tina_kind kind, tina_precision prec,
                                  void* out_host, void* stream)
{
    if (!x_host || !window_host || !out_host) return fail(TINA_ERR_NULL_POINTER, "tina_pfb_batched_host: null pointer");
    if (S < 1 || P < 2 || M < 1 || n_samples < 1) return fail(TINA_ERR_BAD_SHAPE, "tina_pfb_batched_host: bad shape");
    if (kind != TINA_COMPLEX && kind != TINA_REAL) return fail(TINA_ERR_BAD_SHAPE, "tina_pfb_batched_host: bad kind");
    const long long F = n_samples / P - M + 1;
    if (F < 1) return fail(TINA_ERR_BAD_SHAPE, "tina_pfb_batched_host: n_samples too short");
    const size_t esz = kind == TINA_REAL ? 4 : 8;
    const size_t nk = kind == TINA_REAL ? (size_t)P / 2 + 1 : (size_t)P;
    const size_t row_in = (size_t)P * esz, row_out = nk * 8;
    // Every stream gets its own 16-byte-padded slot in the device staging buffers (the host arrays stay
    // dense): each piece is then a 16-byte-aligned single-stream call whatever S, F and P are.
    const size_t in_slot = ((size_t)n_samples * esz + 15) & ~(size_t)15;
    const size_t out_slot = ((size_t)F * row_out + 15) & ~(size_t)15;
    const size_t wb = (size_t)P * M * 4;
    DevCtx* c = nullptr;
    tina_status st = dev_ctx(&c);
    if (st != TINA_OK) return st;
    std::lock_guard<std::mutex> lk(c->host_mu);
    if ((st = stage_reserve(c, 0, in_slot * S)) != TINA_OK) return st;
    if ((st = stage_reserve(c, 1, wb)) != TINA_OK) return st;
    if ((st = stage_reserve(c, 2, out_slot * S)) != TINA_OK) return st;
    char* const d_in = static_cast<char*>(c->stage_p[0]);
    const float* const d_win = static_cast<const float*>(c->stage_p[1]);
    char* const d_out = static_cast<char*>(c->stage_p[2]);
    cudaStream_t cs = (cudaStream_t)stream;
    cudaError_t e = cudaMemcpyAsync(c->stage_p[1], window_host, wb, cudaMemcpyHostToDevice, cs);
    if (e != cudaSuccess) return check_cuda(e, "H2D copy (window)");

    // Pipeline: the batch is cut into pieces (whole streams, or frame ranges of a stream with their
    // (M-1)-block halo); piece i+1 is copied in and piece i-1 copied out while piece i is computed
    // (PCIe is full duplex), on three internal streams chained by events.
    int pieces_per_stream = 1;
    if (F >= 1024) {
        pieces_per_stream = (int)((16 + S - 1) / S);
        while (pieces_per_stream > 1 && F / pieces_per_stream < 512) --pieces_per_stream;
    }
    long long fpp = (F + pieces_per_stream - 1) / pieces_per_stream;
    fpp = (fpp + 255) / 256 * 256;                                   // piece offsets stay 16-byte aligned for every row size
    constexpr int n_pieces_max = 64;
    if (!c->s_in) {
        e = cudaStreamCreateWithFlags(&c->s_in, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->s_cmp, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->s_out, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_start, cudaEventDisableTiming);
        for (int i = 0; i < n_pieces_max && e == cudaSuccess; ++i) {
            e = cudaEventCreateWithFlags(&c->ev_in[i], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_cmp[i], cudaEventDisableTiming);
        }
        if (e != cudaSuccess) { c->s_in = nullptr; return check_cuda(e, "tina_pfb_batched_host: stream / event setup"); }
    }
    e = cudaEventRecord(c->ev_start, cs);                             // everything follows the caller's stream
    if (e == cudaSuccess) e = cudaStreamWaitEvent(c->s_in, c->ev_start, 0);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(c->s_cmp, c->ev_start, 0);
    if (e != cudaSuccess) return check_cuda(e, "tina_pfb_batched_host: stream ordering");
    int piece = 0;
    for (int sidx = 0; sidx < S; ++sidx) {
        for (long long f_lo = 0; f_lo < F; f_lo += fpp, ++piece) {
            const long long nf = (F - f_lo) < fpp ? (F - f_lo) : fpp;
            const int ei = piece % n_pieces_max;
            const size_t h_in = ((size_t)sidx * n_samples + (size_t)f_lo * P) * esz;    // dense host offsets
            const size_t h_out = ((size_t)sidx * F + f_lo) * row_out;
            const size_t dv_in = (size_t)sidx * in_slot + (size_t)f_lo * row_in;        // padded device offsets
            const size_t dv_out = (size_t)sidx * out_slot + (size_t)f_lo * row_out;
            // last piece of a stream also carries the ignored tail samples (< P of them): not needed
            const size_t in_bytes = (size_t)(nf + M - 1) * row_in, out_bytes = (size_t)nf * row_out;
            e = cudaMemcpyAsync(d_in + dv_in, (const char*)x_host + h_in, in_bytes, cudaMemcpyHostToDevice, c->s_in);
            if (e == cudaSuccess) e = cudaEventRecord(c->ev_in[ei], c->s_in);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(c->s_cmp, c->ev_in[ei], 0);
            if (e != cudaSuccess) return check_cuda(e, "H2D copy");
            st = tina_pfb_batched(d_in + dv_in, 1, (nf + M - 1) * (long long)P, P, M, d_win, kind, prec, d_out + dv_out, c->s_cmp);
            if (st != TINA_OK) { cudaDeviceSynchronize(); return st; }
            e = cudaEventRecord(c->ev_cmp[ei], c->s_cmp);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(c->s_out, c->ev_cmp[ei], 0);
            if (e == cudaSuccess) e = cudaMemcpyAsync((char*)out_host + h_out, d_out + dv_out, out_bytes, cudaMemcpyDeviceToHost, c->s_out);
            if (e != cudaSuccess) return check_cuda(e, "D2H copy");
            if ((piece + 1) % n_pieces_max == 0) {
                // event pool wraps: drain before reusing the events
                e = cudaStreamSynchronize(c->s_out);
                if (e != cudaSuccess) return check_cuda(e, "tina_pfb_batched_host: synchronize");
            }
        }
    }
    e = cudaStreamSynchronize(c->s_out);
    if (e == cudaSuccess) e = cudaStreamSynchronize(cs);
    return check_cuda(e, "D2H copy / synchronize");
}

tina_status tina_unfold(const float* x, float* y, long long I, int J, void* stream)
{
    if (!x || !y) return fail(TINA_ERR_NULL_POINTER, "tina_unfold: null pointer");
    if (J < 1 || I < J) return fail(TINA_ERR_BAD_SHAPE, "tina_unfold: need 1 <= J <= I");
    if ((const void*)x == (const void*)y) return fail(TINA_ERR_BAD_SHAPE, "tina_unfold: in-place not supported");
    return simt_unfold(x, y, I, J, (cudaStream_t)stream);
}

tina_status tina_mul(const float* a, const float* b, float* out, long long n, void* stream)
{
    if (n < 0) return fail(TINA_ERR_BAD_SHAPE, "tina_mul: n < 0");
    if (n > 0 && (!a || !b || !out)) return fail(TINA_ERR_NULL_POINTER, "tina_mul: null pointer");
    return arith_ew(a, b, out, n, true, (cudaStream_t)stream);
}

tina_status tina_add(const float* a, const float* b, float* out, long long n, void* stream)
{
    if (n < 0) return fail(TINA_ERR_BAD_SHAPE, "tina_add: n < 0");
    if (n > 0 && (!a || !b || !out)) return fail(TINA_ERR_NULL_POINTER, "tina_add: null pointer");
    return arith_ew(a, b, out, n, false, (cudaStream_t)stream);
}

tina_status tina_sum(const float* x, long long rows, long long n, float* out, void* stream)
{
    if (rows < 0 || n < 0) return fail(TINA_ERR_BAD_SHAPE, "tina_sum: negative size");
    if (rows > 0 && (!out || (n > 0 && !x))) return fail(TINA_ERR_NULL_POINTER, "tina_sum: null pointer");
    return arith_sum(x, rows, n, out, (cudaStream_t)stream);
}

tina_status tina_matmul(const float* x, const float* y, float* z, long long M, long long L, long long N, void* stream)
{
    if (M < 0 || L < 0 || N < 0) return fail(TINA_ERR_BAD_SHAPE, "tina_matmul: negative size");
    if (M > 0 && N > 0 && (!z || (L > 0 && (!x || !y)))) return fail(TINA_ERR_NULL_POINTER, "tina_matmul: null pointer");
    if ((const void*)z == (const void*)x || (const void*)z == (const void*)y)
        return fail(TINA_ERR_BAD_SHAPE, "tina_matmul: in-place not supported");
    return arith_matmul(x, y, z, M, L, N, (cudaStream_t)stream);
}

long long tina_pfb_num_frames(long long n_samples, int P, int M)
{
    if (P < 1 || M < 1 || n_samples < 0) return 0;
    return n_samples / P - M + 1;
}

const char* tina_status_string(tina_status s)
{
    switch (s) {
        case TINA_OK: return "TINA_OK";
        case TINA_ERR_NULL_POINTER: return "TINA_ERR_NULL_POINTER";
        case TINA_ERR_BAD_SHAPE: return "TINA_ERR_BAD_SHAPE";
        case TINA_ERR_UNSUPPORTED: return "TINA_ERR_UNSUPPORTED";
        case TINA_ERR_ALIGNMENT: return "TINA_ERR_ALIGNMENT";
        case TINA_ERR_CUDA: return "TINA_ERR_CUDA";
        case TINA_ERR_OUT_OF_MEMORY: return "TINA_ERR_OUT_OF_MEMORY";
    }
    return "TINA_ERR_UNKNOWN";
}

const char* tina_last_error(void) { return t_err; }

tina_status tina_clear_plan_cache(void)
{
    umma_clear_plans();
    symf_clear_plans();
    dev_ctx_release_all();
    return TINA_OK;
}

int tina_version(void) { return 200; }  /* 0.2.0 */

tina_status tina_reload_options(void) { reload_options(); return TINA_OK; }

int tina_build_is_dev(void)
{
#ifdef TINA_DEV
    return 1;
#else
    return 0;
#endif
}

tina_status tina_probe_peak(int which, int iters, double* tflops, double* ms, void* stream)
{
    if (!tflops) return fail(TINA_ERR_NULL_POINTER, "tina_probe_peak: null pointer");
    if (which < 0 || which > 5 || iters < 1) return fail(TINA_ERR_BAD_SHAPE, "tina_probe_peak: which in 0..5, iters >= 1");
    return probe_peak(which, iters, tflops, ms, (cudaStream_t)stream);
}

const char* tina_last_kernel(void) { return g_last_kernel.load(); }
double tina_last_issued_ratio(void) { return g_last_issued_ratio.load(); }

long long tina_launch_count(void) { return g_launches.load(); }
int tina_last_path(void) { return g_last_path.load(); }

}  // extern "C"
