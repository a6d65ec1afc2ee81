// tina_api.cu -- the C ABI of libtina (include/tina.h): argument validation, dispatch
// between the tcgen05 path and the generic CUDA-core path, host-buffer wrappers.
#include "tina_common.cuh"

#include <cstring>
#include <mutex>

namespace tina {

std::atomic<long long> g_launches{0};
std::atomic<int> g_last_path{kPathNone};
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

// Device staging buffers for the *_host entry points (grown on demand, freed by
// tina_clear_plan_cache).
struct Staging { void* p = nullptr; size_t n = 0; };
static std::mutex g_stage_mu;
static Staging g_stage[3];

static tina_status stage_reserve(int i, size_t bytes)
{
    Staging& s = g_stage[i];
    if (s.n >= bytes) return TINA_OK;
    if (s.p) cudaFree(s.p);
    s.p = nullptr; s.n = 0;
    cudaError_t e = cudaMalloc(&s.p, bytes);
    if (e != cudaSuccess) return check_cuda(e, "cudaMalloc(staging)");
    s.n = bytes;
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
    if (umma_fir(x, taps, y, C, L, M, (cudaStream_t)stream, &fs)) return fs;
    return simt_fir(x, taps, y, C, L, M, (cudaStream_t)stream);
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
    const size_t xb = (size_t)S * n_samples * esz, wb = (size_t)P * M * 4, ob = (size_t)S * F * nk * 8;
    std::lock_guard<std::mutex> lk(g_stage_mu);
    tina_status st;
    if ((st = stage_reserve(0, xb)) != TINA_OK) return st;
    if ((st = stage_reserve(1, wb)) != TINA_OK) return st;
    if ((st = stage_reserve(2, ob)) != TINA_OK) return st;
    cudaStream_t cs = (cudaStream_t)stream;
    cudaError_t e = cudaMemcpyAsync(g_stage[1].p, window_host, wb, cudaMemcpyHostToDevice, cs);
    if (e != cudaSuccess) return check_cuda(e, "H2D copy (window)");

    // Pipeline: the batch is cut into pieces (whole streams, or frame ranges of a stream with their
    // (M-1)-block halo); piece i+1 is copied in and piece i-1 copied out while piece i is computed
    // (PCIe is full duplex), on three internal streams chained by events.
    const size_t row_in = (size_t)P * esz, row_out = nk * 8;
    int pieces_per_stream = 1;
    if (row_in % 16 == 0 && F >= 1024) {
        pieces_per_stream = (int)((16 + S - 1) / S);
        while (pieces_per_stream > 1 && F / pieces_per_stream < 512) --pieces_per_stream;
    }
    long long fpp = (F + pieces_per_stream - 1) / pieces_per_stream;
    fpp = (fpp + 255) / 256 * 256;                                   // even frame counts keep real-kind rows 16-byte aligned
    const int n_pieces_max = 64;
    static cudaStream_t s_in = nullptr, s_cmp = nullptr, s_out = nullptr;
    static cudaEvent_t ev_start = nullptr, ev_in[n_pieces_max], ev_cmp[n_pieces_max];
    if (!s_in) {
        e = cudaStreamCreateWithFlags(&s_in, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&s_cmp, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&s_out, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ev_start, cudaEventDisableTiming);
        for (int i = 0; i < n_pieces_max && e == cudaSuccess; ++i) {
            e = cudaEventCreateWithFlags(&ev_in[i], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ev_cmp[i], cudaEventDisableTiming);
        }
        if (e != cudaSuccess) { s_in = nullptr; return check_cuda(e, "tina_pfb_batched_host: stream / event setup"); }
    }
    e = cudaEventRecord(ev_start, cs);                                // everything follows the caller's stream
    if (e == cudaSuccess) e = cudaStreamWaitEvent(s_in, ev_start, 0);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(s_cmp, ev_start, 0);
    if (e != cudaSuccess) return check_cuda(e, "tina_pfb_batched_host: stream ordering");
    int piece = 0;
    for (int sidx = 0; sidx < S; ++sidx) {
        for (long long f_lo = 0; f_lo < F; f_lo += fpp, ++piece) {
            const long long nf = (F - f_lo) < fpp ? (F - f_lo) : fpp;
            const int ei = piece % n_pieces_max;
            const size_t in_off = ((size_t)sidx * n_samples + (size_t)f_lo * P) * esz;
            // last piece of a stream also carries the ignored tail samples (< P of them): not needed
            const size_t in_bytes = (size_t)(nf + M - 1) * row_in;
            const size_t out_off = ((size_t)sidx * F + f_lo) * row_out, out_bytes = (size_t)nf * row_out;
            e = cudaMemcpyAsync((char*)g_stage[0].p + in_off, (const char*)x_host + in_off, in_bytes, cudaMemcpyHostToDevice, s_in);
            if (e == cudaSuccess) e = cudaEventRecord(ev_in[ei], s_in);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(s_cmp, ev_in[ei], 0);
            if (e != cudaSuccess) return check_cuda(e, "H2D copy");
            st = tina_pfb_batched((char*)g_stage[0].p + in_off, 1, (nf + M - 1) * (long long)P, P, M, (const float*)g_stage[1].p,
                                  kind, prec, (char*)g_stage[2].p + out_off, s_cmp);
            if (st != TINA_OK) { cudaDeviceSynchronize(); return st; }
            e = cudaEventRecord(ev_cmp[ei], s_cmp);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(s_out, ev_cmp[ei], 0);
            if (e == cudaSuccess) e = cudaMemcpyAsync((char*)out_host + out_off, (char*)g_stage[2].p + out_off, out_bytes, cudaMemcpyDeviceToHost, s_out);
            if (e != cudaSuccess) return check_cuda(e, "D2H copy");
            if (piece + 1 >= n_pieces_max && (piece + 1) % n_pieces_max == 0) {
                // event pool wraps: drain before reusing the events
                e = cudaStreamSynchronize(s_out);
                if (e != cudaSuccess) return check_cuda(e, "tina_pfb_batched_host: synchronize");
            }
        }
    }
    e = cudaStreamSynchronize(s_out);
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
    std::lock_guard<std::mutex> lk(g_stage_mu);
    for (auto& s : g_stage) { if (s.p) cudaFree(s.p); s.p = nullptr; s.n = 0; }
    return TINA_OK;
}

int tina_version(void) { return 100; }  /* 0.1.0 */

long long tina_launch_count(void) { return g_launches.load(); }
int tina_last_path(void) { return g_last_path.load(); }

}  // extern "C"
