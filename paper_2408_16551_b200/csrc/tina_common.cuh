// tina_common.cuh -- shared host-side helpers of libtina (status text, launch counter).
#pragma once
#include <cuda_runtime.h>
#include <atomic>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <vector>

#include "../../include/tina.h"

namespace tina {

constexpr int kMaxP = 8192;      // upper bound on P / N (DFT size)
constexpr int kMaxTapsPfb = 64;  // upper bound on M for the PFB
constexpr int kMaxTapsFir = 4096;

enum Path { kPathNone = 0, kPathSimt = 1, kPathUmma = 2 };

extern std::atomic<long long> g_launches;
extern std::atomic<int> g_last_path;
extern std::atomic<const char*> g_last_kernel;        // name of the kernel variant the last device call launched
extern std::atomic<double> g_last_issued_ratio;       // tensor flops issued per pass / useful flops of that call

void set_error(const char* fmt, ...);
tina_status fail(tina_status s, const char* fmt, ...);
tina_status check_cuda(cudaError_t e, const char* what);

// ---- run-time options (environment, read ONCE; tina_reload_options() re-reads them) --------------
// Every option selects between variants that compute the SAME result within the same contract.
// The knobs that change the amount of work or the accuracy contract (TINA_DEBUG_SKIP, TINA_KSPLIT,
// ring depths, TINA_CL4, TINA_PROF) exist only in builds compiled with -DTINA_DEV.
struct Options {
    bool nt256 = false;        // TINA_NT256: 256-column passes with two TMEM stages (dense kernel)
    bool share = false;        // TINA_SHARE: clusters of four share the subfilter stage (dense kernel)
    bool no_out_tma = false;   // TINA_NO_OUT_TMA: real-kind epilogue through registers instead of TMA stores
    bool fir_simt = false;     // TINA_FIR_SIMT: tina_fir on the CUDA-core kernel even where the Toeplitz path applies
    bool fir_v1 = false;       // TINA_FIR_V1: Toeplitz FIR through the round-1 route (pfb_umma_kernel) instead of fir_umma_kernel
    bool ct_no_ws = false;     // TINA_CT_NO_WS: factorised complex kernel without warp specialisation
    bool ctr_ws = false;       // TINA_CTR_WS: warp-specialised factorised real kernel
    bool no_sym = false;       // TINA_NO_SYM: complex dense contraction without the k <-> P-k column pairing
    bool sym_v1 = false;       // TINA_SYM_V1: column-paired contraction with register-window producers (no TMA input staging)
    bool fold = false;         // TINA_SYM_FOLD: complex kind with the row pairs folded as well (pfb_symf_kernel; measured: no faster)
    // -DTINA_DEV only (always 0 / false otherwise):
    int debug_skip = 0, ksplit = 0, a_slots = 0, b_entries = 0, cl4 = 0;
    bool prof = false;
};
const Options& options();
void reload_options();

// ---- cache of encoded TMA tensor maps (per device): a map is a pure function of base pointer, shape and box, so
// a call that repeats the pointers and sizes of an earlier one skips its cuTensorMapEncodeTiled calls
struct TmapKey {
    const void* p[3];          // base pointers (input, window / taps, output)
    long long n[2];            // n_samples / L, ...
    int i[6];                  // S / C, P, M, kind, tap-count template, caller tag
    bool operator==(const TmapKey& o) const { return memcmp(this, &o, sizeof(TmapKey)) == 0; }
};
struct TmapSet { alignas(64) unsigned char m[4][128]; };   // up to four CUtensorMap (128 bytes each)

// ---- per-device state: SM count, kernels whose >48 KB dynamic shared memory opt-in has been set ---
struct DevCtx {
    int dev = -1;
    int n_sm = 0;
    std::mutex mu;
    std::map<const void*, int> smem_attr;   // kernel -> bytes opted in on this device
    std::map<const void*, int> occupancy;   // kernel -> resident CTAs per SM (cached query)
    void* tz_ring = nullptr;                // Toeplitz scratch of tina_fir (tina_umma.cu)
    std::atomic<unsigned> tz_next{0};
    // tina_pfb_batched_host: staging buffers, internal streams and events (tina_api.cu)
    void* stage_p[3] = {nullptr, nullptr, nullptr};
    size_t stage_n[3] = {0, 0, 0};
    cudaStream_t s_in = nullptr, s_cmp = nullptr, s_out = nullptr;
    cudaEvent_t ev_start = nullptr, ev_in[64] = {}, ev_cmp[64] = {};
    std::mutex host_mu;                     // serialises tina_pfb_batched_host on this device
    std::vector<std::pair<TmapKey, TmapSet>> tmaps;   // small round-robin cache (guarded by mu)
    unsigned tmap_next = 0;
};
bool tmap_cache_get(DevCtx* ctx, const TmapKey& key, TmapSet* out);
void tmap_cache_put(DevCtx* ctx, const TmapKey& key, const TmapSet& set);
// context of the CURRENT device (cudaGetDevice), created on first use; the registry is mutex-guarded
tina_status dev_ctx(DevCtx** out);
// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) once per (device, kernel)
tina_status ensure_smem(DevCtx* ctx, const void* func, int bytes, const char* what);
void dev_ctx_release_all();                 // frees per-device scratch (tina_clear_plan_cache)

inline void note_kernel(const char* name, double issued_ratio = 1.0)
{
    g_last_kernel.store(name, std::memory_order_relaxed);
    g_last_issued_ratio.store(issued_ratio, std::memory_order_relaxed);
}
inline void count_launch(int n = 1) { g_launches.fetch_add(n, std::memory_order_relaxed); }
inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// ---- generic CUDA-core path (tina_simt.cu) ------------------------------------------
tina_status simt_fir(const float* x, const float* taps, float* y, int C, long long L, int M,
                     cudaStream_t st, bool per_channel = false);
tina_status simt_unfold(const float* x, float* y, long long I, int J, cudaStream_t st);
// PFB / DFT on CUDA cores: window == nullptr means M == 1 with unit taps (plain DFT).
tina_status simt_pfb(const void* x, int S, long long n_samples, int P, int M, const float* window,
                     bool real, bool inverse, void* out, cudaStream_t st);
tina_status simt_pfb_fir(const void* x, int S, long long n_samples, int P, int M,
                         const float* window, bool real, void* y, cudaStream_t st);

// ---- measured arithmetic ceilings (tina_peaks.cu) -----------------------------------
tina_status probe_peak(int which, int iters, double* tflops, double* ms_out, cudaStream_t st);

// ---- tcgen05 tensor-core path (tina_umma.cu) ----------------------------------------
bool umma_supported(int P, bool real);
tina_status umma_pfb(const void* x, int S, long long n_samples, int P, int M, const float* window,
                     bool real, bool inverse, tina_precision prec, void* out, cudaStream_t st);
void umma_clear_plans();
// complex kind with every distinct column pair (k, P-k) of the Fourier matrix contracted once (tina_sym.cu)
bool sym_supported(int P);
bool sym_real_supported(int P);     // real kind: even / odd samples against the columns of the bins [0, P/4)
tina_status sym_pfb(const void* x, int S, long long n_samples, int P, int M, const float* window, bool real, bool inverse,
                    tina_precision prec, void* out, cudaStream_t st);
// complex kind with the row pairs (p, P-p) folded as well (tina_symf.cu): window == nullptr or M <= 16
bool symf_supported(int P, int M, bool has_window);
tina_status symf_pfb(const void* x, int S, long long n_samples, int P, int M, const float* window, bool inverse,
                     tina_precision prec, void* out, cudaStream_t st);
void symf_clear_plans();
// PFB with the factorised (two-stage, 32 x 32) Fourier stage: complex kind, P = 1024, M <= 16 (tina_ct.cu)
tina_status ct_pfb(const void* x, int S, long long n_samples, int M, const float* window, void* out, cudaStream_t st);
tina_status arith_ew(const float* a, const float* b, float* o, long long n, bool mul, cudaStream_t st);
tina_status arith_sum(const float* x, long long rows, long long n, float* out, cudaStream_t st);
tina_status arith_matmul(const float* x, const float* y, float* z, long long M, long long L, long long N, cudaStream_t st);
tina_status ctr_pfb(const void* x, int S, long long n_samples, int M, const float* window, void* out, cudaStream_t st);
// standalone FIR as a Toeplitz contraction with a resident matrix and TMA-staged signal (tina_firt.cu);
// false = shape not covered (L % 128 != 0 or M > 193): fall back to umma_fir / simt_fir
bool firt_fir(const float* x, const float* taps, float* y, int C, long long L, int M, bool per_channel, cudaStream_t st,
              tina_status* status);
// standalone FIR as a Toeplitz contraction on the tensor cores; false = shape not covered (use simt_fir)
bool umma_fir(const float* x, const float* taps, float* y, int C, long long L, int M, cudaStream_t st,
              tina_status* status);
// subfilter stage only with the register-window kernel; false = shape not covered (use simt_pfb_fir)
bool umma_pfb_fir(const void* x, int S, long long n_samples, int P, int M, const float* window, bool real,
                  void* y, cudaStream_t st, tina_status* status);

}  // namespace tina
