// tina_common.cuh -- shared host-side helpers of libtina (status text, launch counter).
#pragma once
#include <cuda_runtime.h>
#include <atomic>
#include <cstdarg>
#include <cstdint>
#include <cstdio>

#include "../../include/tina.h"

namespace tina {

constexpr int kMaxP = 8192;      // upper bound on P / N (DFT size)
constexpr int kMaxTapsPfb = 64;  // upper bound on M for the PFB
constexpr int kMaxTapsFir = 4096;

enum Path { kPathNone = 0, kPathSimt = 1, kPathUmma = 2 };

extern std::atomic<long long> g_launches;
extern std::atomic<int> g_last_path;

void set_error(const char* fmt, ...);
tina_status fail(tina_status s, const char* fmt, ...);
tina_status check_cuda(cudaError_t e, const char* what);

inline void count_launch(int n = 1) { g_launches.fetch_add(n, std::memory_order_relaxed); }
inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// ---- generic CUDA-core path (tina_simt.cu) ------------------------------------------
tina_status simt_fir(const float* x, const float* taps, float* y, int C, long long L, int M,
                     cudaStream_t st);
tina_status simt_unfold(const float* x, float* y, long long I, int J, cudaStream_t st);
// PFB / DFT on CUDA cores: window == nullptr means M == 1 with unit taps (plain DFT).
tina_status simt_pfb(const void* x, int S, long long n_samples, int P, int M, const float* window,
                     bool real, bool inverse, void* out, cudaStream_t st);
tina_status simt_pfb_fir(const void* x, int S, long long n_samples, int P, int M,
                         const float* window, bool real, void* y, cudaStream_t st);

// ---- tcgen05 tensor-core path (tina_umma.cu) ----------------------------------------
bool umma_supported(int P, bool real);
tina_status umma_pfb(const void* x, int S, long long n_samples, int P, int M, const float* window,
                     bool real, bool inverse, tina_precision prec, void* out, cudaStream_t st);
void umma_clear_plans();
// PFB with the factorised (two-stage, 32 x 32) Fourier stage: complex kind, P = 1024, M <= 16 (tina_ct.cu)
tina_status ct_pfb(const void* x, int S, long long n_samples, int M, const float* window, void* out, cudaStream_t st);
tina_status arith_ew(const float* a, const float* b, float* o, long long n, bool mul, cudaStream_t st);
tina_status arith_sum(const float* x, long long rows, long long n, float* out, cudaStream_t st);
tina_status arith_matmul(const float* x, const float* y, float* z, long long M, long long L, long long N, cudaStream_t st);
tina_status ctr_pfb(const void* x, int S, long long n_samples, int M, const float* window, void* out, cudaStream_t st);
// standalone FIR as a Toeplitz contraction on the tensor cores; false = shape not covered (use simt_fir)
bool umma_fir(const float* x, const float* taps, float* y, int C, long long L, int M, cudaStream_t st,
              tina_status* status);
// subfilter stage only with the register-window kernel; false = shape not covered (use simt_pfb_fir)
bool umma_pfb_fir(const void* x, int S, long long n_samples, int P, int M, const float* window, bool real,
                  void* y, cudaStream_t st, tina_status* status);

}  // namespace tina
