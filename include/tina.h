/*
 * tina.h -- C ABI of libtina: the FIR / DFT / IDFT / Polyphase-Filter-Bank hot path of
 * arxiv 2408.16551 ("TINA"), hand-written CUDA for NVIDIA B200 (sm_100a).
 *
 * All data pointers are DEVICE pointers owned by the caller (e.g. allocated by PyTorch)
 * unless a function name ends in `_host`.  Every call validates its arguments on the
 * host, enqueues its kernels on `stream` (a cudaStream_t passed as void*, NULL = the
 * legacy default stream) and returns WITHOUT synchronising.  The caller must keep
 * x / taps / window / out alive and unmodified until the stream has passed the enqueued
 * work.  The library owns only its plan cache (twiddle matrices + TMA tensor maps, created
 * lazily on first use of a (size, kind, direction, precision) tuple -- that first call
 * allocates device memory and synchronises once), released by tina_clear_plan_cache().
 *
 * Errors: integer status only; nothing is written to the outputs on error; no exceptions,
 * no exit(), no CPU fallback, no other backend.  tina_last_error() gives thread-local text.
 * Thread-safety: the plan cache, the per-device state (SM count, shared-memory opt-ins, scratch) and
 * the option block are behind mutexes; every device entry point may be called concurrently from
 * several host threads and on several devices of one process (state is kept per CUDA device; the
 * current device at call time is the one used).  The `_host` entry point serialises per device.
 * Environment: TINA_* variant switches (TINA_SHARE, TINA_NT256, TINA_NO_OUT_TMA, TINA_FIR_SIMT,
 * TINA_FIR_V1, TINA_CT_NO_WS, TINA_CTR_WS, TINA_NO_SYM, TINA_SYM_V1) select between kernels that compute the same result under the
 * same contract; they are read once (tina_reload_options() re-reads them).  Knobs that skip work or
 * change the accuracy contract exist only in development builds (-DTINA_DEV, tina_build_is_dev()).
 *
 * Notation (0-based everywhere; PAPER.md = /root/reference/PAPER.md):
 *   P  channels / polyphase branches        M  taps per branch
 *   NB = floor(n_samples / P) input blocks   F = NB - M + 1 output frames ("spectra")
 */
#ifndef TINA_H_
#define TINA_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    TINA_OK                = 0,
    TINA_ERR_NULL_POINTER  = 1,
    TINA_ERR_BAD_SHAPE     = 2,  /* sizes < 1, L < M, F < 1, in-place call, odd P for the real kind */
    TINA_ERR_UNSUPPORTED   = 3,  /* size outside the supported set stated per function              */
    TINA_ERR_ALIGNMENT     = 4,  /* a base pointer is not 16-byte aligned                            */
    TINA_ERR_CUDA          = 5,  /* a CUDA runtime / driver call failed; see tina_last_error()       */
    TINA_ERR_OUT_OF_MEMORY = 6
} tina_status;

typedef enum { TINA_COMPLEX = 0, TINA_REAL = 1 } tina_kind;       /* "real_or_complex" input   */

typedef enum {
    TINA_PREC_FP32 = 0,   /* fp32-accurate: error-compensated bf16x3 tensor-core contraction
                             (rel. L2 per frame <= 1e-5 against a float64 reference)           */
    TINA_PREC_BF16 = 1,   /* single-pass bf16 operands, fp32 accumulate (<= 2e-2)              */
    TINA_PREC_FP16 = 2    /* single-pass fp16 operands, fp32 accumulate (the paper's "16 bit",
                             PAPER.md:206): ~5e-4, but |subfiltered sample| must stay < 65504  */
} tina_precision;

/* ---------------------------------------------------------------------------------------
 * FIR filter, Eq. (15), valid mode:
 *     y[c][j] = sum_{k=0}^{M-1} taps[k] * x[c][j + M-1 - k],   j in [0, L-M+1)
 * i.e. a true convolution y(i) = sum_k a(k) x(i-k) evaluated for every i whose whole
 * history exists; the impulse response equals the taps in order.
 *   x    [C][L]       float32, row-major (device)
 *   taps [M]          float32, shared by all C channels (device)
 *   y    [C][L-M+1]   float32, row-major (device), must not overlap x
 * Supported: C >= 1, 1 <= M <= 4096, L >= M.  Even L with M <= 193 runs as a banded-Toeplitz
 * contraction on the tensor cores (blocks of 128 outputs, bf16x3 error-compensated, rel. L2 per
 * channel <= 1e-5, the unfolding view of Eq. (17)-(19)) -- with L % 128 == 0 on
 * the kernel that keeps the Toeplitz band matrix resident in shared memory, stages the signal by
 * TMA and holds the signal operand in tensor memory; any other shape on the CUDA-core
 * register-window kernel (fp32 FMA).  Errors: NULL_POINTER, BAD_SHAPE, UNSUPPORTED
 * (M > 4096), ALIGNMENT (x, y not 16-byte aligned), CUDA.                                          */
tina_status tina_fir(const float* x, const float* taps, float* y,
                     int C, long long L, int M, void* stream);

/* FIR with one tap vector PER CHANNEL: the "multiple FIR filters" that the PFB's subfilter stage
 * combines (Eq. (20): branch p is filtered with its own h_p), each
 * channel being Eq. (15) in valid mode:
 *     y[c][j] = sum_{k=0}^{M-1} taps[c][k] * x[c][j + M-1 - k],   j in [0, L-M+1)
 *   x    [C][L]       float32 (device)      taps [C][M] float32, row c = channel c's taps (device)
 *   y    [C][L-M+1]   float32 (device), must not overlap x
 * Supported: C >= 1, 1 <= M <= 4096, L >= M.  L % 128 == 0 with M <= 193 runs on the tensor-core
 * Toeplitz kernel (the band matrix is rebuilt in shared memory whenever the channel changes; same
 * 1e-5 contract), any other shape on the CUDA-core register-window kernel (fp32 FMA).
 * Errors as tina_fir.                                                                              */
tina_status tina_fir_multi(const float* x, const float* taps, float* y,
                           int C, long long L, int M, void* stream);

/* ---------------------------------------------------------------------------------------
 * DFT / inverse DFT as a dense contraction against the Fourier matrix,
 * Eq. (12) / Eq. (14):
 *     out[b][k] = s * sum_{n=0}^{N-1} x[b][n] * exp(-+ 2 pi i n k / N)
 * forward (inverse == 0): sign -, s = 1;  inverse (inverse != 0): sign +, s = 1/N.
 *   x, out [B][N] complex64, interleaved (re, im) float32 (device); in-place (x == out)
 *   is NOT supported -> BAD_SHAPE.
 * Supported: B >= 1, 2 <= N <= 8192.  N % 32 == 0 runs on the tcgen05 tensor-core path,
 * any other N on the generic CUDA-core path (fp32 regardless of `prec`).                  */
tina_status tina_dft(const void* x, void* out, long long B, int N, int inverse,
                     tina_precision prec, void* stream);

/* ---------------------------------------------------------------------------------------
 * Polyphase filter bank: subfilter stage Eq. (20) followed by a P-point DFT
 * across the branches, fused in one kernel for every M <= 64 when P is a multiple of 64 (the
 * subfiltered signals never touch HBM; 16 < M <= 64 taps are processed in groups of 16 inside the kernel).  Only for
 * 16 < M <= 64 with a P the tensor-core kernel does not tile (not a multiple of 64) the subfilter stage runs as its
 * own kernel into a stream-ordered temporary of S*F*P samples, followed by the contraction -- two launches:
 *     y[f][p] = sum_{m=0}^{M-1} window[m P + p] * x[(f + M-1 - m) P + p]
 *     out[f][k] = sum_{p=0}^{P-1} y[f][p] * exp(-2 pi i p k / P)
 * with x_p(n') = x[n' P + p], h_p(m) = window[m P + p], frame f <-> n' = f + M-1.
 *   x       n_samples complex64 (kind = COMPLEX) or float32 (kind = REAL) (device);
 *           the trailing n_samples mod P samples are ignored
 *   window  [P*M] float32 prototype filter (device)
 *   out     [F][P] complex64 (COMPLEX, k in [0,P)) or [F][P/2+1] complex64 (REAL, half
 *           spectrum k in [0,P/2]) (device), F = tina_pfb_num_frames(n_samples, P, M)
 * Supported: 2 <= P <= 8192 (even for REAL), 1 <= M <= 64, F >= 1.  COMPLEX with
 * P % 32 == 0 and REAL with P % 64 == 0 run on the tensor-core path; other P on the
 * generic CUDA-core path (fp32 regardless of `prec`).  Where P % 64 == 0 (REAL: and P >= 128)
 * the tensor-core path contracts every distinct column pair of the Fourier matrix once
 * (bins k and P-k, REAL: k and P/2-k, share their cosine / sine sums; half the tensor
 * flops, same result and contract) with the input window and taps staged by TMA.
 * tina_pfb_batched: S independent streams in one launch, x [S][n_samples],
 * out [S][F][...]; n_samples must then keep every stream 16-byte aligned
 * (n_samples even for COMPLEX, % 4 == 0 for REAL) else ALIGNMENT.                          */
tina_status tina_pfb(const void* x, long long n_samples, int P, int M, const float* window,
                     tina_kind kind, tina_precision prec, void* out, void* stream);
tina_status tina_pfb_batched(const void* x, int S, long long n_samples, int P, int M,
                             const float* window, tina_kind kind, tina_precision prec,
                             void* out, void* stream);

/* PFB with a FACTORISED Fourier stage ("either a Discrete or Fast Fourier Transform"):
 * same arguments and the same result as tina_pfb_batched (fp32-accurate, rel. L2 per frame <= 1e-5),
 * but the P-point DFT is computed as two stages of sqrt(P)-point DFTs (both stages tensor-core contractions
 * against one small Fourier matrix, twiddle multiply in between, all on chip): 16 P sqrt(P) instead of 8 P^2
 * flops per complex frame, i.e. HBM / FMA bound instead of tensor bound.  Reported separately from the dense
 * contraction that tina_pfb implements.  Supported in this version: kind = COMPLEX with P = 1024 (32 x 32),
 * M <= 16, and kind = REAL with P = 4096 (64 x 64; BASELINE config 5), M <= 8; anything else -> UNSUPPORTED. */
tina_status tina_pfb_fft_batched(const void* x, int S, long long n_samples, int P, int M,
                                 const float* window, tina_kind kind, void* out, void* stream);

/* Subfilter stage only (Eq. (20); Fig. 3 left column):
 *   y [S][F][P] complex64 (COMPLEX) or float32 (REAL).  Same argument rules as above.      */
tina_status tina_pfb_fir_batched(const void* x, int S, long long n_samples, int P, int M,
                                 const float* window, tina_kind kind, void* y, void* stream);

/* Host-buffer entry point (the end-to-end path timed as `e2e` by bench.py):
 * x_host / window_host / out_host are HOST pointers (pinned memory recommended; pageable memory
 * works but copies synchronously).  The call allocates device staging buffers on first use (cached,
 * grown as needed), cuts the batch into pieces (whole streams, or frame ranges of a stream with
 * their (M-1)-block halo) and pipelines host->device copy, the device path and device->host copy of
 * successive pieces on three internal streams ordered after `stream`; it returns after the last
 * result byte has landed in out_host (SYNCHRONOUS).  Results are bit-identical to the device call.
 * Not re-entrant (the staging buffers are shared; concurrent calls serialise on a mutex).       */
tina_status tina_pfb_batched_host(const void* x_host, int S, long long n_samples, int P, int M,
                                  const float* window_host, tina_kind kind, tina_precision prec,
                                  void* out_host, void* stream);

/* Unfolding, Eq. (17): Y(i, j) = X(i + j), i in [0, I-J+1), j in [0, J)
 * -- e.g. X = [1,2,3,4], J = 2 gives [[1,2],[2,3],[3,4]] (the paper's worked example).
 *   x [I] float32 (device), y [I-J+1][J] float32 row-major (device), must not overlap x.
 * Supported: 1 <= J <= I.  Memory-bound gather (each output written once, coalesced; the J-fold
 * re-reads of x are served by L1 / L2).  Errors: NULL_POINTER, BAD_SHAPE, CUDA.                  */
tina_status tina_unfold(const float* x, float* y, long long I, int J, void* stream);

/* Arithmetic building blocks of the paper's section 3 (device pointers, float32, row-major):
 *   tina_mul    Eq. (6):   out[c] = a[c] * b[c],        c in [0, n)
 *   tina_add    Eq. (10):  out[c] = b[c] + a[c]
 *   tina_sum    Eq. (11):  out[r] = sum_c x[r][c],      x [rows][n], out [rows]; accumulated in
 *               short float32 chains combined in double precision; rows <= 65535; n = 0 gives 0
 *   tina_matmul Eq. (7):  z[m][n] = sum_l x[m][l] y[l][n],  x [M][L], y [L][N], z [M][N];
 *               float32 FMAs on the CUDA cores (a plain GEMM); z must not alias x or y; L = 0 gives zeros
 * out may alias a or b in tina_mul / tina_add.  n, rows, M, L, N >= 0 else BAD_SHAPE; NULL_POINTER for a null
 * pointer with non-empty data; CUDA on a launch failure.  All calls are asynchronous on `stream`.         */
tina_status tina_mul(const float* a, const float* b, float* out, long long n, void* stream);
tina_status tina_add(const float* a, const float* b, float* out, long long n, void* stream);
tina_status tina_sum(const float* x, long long rows, long long n, float* out, void* stream);
tina_status tina_matmul(const float* x, const float* y, float* z, long long M, long long L, long long N, void* stream);

/* tina_sum for callers that may not allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): Eq. (11) exactly as tina_sum computes it -- same blocks per
 * row, same float32 chains, same double-precision combination, so the results are bit-identical -- but the
 * per-block partial sums go to a file-scope `static __device__` array of 2 * TINA_SUM_STATIC_MAX_ROWS doubles
 * (64 KB) instead of a cudaMallocAsync temporary.  Every GPU that loads the library holds that array until the
 * process exits.  The call makes no cudaMalloc / cudaFree / allocating library call (its first use on a device
 * looks the array's address up with cudaGetSymbolAddress).  x, out: device pointers as in tina_sum.
 * Limit: rows <= TINA_SUM_STATIC_MAX_ROWS, else UNSUPPORTED (tina_last_error names the limit); n is unlimited.
 * ALL calls on a device share the one array: calls that overlap on the GPU (different streams, or graphs replayed
 * concurrently) race on it and give wrong sums -- order them on one stream or with events.  The array keeps the
 * previous call's partials; nothing needs clearing, because every entry a call reads it has written first.
 * Errors: BAD_SHAPE (negative size), UNSUPPORTED (rows over the limit), NULL_POINTER, CUDA.                   */
#define TINA_SUM_STATIC_MAX_ROWS 4096
tina_status tina_sum_static(const float* x, long long rows, long long n, float* out, void* stream);

/* F = floor(n_samples / P) - M + 1; <= 0 means the input is too short.                     */
long long   tina_pfb_num_frames(long long n_samples, int P, int M);

const char* tina_status_string(tina_status s);   /* static storage                          */
const char* tina_last_error(void);               /* thread-local detail text, "" if none    */
tina_status tina_clear_plan_cache(void);         /* frees cached twiddles / staging buffers */
int         tina_version(void);                  /* major*10000 + minor*100 + patch         */
tina_status tina_reload_options(void);           /* re-read the TINA_* variant switches     */
int         tina_build_is_dev(void);             /* 1: built with -DTINA_DEV (debug knobs)  */

/* Measured arithmetic ceilings of the device (bare loops, no memory traffic; the denominators of the
 * rooflines bench.py reports -- SURVEY.md section 8(d)).  which: 0 = fp32 fma.rn.f32 on the CUDA cores,
 * 1 = packed fma.rn.f32x2, 2 = tcgen05.mma kind::tf32, 3 = tcgen05.mma kind::f16 with bf16 operands
 * (M = 128, N = 256 per instruction, operands in shared memory), 4 / 5 = the bf16 loop with N = 128 / 64.  Runs `iters` loop iterations per thread
 * (FMA) or MMA groups per SM (tensor) after a short warm-up, SYNCHRONISES, and returns TFLOP/s in *tflops
 * and the elapsed milliseconds in *ms (host pointers; ms may be NULL).                                  */
tina_status tina_probe_peak(int which, int iters, double* tflops, double* ms, void* stream);

/* Introspection used by the tests and bench.py: number of kernel launches the library has
 * enqueued since process start (monotonic), and which path the last device call used
 * (0 = none yet, 1 = generic CUDA-core, 2 = tcgen05 tensor-core).                           */
long long   tina_launch_count(void);
int         tina_last_path(void);
/* Name of the kernel variant the last device call launched (static storage), and the tensor-core flops that
 * kernel issues PER PASS divided by the method's useful flops (8 P^2 per complex frame, 2 P^2 + 4 P per real
 * frame): 1.0 for the plain dense contraction, 0.5 where each distinct column pair of the Fourier matrix is
 * contracted once.  bench.py multiplies it by the number of bf16 passes (3 for TINA_PREC_FP32).          */
const char* tina_last_kernel(void);
double      tina_last_issued_ratio(void);

#ifdef __cplusplus
}
#endif
#endif /* TINA_H_ */
