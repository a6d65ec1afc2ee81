// tina_simt.cu -- CUDA-core kernels of libtina (sm_100a):
//   * fir_kernel        standalone FIR, Eq. (15) PAPER.md:171 (register-tiled, smem-staged)
//   * pfb_simt_kernel   generic-size PFB / DFT: Eq. (20) PAPER.md:230 + direct DFT Eq. (12)/(14)
//   * pfb_fir_kernel    subfilter stage only (Fig. 3 left column)
// These serve sizes the tcgen05 path does not cover and the HBM-bound regime (small P).
#include "tina_common.cuh"

namespace tina {

// =====================================================================================
// FIR: y[c][j] = sum_k a[k] x[c][j + M-1-k] = sum_i a[M-1-i] x[c][j+i]
// One CTA computes FIR_TILE consecutive outputs of one channel.  Each thread owns 8
// consecutive outputs and slides an 8-register window over the staged input, so the hot
// loop is 64 FFMA per 8 LDS(x) + 2 broadcast LDS.128 (taps).  The staged input uses a
// 9-words-per-8 skew so that the stride-8 per-thread walk is bank-conflict free.
// =====================================================================================
constexpr int FIR_THREADS = 256;
constexpr int FIR_PER_THREAD = 8;
constexpr int FIR_TILE = FIR_THREADS * FIR_PER_THREAD;  // 2048 outputs per CTA

__device__ __forceinline__ int skew(int e) { return e + (e >> 3); }

__global__ void __launch_bounds__(FIR_THREADS)
fir_kernel(const float* __restrict__ x, const float* __restrict__ taps, float* __restrict__ y,
           long long L, int M, long long Lo, int tiles_per_chan)
{
    extern __shared__ __align__(16) float smem[];
    const int Mp = (M + 7) & ~7;                       // taps padded to a multiple of 8
    float* s_taps = smem;                              // [Mp]  reversed: s_taps[i] = a[M-1-i]
    float* s_x = smem + Mp;                            // skewed [FIR_TILE + Mp + 8]

    const int c = blockIdx.x / tiles_per_chan;
    const long long j0 = (long long)(blockIdx.x % tiles_per_chan) * FIR_TILE;
    const float* xc = x + (long long)c * L;
    const int n_out = (int)min((long long)FIR_TILE, Lo - j0);
    const int n_in = n_out + M - 1;
    const int n_stage = FIR_TILE + Mp + 8;

    for (int i = threadIdx.x; i < Mp; i += FIR_THREADS) s_taps[i] = (i < M) ? taps[M - 1 - i] : 0.f;
    for (int e = threadIdx.x; e < n_stage; e += FIR_THREADS)
        s_x[skew(e)] = (e < n_in) ? __ldg(xc + j0 + e) : 0.f;
    __syncthreads();

    const int t0 = threadIdx.x * FIR_PER_THREAD;
    float acc[8], xr[8];
#pragma unroll
    for (int r = 0; r < 8; ++r) { acc[r] = 0.f; xr[r] = s_x[skew(t0 + r)]; }

    for (int i0 = 0; i0 < Mp; i0 += 8) {
        const float4 ta = *reinterpret_cast<const float4*>(s_taps + i0);
        const float4 tb = *reinterpret_cast<const float4*>(s_taps + i0 + 4);
        const float tp[8] = {ta.x, ta.y, ta.z, ta.w, tb.x, tb.y, tb.z, tb.w};
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int r = 0; r < 8; ++r) acc[r] = fmaf(tp[u], xr[(r + u) & 7], acc[r]);
            xr[u] = s_x[skew(t0 + i0 + u + 8)];       // slot u held x[t0+i0+u], no longer needed
        }
    }
    __syncthreads();                                   // everyone done reading s_x
#pragma unroll
    for (int r = 0; r < 8; ++r) s_x[skew(t0 + r)] = acc[r];
    __syncthreads();
    float* yc = y + (long long)c * Lo + j0;
    for (int e = threadIdx.x; e < n_out; e += FIR_THREADS) yc[e] = s_x[skew(e)];
}

tina_status simt_fir(const float* x, const float* taps, float* y, int C, long long L, int M,
                     cudaStream_t st)
{
    const long long Lo = L - M + 1;
    const long long tiles = (Lo + FIR_TILE - 1) / FIR_TILE;
    if (tiles * C > 0x7fffffffLL) return fail(TINA_ERR_UNSUPPORTED, "tina_fir: C*L too large for one grid");
    const int Mp = (M + 7) & ~7;
    const int n_stage = FIR_TILE + Mp + 8;
    const size_t smem = sizeof(float) * (Mp + n_stage + (n_stage >> 3) + 8);
    static bool attr_done = false;
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(fir_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024);
        if (e != cudaSuccess) return check_cuda(e, "cudaFuncSetAttribute(fir_kernel)");
        attr_done = true;
    }
    fir_kernel<<<(unsigned)(tiles * C), FIR_THREADS, smem, st>>>(x, taps, y, L, M, Lo, (int)tiles);
    count_launch();
    g_last_path = kPathSimt;
    return check_cuda(cudaGetLastError(), "fir_kernel launch");
}

// =====================================================================================
// Generic-size PFB / DFT on CUDA cores.
// One CTA handles TF consecutive frames of one stream: (1) subfilter stage into a shared
// y tile, Eq. (20); (2) direct DFT across the P branches with a shared twiddle table
// W[r] = exp(-+2 pi i r / P), r = (p k) mod P advanced in integers.
// =====================================================================================
constexpr int PFB_SIMT_THREADS = 256;

template <bool REAL>
__global__ void __launch_bounds__(PFB_SIMT_THREADS)
pfb_simt_kernel(const void* __restrict__ x_, long long stream_stride, int P, int M,
                const float* __restrict__ window, long long F, int TF, int tiles_per_stream,
                int inverse, float scale, void* __restrict__ out_)
{
    extern __shared__ __align__(16) float smem[];
    float2* s_w = reinterpret_cast<float2*>(smem);                 // [P] twiddles
    float*  s_y = smem + 2 * P;                                    // [TF][P] (float or float2)

    const int s = blockIdx.x / tiles_per_stream;
    const long long f0 = (long long)(blockIdx.x % tiles_per_stream) * TF;
    const int nf = (int)min((long long)TF, F - f0);
    const int NK = REAL ? P / 2 + 1 : P;

    for (int r = threadIdx.x; r < P; r += blockDim.x) {
        double sn, cs;
        sincospi(2.0 * (double)r / (double)P, &sn, &cs);
        s_w[r] = make_float2((float)cs, (float)(inverse ? sn : -sn));
    }
    // ---- subfilter stage -------------------------------------------------------------
    if (REAL) {
        const float* x = reinterpret_cast<const float*>(x_) + (long long)s * stream_stride;
        for (int e = threadIdx.x; e < nf * P; e += blockDim.x) {
            const int f = e / P, p = e - f * P;
            float acc = 0.f;
            if (window) {
                for (int m = 0; m < M; ++m)
                    acc = fmaf(__ldg(window + (long long)m * P + p),
                               __ldg(x + (f0 + f + M - 1 - m) * P + p), acc);
            } else {
                acc = __ldg(x + (f0 + f) * P + p);
            }
            s_y[e] = acc;
        }
    } else {
        const float2* x = reinterpret_cast<const float2*>(x_) + (long long)s * stream_stride;
        float2* sy = reinterpret_cast<float2*>(s_y);
        for (int e = threadIdx.x; e < nf * P; e += blockDim.x) {
            const int f = e / P, p = e - f * P;
            float2 acc = make_float2(0.f, 0.f);
            if (window) {
                for (int m = 0; m < M; ++m) {
                    const float h = __ldg(window + (long long)m * P + p);
                    const float2 v = __ldg(x + (f0 + f + M - 1 - m) * P + p);
                    acc.x = fmaf(h, v.x, acc.x);
                    acc.y = fmaf(h, v.y, acc.y);
                }
            } else {
                acc = __ldg(x + (f0 + f) * P + p);
            }
            sy[e] = acc;
        }
    }
    __syncthreads();
    // ---- Fourier stage ---------------------------------------------------------------
    float2* out = reinterpret_cast<float2*>(out_) + ((long long)s * F + f0) * NK;
    for (int e = threadIdx.x; e < nf * NK; e += blockDim.x) {
        const int f = e / NK, k = e - f * NK;
        float ar = 0.f, ai = 0.f;
        int r = 0;
        if (REAL) {
            const float* yr = s_y + f * P;
            for (int p = 0; p < P; ++p) {
                const float2 w = s_w[r];
                ar = fmaf(yr[p], w.x, ar);
                ai = fmaf(yr[p], w.y, ai);
                r += k; if (r >= P) r -= P;
            }
        } else {
            const float2* yc = reinterpret_cast<const float2*>(s_y) + f * P;
            for (int p = 0; p < P; ++p) {
                const float2 w = s_w[r];
                const float2 v = yc[p];
                ar = fmaf(v.x, w.x, ar); ar = fmaf(-v.y, w.y, ar);
                ai = fmaf(v.x, w.y, ai); ai = fmaf(v.y, w.x, ai);
                r += k; if (r >= P) r -= P;
            }
        }
        out[e] = make_float2(ar * scale, ai * scale);
    }
}

tina_status simt_pfb(const void* x, int S, long long n_samples, int P, int M, const float* window,
                     bool real, bool inverse, void* out, cudaStream_t st)
{
    const long long F = n_samples / P - M + 1;
    const int elem = real ? 1 : 2;                       // floats per y element
    const long long budget = 40 * 1024 / 4;              // floats of smem for the y tile
    int TF = (int)(budget / ((long long)P * elem));
    if (TF < 1) TF = 1;
    if (TF > 64) TF = 64;
    // keep at least ~2 waves of CTAs when the problem is small
    while (TF > 1 && (F + TF - 1) / TF * S < 2 * 148) TF >>= 1;
    const long long tiles = (F + TF - 1) / TF;
    if (tiles * S > 0x7fffffffLL) return fail(TINA_ERR_UNSUPPORTED, "tina_pfb: too many tiles");
    const size_t smem = sizeof(float) * (2 * (size_t)P + (size_t)TF * P * elem);
    static bool attr_done = false;
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(pfb_simt_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(pfb_simt_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        if (e != cudaSuccess) return check_cuda(e, "cudaFuncSetAttribute(pfb_simt_kernel)");
        attr_done = true;
    }
    const float scale = inverse ? (float)(1.0 / (double)P) : 1.f;
    if (real)
        pfb_simt_kernel<true><<<(unsigned)(tiles * S), PFB_SIMT_THREADS, smem, st>>>(
            x, n_samples, P, M, window, F, TF, (int)tiles, inverse ? 1 : 0, scale, out);
    else
        pfb_simt_kernel<false><<<(unsigned)(tiles * S), PFB_SIMT_THREADS, smem, st>>>(
            x, n_samples, P, M, window, F, TF, (int)tiles, inverse ? 1 : 0, scale, out);
    count_launch();
    g_last_path = kPathSimt;
    return check_cuda(cudaGetLastError(), "pfb_simt_kernel launch");
}

// =====================================================================================
// Subfilter stage only: y[s][f][p] = sum_m w[mP+p] x[s][(f+M-1-m)P+p].
// A thread owns one 8-byte column (one complex sample, or two adjacent real branches) and
// RUN consecutive frames, walking the RUN+M-1 input rows once: HBM sees each sample once,
// the (M-1)-row halo between neighbouring runs is served by L2.
// =====================================================================================
constexpr int PF_RUN = 16;

template <bool REAL>
__global__ void __launch_bounds__(256)
pfb_fir_kernel(const float2* __restrict__ x, long long stream_stride2, int P2, int M,
               const float* __restrict__ window, long long F, float2* __restrict__ y,
               long long total_cols, int runs_per_stream)
{
    // column index c in [0,P2): float2 column (P2 = P for complex, P/2 for real)
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= total_cols) return;
    const int c = (int)(gid % P2);
    const long long rs = gid / P2;
    const int run = (int)(rs % runs_per_stream);
    const int s = (int)(rs / runs_per_stream);
    const long long f0 = (long long)run * PF_RUN;
    const int nf = (int)min((long long)PF_RUN, F - f0);
    const float2* xs = x + (long long)s * stream_stride2 + c;
    const int Pw = REAL ? 2 * P2 : P2;                   // window row length P

    float2 acc[PF_RUN];
#pragma unroll
    for (int r = 0; r < PF_RUN; ++r) acc[r] = make_float2(0.f, 0.f);
    for (int i = 0; i < nf + M - 1; ++i) {
        const float2 v = __ldg(xs + (f0 + i) * P2);
#pragma unroll
        for (int r = 0; r < PF_RUN; ++r) {
            const int m = r + M - 1 - i;                 // input row f0+i feeds frame f0+r with tap m
            if (m >= 0 && m < M && r < nf) {
                if (REAL) {
                    const float2 h = __ldg(reinterpret_cast<const float2*>(window + (long long)m * Pw) + c);
                    acc[r].x = fmaf(h.x, v.x, acc[r].x);
                    acc[r].y = fmaf(h.y, v.y, acc[r].y);
                } else {
                    const float h = __ldg(window + (long long)m * Pw + c);
                    acc[r].x = fmaf(h, v.x, acc[r].x);
                    acc[r].y = fmaf(h, v.y, acc[r].y);
                }
            }
        }
    }
    float2* ys = y + ((long long)s * F + f0) * P2 + c;
#pragma unroll
    for (int r = 0; r < PF_RUN; ++r)
        if (r < nf) ys[(long long)r * P2] = acc[r];
}

tina_status simt_pfb_fir(const void* x, int S, long long n_samples, int P, int M,
                         const float* window, bool real, void* y, cudaStream_t st)
{
    const long long F = n_samples / P - M + 1;
    const int P2 = real ? P / 2 : P;
    const long long stride2 = real ? n_samples / 2 : n_samples;
    const long long runs = (F + PF_RUN - 1) / PF_RUN;
    const long long total = runs * S * P2;
    const long long blocks = (total + 255) / 256;
    if (blocks > 0x7fffffffLL) return fail(TINA_ERR_UNSUPPORTED, "tina_pfb_fir: too large");
    if (real)
        pfb_fir_kernel<true><<<(unsigned)blocks, 256, 0, st>>>(
            (const float2*)x, stride2, P2, M, window, F, (float2*)y, total, (int)runs);
    else
        pfb_fir_kernel<false><<<(unsigned)blocks, 256, 0, st>>>(
            (const float2*)x, stride2, P2, M, window, F, (float2*)y, total, (int)runs);
    count_launch();
    g_last_path = kPathSimt;
    return check_cuda(cudaGetLastError(), "pfb_fir_kernel launch");
}

}  // namespace tina
