// tina_arith.cu -- the arithmetic building blocks of the paper's section 3:
// elementwise multiply Eq. (6), elementwise add Eq. (10), summation Eq. (11), matrix-matrix multiply Eq. (7).
// The first three are HBM-bound streaming kernels (float4 grid-stride loops sized to the SM count); the matrix
// product is a register-tiled CUDA-core SGEMM (fp32 FMAs, 128 x 128 x 16 tiles) -- a plain GEMM, not the
// tensor-core path, which this library reserves for contractions against a FIXED matrix (DFT / Toeplitz).
#include "tina_common.cuh"

#include <cstdint>

namespace tina {

namespace {

int sm_count()
{
    DevCtx* ctx = nullptr;
    return dev_ctx(&ctx) == TINA_OK ? ctx->n_sm : 148;      // grid sizing only
}

template <bool MUL>
__global__ void __launch_bounds__(256)
ew_kernel(const float* __restrict__ a, const float* __restrict__ b, float* __restrict__ o, long long n, int vec)
{
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x, nth = (long long)gridDim.x * blockDim.x;
    long long done = 0;
    if (vec) {                                             // all three pointers 16-byte aligned
        const long long n4 = n >> 2;
        const float4* a4 = reinterpret_cast<const float4*>(a);
        const float4* b4 = reinterpret_cast<const float4*>(b);
        float4* o4 = reinterpret_cast<float4*>(o);
        for (long long i = tid; i < n4; i += nth) {
            const float4 u = __ldg(a4 + i), v = __ldg(b4 + i);
            o4[i] = MUL ? make_float4(u.x * v.x, u.y * v.y, u.z * v.z, u.w * v.w)
                        : make_float4(v.x + u.x, v.y + u.y, v.z + u.z, v.w + u.w);
        }
        done = n4 << 2;
    }
    for (long long i = done + tid; i < n; i += nth) o[i] = MUL ? a[i] * b[i] : b[i] + a[i];
}

// One block sums elements [bx * chunk, min(n, (bx + 1) * chunk)) of row r: eight independent fp32 accumulators per
// thread (short chains), then double precision across the thread, the warp and the block.
__global__ void __launch_bounds__(256)
sum_kernel(const float* __restrict__ x, long long n, long long chunk, double* __restrict__ partial, float* __restrict__ out)
{
    const long long r = blockIdx.y;
    const float* xr = x + r * n;
    const long long lo = (long long)blockIdx.x * chunk, hi = lo + chunk < n ? lo + chunk : n;
    float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    long long i = lo + threadIdx.x;
    for (; i + 7 * 256 < hi; i += 8 * 256) {
#pragma unroll
        for (int u = 0; u < 8; ++u) acc[u] += __ldg(xr + i + u * 256);
    }
    for (int u = 0; i < hi; i += 256, u = (u + 1) & 7) acc[u] += __ldg(xr + i);
    double s = 0.0;
#pragma unroll
    for (int u = 0; u < 8; ++u) s += (double)acc[u];
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
    __shared__ double ws[8];
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
#pragma unroll
        for (int w = 0; w < 8; ++w) t += ws[w];
        if (partial) partial[r * gridDim.x + blockIdx.x] = t;
        else out[r] = (float)t;
    }
}

__global__ void __launch_bounds__(256)
sum_final_kernel(const double* __restrict__ partial, int gx, float* __restrict__ out, long long rows)
{
    const long long r = (long long)blockIdx.x * 8 + (threadIdx.x >> 5);
    if (r >= rows) return;
    double s = 0.0;
    for (int i = threadIdx.x & 31; i < gx; i += 32) s += partial[r * gx + i];
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
    if ((threadIdx.x & 31) == 0) out[r] = (float)s;
}

// Z = X Y, row-major fp32.  128 x 128 output tile per 256-thread block, 8 x 8 outputs per thread (two 4-wide strips
// 64 apart in each direction so that shared-memory reads are conflict-free float4s), K stepped by 16 through shared
// memory; X is stored transposed ([k][m]) while it is staged.  Ragged edges are zero-filled on load and masked on store.
constexpr int GM = 128, GN = 128, GK = 16;

__global__ void __launch_bounds__(256)
matmul_kernel(const float* __restrict__ X, const float* __restrict__ Y, float* __restrict__ Z, long long M, long long L,
              long long N)
{
    __shared__ __align__(16) float xs[GK][GM + 4];
    __shared__ __align__(16) float ys[GK][GN + 4];
    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    const long long m0 = (long long)blockIdx.y * GM, n0 = (long long)blockIdx.x * GN;
    float acc[8][8];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[i][j] = 0.f;
    for (long long k0 = 0; k0 < L; k0 += GK) {
#pragma unroll
        for (int e = 0; e < 8; ++e) {                      // 128 x 16 elements of X: thread -> (row, k)
            const int idx = tid + e * 256, mm = idx >> 4, kk = idx & 15;
            xs[kk][mm] = (m0 + mm < M && k0 + kk < L) ? __ldg(X + (m0 + mm) * L + k0 + kk) : 0.f;
        }
#pragma unroll
        for (int e = 0; e < 8; ++e) {                      // 16 x 128 elements of Y: thread -> (k, col)
            const int idx = tid + e * 256, kk = idx >> 7, nn = idx & 127;
            ys[kk][nn] = (k0 + kk < L && n0 + nn < N) ? __ldg(Y + (k0 + kk) * N + n0 + nn) : 0.f;
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < GK; ++kk) {
            const float4 a0 = *reinterpret_cast<const float4*>(&xs[kk][4 * ty]);
            const float4 a1 = *reinterpret_cast<const float4*>(&xs[kk][64 + 4 * ty]);
            const float4 b0 = *reinterpret_cast<const float4*>(&ys[kk][4 * tx]);
            const float4 b1 = *reinterpret_cast<const float4*>(&ys[kk][64 + 4 * tx]);
            const float av[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
            const float bv[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 8; ++j) acc[i][j] = fmaf(av[i], bv[j], acc[i][j]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const long long m = m0 + (i < 4 ? 4 * ty + i : 64 + 4 * ty + i - 4);
        if (m >= M) continue;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const long long n = n0 + (j < 4 ? 4 * tx + j : 64 + 4 * tx + j - 4);
            if (n < N) Z[m * N + n] = acc[i][j];
        }
    }
}

}  // namespace

tina_status arith_ew(const float* a, const float* b, float* o, long long n, bool mul, cudaStream_t st)
{
    if (n == 0) return TINA_OK;
    const int vec = ((reinterpret_cast<uintptr_t>(a) | reinterpret_cast<uintptr_t>(b) | reinterpret_cast<uintptr_t>(o)) & 15) == 0;
    long long blocks = (n / 4 + 255) / 256;
    const long long cap = (long long)sm_count() * 8;
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    if (mul) ew_kernel<true><<<(unsigned)blocks, 256, 0, st>>>(a, b, o, n, vec);
    else ew_kernel<false><<<(unsigned)blocks, 256, 0, st>>>(a, b, o, n, vec);
    count_launch();
    g_last_path = kPathSimt; note_kernel("ew_kernel");
    return check_cuda(cudaGetLastError(), "ew_kernel launch");
}

tina_status arith_sum(const float* x, long long rows, long long n, float* out, cudaStream_t st)
{
    if (rows == 0) return TINA_OK;
    if (rows > 65535) return fail(TINA_ERR_UNSUPPORTED, "tina_sum: at most 65535 rows");
    // blocks per row: enough to fill the GPU, at least 4096 elements each
    long long gx = ((long long)sm_count() * 8 + rows - 1) / rows;
    const long long need = (n + 4095) / 4096;
    if (gx > need) gx = need;
    if (gx < 1) gx = 1;
    const long long chunk = ((n + gx - 1) / gx + 255) / 256 * 256;
    g_last_path = kPathSimt; note_kernel("sum_kernel");
    if (gx == 1) {
        sum_kernel<<<dim3(1, (unsigned)rows), 256, 0, st>>>(x, n, chunk > 0 ? chunk : 256, nullptr, out);
        count_launch();
        return check_cuda(cudaGetLastError(), "sum_kernel launch");
    }
    double* partial = nullptr;
    cudaError_t e = cudaMallocAsync(reinterpret_cast<void**>(&partial), (size_t)rows * gx * sizeof(double), st);
    if (e != cudaSuccess) return check_cuda(e, "cudaMallocAsync(sum partials)");
    sum_kernel<<<dim3((unsigned)gx, (unsigned)rows), 256, 0, st>>>(x, n, chunk, partial, nullptr);
    sum_final_kernel<<<(unsigned)((rows + 7) / 8), 256, 0, st>>>(partial, (int)gx, out, rows);
    count_launch();
    count_launch();
    e = cudaGetLastError();
    cudaFreeAsync(partial, st);
    return check_cuda(e, "sum_kernel launch");
}

tina_status arith_matmul(const float* x, const float* y, float* z, long long M, long long L, long long N, cudaStream_t st)
{
    if (M == 0 || N == 0) return TINA_OK;
    const long long gy = (M + GM - 1) / GM, gx = (N + GN - 1) / GN;
    if (gy > 65535) return fail(TINA_ERR_UNSUPPORTED, "tina_matmul: M too large");
    matmul_kernel<<<dim3((unsigned)gx, (unsigned)gy), 256, 0, st>>>(x, y, z, M, L, N);
    count_launch();
    g_last_path = kPathSimt; note_kernel("matmul_kernel");
    return check_cuda(cudaGetLastError(), "matmul_kernel launch");
}

}  // namespace tina

// ---- tina_sum_static: Eq. (11) with the per-block partial sums in a file-scope device array instead of a
// cudaMallocAsync temporary, for callers that may not allocate (CUDA graph capture, tight serving loops).
// The array is part of this module's image on every GPU that loads libtina.so and is held until the process exits.
// In host code `g_sum_static_scratch` is a host-side stand-in, not a device address, so it is never passed to a
// kernel: the device address is looked up once per device with cudaGetSymbolAddress, with that device current.
namespace {

constexpr long long kSumStaticRows = TINA_SUM_STATIC_MAX_ROWS;            // documented limit (include/tina.h)
constexpr long long kSumStaticScratch = 2 * TINA_SUM_STATIC_MAX_ROWS;     // doubles: 8192 x 8 bytes = 64 KB
static __device__ __align__(256) double g_sum_static_scratch[kSumStaticScratch];

constexpr int kSumStaticMaxDev = 64;
std::mutex g_sum_static_mu;
double* g_sum_static_ptr[kSumStaticMaxDev] = {};                          // per device, filled on first use

tina_status sum_static_scratch(double** out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return tina::check_cuda(e, "cudaGetDevice");
    if (dev < 0 || dev >= kSumStaticMaxDev) return tina::fail(TINA_ERR_UNSUPPORTED, "tina_sum_static: device ordinal %d >= %d", dev, kSumStaticMaxDev);
    std::lock_guard<std::mutex> lk(g_sum_static_mu);
    if (!g_sum_static_ptr[dev]) {
        double* p = nullptr;
        e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_sum_static_scratch);
        if (e != cudaSuccess || !p) return tina::check_cuda(e != cudaSuccess ? e : cudaErrorInvalidSymbol, "cudaGetSymbolAddress(sum scratch)");
        g_sum_static_ptr[dev] = p;
    }
    *out = g_sum_static_ptr[dev];
    return TINA_OK;
}

}  // namespace

extern "C" tina_status tina_sum_static(const float* x, long long rows, long long n, float* out, void* stream)
{
    using namespace tina;
    if (rows < 0 || n < 0) return fail(TINA_ERR_BAD_SHAPE, "tina_sum_static: negative size");
    if (rows > kSumStaticRows)
        return fail(TINA_ERR_UNSUPPORTED, "tina_sum_static: rows = %lld exceeds the static scratch limit of %lld rows (use tina_sum)",
                    rows, kSumStaticRows);
    if (rows > 0 && (!out || (n > 0 && !x))) return fail(TINA_ERR_NULL_POINTER, "tina_sum_static: null pointer");
    if (rows == 0) return TINA_OK;
    cudaStream_t st = (cudaStream_t)stream;
    // the decomposition of arith_sum (same blocks per row and chunk, hence the same rounding order), except that a
    // single block per row also goes through the scratch: one code path, every partial written before it is read
    long long gx = ((long long)sm_count() * 8 + rows - 1) / rows;
    const long long need = (n + 4095) / 4096;
    if (gx > need) gx = need;
    if (gx < 1) gx = 1;
    if (rows * gx > kSumStaticScratch) gx = kSumStaticScratch / rows;     // >= 2 since rows <= kSumStaticScratch / 2
    const long long chunk = ((n + gx - 1) / gx + 255) / 256 * 256;
    double* partial = nullptr;
    tina_status s = sum_static_scratch(&partial);
    if (s != TINA_OK) return s;
    g_last_path = kPathSimt; note_kernel("sum_kernel<static scratch>");
    sum_kernel<<<dim3((unsigned)gx, (unsigned)rows), 256, 0, st>>>(x, n, chunk > 0 ? chunk : 256, partial, nullptr);
    sum_final_kernel<<<(unsigned)((rows + 7) / 8), 256, 0, st>>>(partial, (int)gx, out, rows);
    count_launch(2);
    return check_cuda(cudaGetLastError(), "sum_kernel launch (static scratch)");
}
