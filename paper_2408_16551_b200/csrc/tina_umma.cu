// tina_umma.cu -- the fused PFB / DFT kernel of libtina on the sm_100a tensor cores.
//
// One persistent, warp-specialised kernel computes, per 128-frame tile,
//     y[f][c]   = sum_m w[m][c] * x[f + M-1-m][c]          (Eq. (20); CUDA cores)
//     out[f][n] = sum_c y[f][c] * T[c][n]                   (Eq. (12)-(13); tcgen05)
// where x is viewed as a real [NB][K] matrix (K = 2P interleaved re/im for the complex kind,
// K = P for the real kind), and T is the real block form of the Fourier matrix (N = K columns).
// y is split on the fly into bf16 hi + lo parts and written straight into the swizzled shared
// memory tiles the MMA consumes: the subfiltered signal never touches HBM.  fp32 accuracy
// comes from the error-compensated product  y*T ~= y_lo*T_hi + y_hi*T_hi + y_hi*T_lo  (bf16x3,
// fp32 accumulation in TMEM); TINA_PREC_BF16 issues the single y_hi*T_hi pass.
//
// Warp roles (512 threads, 1 CTA per SM):
//   warp 0      TMA producer: twiddle tiles T_hi / T_lo  -> B ring (4 x 32 KB, SWIZZLE_128B)
//   warp 1      MMA issuer (one elected lane): tcgen05.mma kind::f16, M=128, N<=256, K=16
//   warp 2      TMEM allocator
//   warps 4-7   epilogue: tcgen05.ld (TMEM -> registers) -> global stores
//   warps 8-15  FIR producers: polyphase MAC in fp32 registers -> bf16 hi/lo -> A ring
#include "tina_common.cuh"
#include "tina_ptx.cuh"

#include <cuda.h>
#include <cuda_bf16.h>

#include <map>
#include <mutex>
#include <tuple>

namespace tina {

using namespace ptx;

constexpr int BM = 128;                  // frames per tile (UMMA M)
constexpr int KC = 64;                   // K elements per pipeline chunk (one 128-byte swizzle row)
constexpr int NSUB = 256;                // columns per MMA instruction / B ring entry
constexpr int NT_MAX = 512;              // accumulator columns per pass (all of TMEM)
constexpr int A_PART_BYTES = BM * KC * 2;        // 16 KB
constexpr int A_RING_BYTES = 64 * 1024;
constexpr int B_ENTRY_BYTES = NSUB * KC * 2;     // 32 KB
constexpr int NB_RING = 4;
constexpr int UMMA_THREADS = 512;
constexpr int PROD_WARP0 = 8, N_PROD_WARPS = 8, FPW = BM / N_PROD_WARPS;   // 16 frames per producer warp
constexpr int EPI_WARP0 = 4;
constexpr int KSPLIT_MAX = 1024;            // longest accumulation chain kept in TMEM (K elements)

struct SmemCtl {
    uint64_t a_full[4], a_empty[4];
    uint64_t b_full[NB_RING], b_empty[NB_RING];
    uint64_t t_full[2], t_empty[2];
    uint32_t tmem_base;
};
constexpr size_t UMMA_SMEM_BYTES = 1024 + A_RING_BYTES + NB_RING * B_ENTRY_BYTES + sizeof(SmemCtl);

struct UmmaParams {
    const float* x;            // [S][stream_stride] floats
    const float* window;       // [M][P] or nullptr (M == 1, unit taps)
    float* out;                // [S][F][out_row] floats
    long long stream_stride;   // floats between streams of x
    long long F, NBLK;         // frames per stream, input blocks per stream
    long long out_row;         // floats per output row (complex: 2P, real: P+2)
    int K;                     // floats per input row = GEMM K = GEMM N
    int P, M;
    int tiles_per_stream, n_passes, total_work;
    int parts;                 // 2: bf16x3 (hi+lo), 1: single bf16 pass
    int k_splits, kc_per_split; // accumulation chains per tile
};

// =====================================================================================
// Plan: twiddle matrix Tt[part][n][c] (bf16, "K-major" = row n holds the K contraction index)
// built on the device from float64 sincospi, + its TMA tensor map.
// =====================================================================================
__global__ void twiddle_kernel(__nv_bfloat16* __restrict__ tt, int P, int real, int inverse, int parts)
{
    const int N = real ? P : 2 * P;
    const long long total = (long long)N * N;
    const double scale = inverse ? 1.0 / (double)P : 1.0;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total;
         e += (long long)gridDim.x * blockDim.x) {
        const int n = (int)(e / N), c = (int)(e % N);
        double v;
        if (real) {
            // n = 0: DC, n = 1: Nyquist (packed into the always-zero Im X[0] column),
            // n = 2k: cos, n = 2k+1: -sin  (k >= 1)
            if (n == 0) v = 1.0;
            else if (n == 1) v = (c & 1) ? -1.0 : 1.0;
            else {
                const int k = n >> 1;
                const long long r = ((long long)c * k) % P;
                double sn, cs;
                sincospi(2.0 * (double)r / (double)P, &sn, &cs);
                v = (n & 1) ? -sn : cs;
            }
        } else {
            const int k = n >> 1, j = n & 1, p = c >> 1, i = c & 1;
            const long long r = ((long long)p * k) % P;
            double sn, cs;
            sincospi(2.0 * (double)r / (double)P, &sn, &cs);
            if (inverse) sn = -sn;
            // Xr += yr*cs + yi*sn ; Xi += -yr*sn + yi*cs   (forward, exp(-i theta))
            v = (j == 0) ? (i == 0 ? cs : sn) : (i == 0 ? -sn : cs);
        }
        v *= scale;
        const __nv_bfloat16 hi = __double2bfloat16(v);
        tt[e] = hi;
        if (parts > 1) tt[total + e] = __double2bfloat16(v - (double)__bfloat162float(hi));
    }
}

struct Plan {
    __nv_bfloat16* tt = nullptr;
    CUtensorMap tmap;
};
using PlanKey = std::tuple<int, int, int, int, int>;   // device, P, real, inverse, parts
static std::mutex g_plan_mu;
static std::map<PlanKey, Plan> g_plans;

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn()
{
    static EncodeTiledFn fn = nullptr;
    if (fn) return fn;
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) != cudaSuccess ||
        qres != cudaDriverEntryPointSuccess)
        return nullptr;
    fn = reinterpret_cast<EncodeTiledFn>(p);
    return fn;
}

static tina_status get_plan(int P, bool real, bool inverse, int parts, cudaStream_t st, const Plan** out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return check_cuda(e, "cudaGetDevice");
    std::lock_guard<std::mutex> lk(g_plan_mu);
    const PlanKey key{dev, P, real ? 1 : 0, inverse ? 1 : 0, parts};
    auto it = g_plans.find(key);
    if (it != g_plans.end()) { *out = &it->second; return TINA_OK; }

    const int N = real ? P : 2 * P;
    Plan pl;
    const size_t bytes = (size_t)parts * N * N * sizeof(__nv_bfloat16);
    e = cudaMalloc(&pl.tt, bytes);
    if (e != cudaSuccess) return check_cuda(e, "cudaMalloc(twiddles)");
    twiddle_kernel<<<592, 256, 0, st>>>(pl.tt, P, real ? 1 : 0, inverse ? 1 : 0, parts);
    count_launch();
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { cudaFree(pl.tt); return check_cuda(e, "twiddle_kernel"); }

    EncodeTiledFn enc = encode_fn();
    if (!enc) { cudaFree(pl.tt); return fail(TINA_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found"); }
    const cuuint64_t dims[2] = {(cuuint64_t)N, (cuuint64_t)parts * N};       // innermost (K) first
    const cuuint64_t strides[1] = {(cuuint64_t)N * sizeof(__nv_bfloat16)};
    const cuuint32_t box[2] = {(cuuint32_t)KC, (cuuint32_t)(N < NSUB ? N : NSUB)};
    const cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(&pl.tmap, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, pl.tt, dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                     CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { cudaFree(pl.tt); return fail(TINA_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r); }
    auto ins = g_plans.emplace(key, pl);
    *out = &ins.first->second;
    return TINA_OK;
}

void umma_clear_plans()
{
    std::lock_guard<std::mutex> lk(g_plan_mu);
    for (auto& kv : g_plans) cudaFree(kv.second.tt);
    g_plans.clear();
}

// =====================================================================================
// FIR producer: one warp computes FPW (16) consecutive frames x 64 scalar columns of the
// subfiltered signal (Eq. (20)) and writes them, split into bf16 hi / lo, into an A-ring slot
// in the canonical K-major SWIZZLE_128B layout.  Each lane owns two adjacent scalar columns
// (one complex sample, or two real branches); the last MT input rows live in a rotating
// register window, so every input sample is loaded once per warp and every output costs MT
// packed FMAs (fma.rn.f32x2).  All global loads are issued before the wait on the slot.
// =====================================================================================
struct RingPos {
    uint32_t idx = 0, phase = 0;
    __device__ __forceinline__ void advance(uint32_t n) { if (++idx == n) { idx = 0; phase ^= 1; } }
};

__device__ __forceinline__ float2 ffma2(float2 a, float2 b, float2 c)
{
    float2 d;
    asm("{\n\t.reg .b64 ra, rb, rc, rd;\n\tmov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\tmov.b64 rc, {%6, %7};\n\t"
        "fma.rn.f32x2 rd, ra, rb, rc;\n\tmov.b64 {%0, %1}, rd;\n\t}"
        : "=f"(d.x), "=f"(d.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y), "f"(c.x), "f"(c.y));
    return d;
}
__device__ __forceinline__ float2 fmul2(float2 a, float2 b)
{
    float2 d;
    asm("{\n\t.reg .b64 ra, rb, rd;\n\tmov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\t"
        "mul.rn.f32x2 rd, ra, rb;\n\tmov.b64 {%0, %1}, rd;\n\t}"
        : "=f"(d.x), "=f"(d.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return d;
}
__device__ __forceinline__ void sts32(uint32_t addr, uint32_t v)
{
    asm volatile("st.shared.b32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ float2 ldg_f2(const float* p)
{
    return __ldg(reinterpret_cast<const float2*>(p));
}

template <int MT, bool REAL, bool CHECK>
__device__ __forceinline__ void fir_chunk(const UmmaParams& prm, const float* __restrict__ xc, int c0, long long f0,
                                          uint32_t a_ring_s, uint32_t a_slot_bytes, const uint32_t (&swz)[8],
                                          SmemCtl* ctl, const RingPos& a, bool split)
{
    constexpr int WA = MT > 0 ? MT : 1;
    const int M = prm.M;
    const long long K = prm.K;
    float2 tap[WA], row[WA - 1 + FPW];
    // ---- all global loads first (taps, then the FPW + WA - 1 input rows this warp touches)
    if (MT > 0) {
#pragma unroll
        for (int m = 0; m < WA; ++m) {
            if (m < M) {
                if (REAL) tap[m] = ldg_f2(prm.window + (long long)m * prm.P + c0);
                else { const float h = __ldg(prm.window + (long long)m * prm.P + (c0 >> 1)); tap[m] = make_float2(h, h); }
            } else tap[m] = make_float2(0.f, 0.f);
        }
    }
    {
        const long long r0 = f0 + M - WA;                 // first row of the window of frame f0
        const float* p = xc + r0 * K;
#pragma unroll
        for (int j = 0; j < WA - 1 + FPW; ++j) {
            if (CHECK) {
                const long long r = r0 + j;
                row[j] = (r >= 0 && r < prm.NBLK) ? ldg_f2(p) : make_float2(0.f, 0.f);
            } else {
                row[j] = ldg_f2(p);
            }
            p += K;
        }
    }
    mbar_wait(smem_u32(&ctl->a_empty[a.idx]), a.phase ^ 1);
    const uint32_t slot = a_ring_s + a.idx * a_slot_bytes;
    // ---- frame i uses rows i .. i + WA - 1 (row i + WA - 1 - m pairs with tap m)
#pragma unroll
    for (int i = 0; i < FPW; ++i) {
        float2 y;
        if (MT > 0) {
            y = fmul2(tap[0], row[i + WA - 1]);
#pragma unroll
            for (int m = 1; m < WA; ++m) y = ffma2(tap[m], row[i + WA - 1 - m], y);
        } else {
            y = row[i];
        }
        const __nv_bfloat162 hi = __floats2bfloat162_rn(y.x, y.y);
        const uint32_t hb = *reinterpret_cast<const uint32_t*>(&hi);
        const uint32_t addr = slot + swz[i & 7] + (uint32_t)i * 128u;
        sts32(addr, hb);
        if (split) {
            const float lx = y.x - __uint_as_float(hb << 16);
            const float ly = y.y - __uint_as_float(hb & 0xffff0000u);
            const __nv_bfloat162 lo = __floats2bfloat162_rn(lx, ly);
            sts32(addr + A_PART_BYTES, *reinterpret_cast<const uint32_t*>(&lo));
        }
    }
    fence_proxy_async();
}

// =====================================================================================
// The fused kernel.  MT = compile-time tap count the sliding window is unrolled for
// (taps m >= M are zero; MT == 0: no window, y = x, i.e. a plain DFT batch).
// =====================================================================================
template <int MT, bool REAL>
__global__ void __launch_bounds__(UMMA_THREADS, 1)
pfb_umma_kernel(const __grid_constant__ CUtensorMap tmap_b, const UmmaParams prm)
{
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    uint8_t* a_ring = smem;
    uint8_t* b_ring = smem + A_RING_BYTES;
    SmemCtl* ctl = reinterpret_cast<SmemCtl*>(b_ring + NB_RING * B_ENTRY_BYTES);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int parts = prm.parts;
    const uint32_t a_slot_bytes = A_PART_BYTES * parts;
    const uint32_t n_a = A_RING_BYTES / a_slot_bytes;            // 2 (bf16x3) or 4 (single pass)
    const int N = prm.K;
    const int n_kc = prm.K / KC;
    const int nt_max = N < NT_MAX ? N : NT_MAX;
    const uint32_t n_acc = nt_max <= 256 ? 2 : 1;                 // TMEM accumulator stages
    const uint32_t b_box_bytes = (uint32_t)(N < NSUB ? N : NSUB) * KC * 2;

    if (warp == 0 && lane == 0) {
        prefetch_tmap(&tmap_b);
        for (int i = 0; i < 4; ++i) { mbar_init(smem_u32(&ctl->a_full[i]), N_PROD_WARPS); mbar_init(smem_u32(&ctl->a_empty[i]), 1); }
        for (int i = 0; i < NB_RING; ++i) { mbar_init(smem_u32(&ctl->b_full[i]), 1); mbar_init(smem_u32(&ctl->b_empty[i]), 1); }
        for (int i = 0; i < 2; ++i) { mbar_init(smem_u32(&ctl->t_full[i]), 1); mbar_init(smem_u32(&ctl->t_empty[i]), 4); }
        fence_mbar_init();
    }
    if (warp == 2) {
        tmem_alloc<1>(smem_u32(&ctl->tmem_base), 512);
        tmem_relinquish<1>();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = ctl->tmem_base;

    if (warp == 0) {
        // ============================ TMA producer: twiddle tiles ============================
        if (lane == 0) {
            RingPos b;
            for (int w = blockIdx.x; w < prm.total_work; w += gridDim.x) {
                const int n0 = (w % prm.n_passes) * NT_MAX;
                const int nt = min(NT_MAX, N - n0);
                const int n_sub = (nt + NSUB - 1) / NSUB;
                for (int kc = 0; kc < n_kc; ++kc)
                    for (int nh = 0; nh < n_sub; ++nh)
                        for (int part = 0; part < parts; ++part) {
                            mbar_wait(smem_u32(&ctl->b_empty[b.idx]), b.phase ^ 1);
                            const uint32_t bar = smem_u32(&ctl->b_full[b.idx]);
                            mbar_expect_tx(bar, b_box_bytes);
                            tma_load_2d(smem_u32(b_ring + b.idx * B_ENTRY_BYTES), &tmap_b, bar,
                                        kc * KC, part * N + n0 + nh * NSUB);
                            b.advance(NB_RING);
                        }
            }
        }
    } else if (warp == 1) {
        // ============================ MMA issuer ============================================
        RingPos a, b, t;
        for (int w = blockIdx.x; w < prm.total_work; w += gridDim.x) {
            const int n0 = (w % prm.n_passes) * NT_MAX;
            const int nt = min(NT_MAX, N - n0);
            const int n_sub = (nt + NSUB - 1) / NSUB;
            for (int ks = 0; ks < prm.k_splits; ++ks) {
            mbar_wait(smem_u32(&ctl->t_empty[t.idx]), t.phase ^ 1);
            tc_fence_after();
            const uint32_t d_base = tmem_base + t.idx * 256;
            const int kc_begin = ks * prm.kc_per_split, kc_end = min(n_kc, kc_begin + prm.kc_per_split);
            for (int kc = kc_begin; kc < kc_end; ++kc) {
                mbar_wait(smem_u32(&ctl->a_full[a.idx]), a.phase);
                tc_fence_after();
                const uint32_t a_hi = smem_u32(a_ring + a.idx * a_slot_bytes);
                const uint32_t a_lo = a_hi + A_PART_BYTES;
                for (int nh = 0; nh < n_sub; ++nh) {
                    const int nw = min(NSUB, nt - nh * NSUB);
                    const uint32_t idesc = idesc_bf16(BM, nw);
                    const uint32_t d = d_base + nh * NSUB;
                    // ---- B_hi: (A_lo x B_hi) then (A_hi x B_hi)
                    mbar_wait(smem_u32(&ctl->b_full[b.idx]), b.phase);
                    tc_fence_after();
                    if (lane == 0) {
                        const uint64_t bd = smem_desc_sw128(smem_u32(b_ring + b.idx * B_ENTRY_BYTES));
                        uint32_t acc = kc > kc_begin;
                        if (parts > 1) {
                            const uint64_t ad = smem_desc_sw128(a_lo);
#pragma unroll
                            for (int k = 0; k < KC / 16; ++k) { umma_bf16<1>(d, ad + 2 * k, bd + 2 * k, idesc, acc); acc = 1; }
                        }
                        const uint64_t ad = smem_desc_sw128(a_hi);
#pragma unroll
                        for (int k = 0; k < KC / 16; ++k) { umma_bf16<1>(d, ad + 2 * k, bd + 2 * k, idesc, acc); acc = 1; }
                        umma_commit(smem_u32(&ctl->b_empty[b.idx]));
                    }
                    __syncwarp();
                    b.advance(NB_RING);
                    // ---- B_lo: (A_hi x B_lo)
                    if (parts > 1) {
                        mbar_wait(smem_u32(&ctl->b_full[b.idx]), b.phase);
                        tc_fence_after();
                        if (lane == 0) {
                            const uint64_t bd = smem_desc_sw128(smem_u32(b_ring + b.idx * B_ENTRY_BYTES));
                            const uint64_t ad = smem_desc_sw128(a_hi);
#pragma unroll
                            for (int k = 0; k < KC / 16; ++k) umma_bf16<1>(d, ad + 2 * k, bd + 2 * k, idesc, 1);
                            umma_commit(smem_u32(&ctl->b_empty[b.idx]));
                        }
                        __syncwarp();
                        b.advance(NB_RING);
                    }
                }
                if (lane == 0) {
                    umma_commit(smem_u32(&ctl->a_empty[a.idx]));
                    if (kc == kc_end - 1) umma_commit(smem_u32(&ctl->t_full[t.idx]));
                }
                __syncwarp();
                a.advance(n_a);
            }
            t.advance(n_acc);
            }
        }
    } else if (warp >= EPI_WARP0 && warp < EPI_WARP0 + 4) {
        // ============================ epilogue: TMEM -> global ==============================
        const int q = warp - EPI_WARP0;
        RingPos t;
        for (int w = blockIdx.x; w < prm.total_work; w += gridDim.x) {
            const int tile = w / prm.n_passes;
            const int n0 = (w % prm.n_passes) * NT_MAX;
            const int nt = min(NT_MAX, N - n0);
            const int s = tile / prm.tiles_per_stream;
            const long long row = (long long)(tile % prm.tiles_per_stream) * BM + q * 32 + lane;
            const bool valid = row < prm.F;
            float* orow = prm.out + ((long long)s * prm.F + row) * prm.out_row;
            for (int ks = 0; ks < prm.k_splits; ++ks) {
                mbar_wait(smem_u32(&ctl->t_full[t.idx]), t.phase);
                tc_fence_after();
                const uint32_t taddr = tmem_base + t.idx * 256 + ((uint32_t)(q * 32) << 16);
                for (int cb = 0; cb < nt; cb += 32) {
                    uint32_t r[32];
                    tmem_ld32(taddr + cb, r);
                    tmem_ld_wait();
                    if (valid) {
                        const int n = n0 + cb;
                        float4* o4 = reinterpret_cast<float4*>(orow + n);     // complex rows are 16-byte aligned
                        float2* o2 = reinterpret_cast<float2*>(orow + n);     // real rows only 8-byte aligned
                        if (ks > 0) {
                            // later accumulation chains: out += chain (fp32 round-to-nearest add)
                            if (REAL) {
#pragma unroll
                                for (int j = 0; j < 16; ++j) {
                                    const float2 o = o2[j];
                                    r[2 * j] = __float_as_uint(o.x + __uint_as_float(r[2 * j]));
                                    r[2 * j + 1] = __float_as_uint(o.y + __uint_as_float(r[2 * j + 1]));
                                }
                            } else {
#pragma unroll
                                for (int j = 0; j < 8; ++j) {
                                    const float4 o = o4[j];
                                    r[4 * j] = __float_as_uint(o.x + __uint_as_float(r[4 * j]));
                                    r[4 * j + 1] = __float_as_uint(o.y + __uint_as_float(r[4 * j + 1]));
                                    r[4 * j + 2] = __float_as_uint(o.z + __uint_as_float(r[4 * j + 2]));
                                    r[4 * j + 3] = __float_as_uint(o.w + __uint_as_float(r[4 * j + 3]));
                                }
                            }
                        }
                        if (REAL) {
                            if (n == 0) {
                                // columns 0 / 1 carry Re X[0] and Re X[P/2]; both bins are purely real
                                float2* ny = reinterpret_cast<float2*>(orow + prm.P);
                                float nyq = __uint_as_float(r[1]);
                                if (ks > 0) nyq += ny->x;                     // out[1] == 0 was added above: r[1] is still the chain value
                                *ny = make_float2(nyq, 0.f);
                                r[1] = 0u;
                            }
#pragma unroll
                            for (int j = 0; j < 16; ++j)
                                o2[j] = make_float2(__uint_as_float(r[2 * j]), __uint_as_float(r[2 * j + 1]));
                        } else {
#pragma unroll
                            for (int j = 0; j < 8; ++j)
                                o4[j] = make_float4(__uint_as_float(r[4 * j]), __uint_as_float(r[4 * j + 1]),
                                                    __uint_as_float(r[4 * j + 2]), __uint_as_float(r[4 * j + 3]));
                        }
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&ctl->t_empty[t.idx]));
                t.advance(n_acc);
            }
        }
    } else if (warp >= PROD_WARP0) {
        // ============================ FIR producers =========================================
        const int pw = warp - PROD_WARP0;
        const uint32_t a_ring_s = smem_u32(a_ring);
        // byte offset of this lane's 4-byte cell in row 0 of an A tile, for each swizzle phase (row & 7):
        // row r, 16-byte chunk (lane >> 2) is stored at chunk position (lane >> 2) ^ (r & 7)
        uint32_t swz[8];
#pragma unroll
        for (int j = 0; j < 8; ++j)
            swz[j] = (uint32_t)(pw * FPW) * 128u + ((((uint32_t)lane >> 2) ^ (uint32_t)j) << 4) + ((uint32_t)lane & 3u) * 4u;
        RingPos a;
        for (int w = blockIdx.x; w < prm.total_work; w += gridDim.x) {
            const int tile = w / prm.n_passes;
            const int s = tile / prm.tiles_per_stream;
            const long long f0 = (long long)(tile % prm.tiles_per_stream) * BM + pw * FPW;
            const float* xs = prm.x + (long long)s * prm.stream_stride + 2 * lane;
            // rows f0 + M - WA .. f0 + FPW + M - 2 are touched; interior tiles need no bounds checks
            constexpr int WA = MT > 0 ? MT : 1;
            const bool interior = (f0 + prm.M - WA >= 0) && (f0 + FPW + prm.M - 1 <= prm.NBLK);
            for (int kc = 0; kc < n_kc; ++kc) {
                if (interior)
                    fir_chunk<MT, REAL, false>(prm, xs + kc * KC, kc * KC + 2 * lane, f0, a_ring_s, a_slot_bytes, swz,
                                               ctl, a, parts > 1);
                else
                    fir_chunk<MT, REAL, true>(prm, xs + kc * KC, kc * KC + 2 * lane, f0, a_ring_s, a_slot_bytes, swz,
                                              ctl, a, parts > 1);
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&ctl->a_full[a.idx]));
                a.advance(n_a);
            }
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 2) tmem_dealloc<1>(tmem_base, 512);
}

// =====================================================================================
// Host side
// =====================================================================================
bool umma_supported(int P, bool real)
{
    if (P < 32 || P > kMaxP) return false;
    return real ? (P % 64 == 0) : (P % 32 == 0);
}

template <int MT, bool REAL>
static tina_status launch_umma(const CUtensorMap& tmap, const UmmaParams& prm, int grid, cudaStream_t st)
{
    static bool attr_done = false;
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(pfb_umma_kernel<MT, REAL>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)UMMA_SMEM_BYTES);
        if (e != cudaSuccess) return check_cuda(e, "cudaFuncSetAttribute(pfb_umma_kernel)");
        attr_done = true;
    }
    pfb_umma_kernel<MT, REAL><<<grid, UMMA_THREADS, UMMA_SMEM_BYTES, st>>>(tmap, prm);
    count_launch();
    g_last_path = kPathUmma;
    return check_cuda(cudaGetLastError(), "pfb_umma_kernel launch");
}

tina_status umma_pfb(const void* x, int S, long long n_samples, int P, int M, const float* window,
                     bool real, bool inverse, tina_precision prec, void* out, cudaStream_t st)
{
    const int K = real ? P : 2 * P;
    const long long NBLK = n_samples / P;
    const long long F = NBLK - M + 1;
    const int parts = prec == TINA_PREC_BF16 ? 1 : 2;

    if (window && M > 16) {
        // Rare shape: more taps than the register window is unrolled for.  Run the subfilter
        // stage on its own into a stream-ordered temporary, then the contraction as a DFT batch.
        float* y = nullptr;
        const size_t bytes = (size_t)S * F * K * sizeof(float);
        cudaError_t e = cudaMallocAsync(reinterpret_cast<void**>(&y), bytes, st);
        if (e != cudaSuccess) return check_cuda(e, "cudaMallocAsync(subfiltered)");
        tina_status s1 = simt_pfb_fir(x, S, n_samples, P, M, window, real, y, st);
        if (s1 == TINA_OK) s1 = umma_pfb(y, 1, (long long)S * F * P, P, 1, nullptr, real, inverse, prec, out, st);
        cudaFreeAsync(y, st);
        return s1;
    }

    const Plan* plan = nullptr;
    tina_status ps = get_plan(P, real, inverse, parts, st, &plan);
    if (ps != TINA_OK) return ps;

    UmmaParams prm;
    prm.x = static_cast<const float*>(x);
    prm.window = window;
    prm.out = static_cast<float*>(out);
    prm.stream_stride = real ? n_samples : 2 * n_samples;
    prm.F = F;
    prm.NBLK = NBLK;
    prm.out_row = real ? P + 2 : 2 * P;
    prm.K = K;
    prm.P = P;
    prm.M = M;
    prm.tiles_per_stream = (int)((F + BM - 1) / BM);
    prm.n_passes = (K + NT_MAX - 1) / NT_MAX;
    const long long total = (long long)S * prm.tiles_per_stream * prm.n_passes;
    if (total > 0x7fffffffLL) return fail(TINA_ERR_UNSUPPORTED, "tina_pfb: too many tiles");
    prm.total_work = (int)total;
    prm.parts = parts;
    prm.k_splits = (K + KSPLIT_MAX - 1) / KSPLIT_MAX;
    prm.kc_per_split = ((K / KC) + prm.k_splits - 1) / prm.k_splits;

    static int n_sm = 0;
    if (!n_sm) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaError_t e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess || n_sm < 1) { n_sm = 0; return check_cuda(e, "cudaDeviceGetAttribute(SM count)"); }
    }
    const int grid = prm.total_work < n_sm ? prm.total_work : n_sm;

#define TINA_LAUNCH(MT_)                                                                           \
    (real ? launch_umma<MT_, true>(plan->tmap, prm, grid, st) : launch_umma<MT_, false>(plan->tmap, prm, grid, st))
    if (!window) return TINA_LAUNCH(0);
    if (M <= 4) return TINA_LAUNCH(4);
    if (M <= 8) return TINA_LAUNCH(8);
    return TINA_LAUNCH(16);
#undef TINA_LAUNCH
}

}  // namespace tina
