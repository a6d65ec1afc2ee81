// tina_peaks.cu -- measured arithmetic ceilings of the box, for the rooflines bench.py reports
// ("the builder must measure both [TF32, fp32 FMA] with a micro-benchmark on
// the box and commit the numbers").  Four bare loops, no memory traffic in the timed part:
//   TINA_PEAK_FFMA   fp32 fma.rn.f32          (CUDA cores, 8 independent chains per thread)
//   TINA_PEAK_FFMA2  packed fma.rn.f32x2      (the instruction the subfilter stage uses)
//   TINA_PEAK_TF32   tcgen05.mma kind::tf32   (M = 128, N = 256, K = 8 per instruction, operands in smem)
//   TINA_PEAK_BF16   tcgen05.mma kind::f16    (bf16, M = 128, N = 256, K = 16) -- cross-check of the
//                                              driver's cuBLAS figure in MEASURED_PEAKS.json
//   4 / 5            the same bf16 loop with N = 128 / N = 64 columns per instruction (how the tensor rate
//                    falls with narrow tiles: the Toeplitz FIR uses N = 128)
// Operands are pseudo-random (not zeros): the tensor-pipe power draw, and with it the clock the part
// sustains, depends on the data toggling.
#include "tina_common.cuh"
#include "tina_ptx.cuh"

namespace tina {

using namespace ptx;

template <bool PACKED>
__global__ void __launch_bounds__(512)
peak_fma_kernel(float* sink, int iters, float seed)
{
    float a[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) a[i] = seed + (float)(threadIdx.x + i) * 1e-3f;
    const float m = 0.999f, c = 1e-3f;
    for (int it = 0; it < iters; ++it) {
        if (PACKED) {
#pragma unroll
            for (int i = 0; i < 16; i += 2)
                asm volatile("{\n\t.reg .b64 ra, rm, rc;\n\tmov.b64 ra, {%0, %1};\n\tmov.b64 rm, {%2, %2};\n\tmov.b64 rc, {%3, %3};\n\t"
                             "fma.rn.f32x2 ra, ra, rm, rc;\n\tmov.b64 {%0, %1}, ra;\n\t}"
                             : "+f"(a[i]), "+f"(a[i + 1]) : "f"(m), "f"(c));
        } else {
#pragma unroll
            for (int i = 0; i < 16; ++i) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a[i]) : "f"(m), "f"(c));
        }
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += a[i];
    if (s == 123.456f) sink[0] = s;          // never true: keeps the chains live
}

// One CTA per SM: thread 0 issues `iters` groups of four K-steps alternately into the two 256-column halves
// of TMEM; a commit + wait every 8 groups bounds the queue.  A: 128 rows x 128 bytes, B: 256 rows x 128 bytes,
// both K-major SWIZZLE_128B tiles (32 bytes of K per instruction for either kind).
__device__ __forceinline__ void umma_tf32_cg1(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}

template <bool TF32>
__global__ void __launch_bounds__(128, 1)
peak_umma_kernel(int iters, int n_cols)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    uint8_t* a_tile = smem;                         // 16 KB
    uint8_t* b_tile = smem + 16384;                 // 32 KB
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem + 49152);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + 49152 + 64);
    // pseudo-random operand bits with small magnitudes (exponent fixed around 1.0 for either format)
    uint32_t* w = reinterpret_cast<uint32_t*>(smem);
    for (int i = threadIdx.x; i < 49152 / 4; i += blockDim.x) {
        uint32_t h = (uint32_t)i * 2654435761u + blockIdx.x * 40503u;
        h ^= h >> 15; h *= 2246822519u; h ^= h >> 13;
        w[i] = TF32 ? (0x3f800000u | (h & 0x007fe000u) | (h & 0x80000000u))
                    : (0x3f803f80u | (h & 0x007f007fu) | (h & 0x80008000u));
    }
    if (threadIdx.x == 0) { mbar_init(smem_u32(bar), 1); fence_mbar_init(); }
    fence_proxy_async();
    if (threadIdx.x < 32) { tmem_alloc<1>(smem_u32(tmem_slot), 512); tmem_relinquish<1>(); }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    // one ELECTED thread issues (under `threadIdx.x == 0` ptxas wraps every tcgen05.mma in an any-thread loop, and the
    // narrow-tile figures then measure the issuing thread instead of the tensor pipe)
    if (threadIdx.x < 32 && elect_one()) {
        const uint64_t ad = smem_desc_sw128(smem_u32(a_tile)), bd = smem_desc_sw128(smem_u32(b_tile));
        // kind::tf32: a/b format 2; kind::f16 with bf16: format 1; fp32 accumulate; M = 128, N = 256
        const uint32_t fmt = TF32 ? 2u : 1u;
        const uint32_t idesc = (1u << 4) | (fmt << 7) | (fmt << 10) | (((uint32_t)n_cols >> 3) << 17) | ((128u >> 4) << 24);
        uint32_t phase = 0;
        for (int it = 0; it < iters; ++it) {
            const uint32_t d = tmem + (uint32_t)(it & 1) * 256u;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                if (TF32) umma_tf32_cg1(d, ad + 2 * k, bd + 2 * k, idesc, (it > 1 || k > 0) ? 1u : 0u);
                else umma_bf16<1>(d, ad + 2 * k, bd + 2 * k, idesc, (it > 1 || k > 0) ? 1u : 0u);
            }
            if ((it & 7) == 7 || it == iters - 1) {
                umma_commit(smem_u32(bar));
                mbar_wait(smem_u32(bar), phase);
                phase ^= 1;
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (threadIdx.x < 32) tmem_dealloc<1>(tmem, 512);
}

tina_status probe_peak(int which, int iters, double* tflops, double* ms_out, cudaStream_t st)
{
    DevCtx* ctx = nullptr;
    tina_status cs = dev_ctx(&ctx);
    if (cs != TINA_OK) return cs;
    cudaEvent_t e0, e1;
    cudaError_t e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    if (e != cudaSuccess) return check_cuda(e, "cudaEventCreate");
    double flops = 0;
    float* sink = nullptr;
    auto launch = [&](int n) -> cudaError_t {
        if (which == 0 || which == 1) {
            const int blocks = ctx->n_sm * 4;
            if (which == 0) peak_fma_kernel<false><<<blocks, 512, 0, st>>>(sink, n, 1.f);
            else            peak_fma_kernel<true><<<blocks, 512, 0, st>>>(sink, n, 1.f);
            flops = (double)blocks * 512 * (double)n * 16 * 2;
        } else {
            const int smem = 49152 + 128;
            const int ncols = which == 4 ? 128 : (which == 5 ? 64 : 256);
            if (which == 2) peak_umma_kernel<true><<<ctx->n_sm, 128, smem, st>>>(n, ncols);
            else            peak_umma_kernel<false><<<ctx->n_sm, 128, smem, st>>>(n, ncols);
            flops = (double)ctx->n_sm * (double)n * 4 * 2.0 * 128 * ncols * (which == 2 ? 8 : 16);
        }
        count_launch();
        return cudaGetLastError();
    };
    if (which >= 2) {
        const void* k = which == 2 ? (const void*)peak_umma_kernel<true> : (const void*)peak_umma_kernel<false>;
        if ((cs = ensure_smem(ctx, k, 49152 + 128, "peak_umma_kernel setup")) != TINA_OK) return cs;
    } else {
        e = cudaMalloc(&sink, 4);
        if (e != cudaSuccess) return check_cuda(e, "cudaMalloc(sink)");
    }
    e = launch(iters > 64 ? 64 : iters);                     // warm-up
    if (e == cudaSuccess) e = cudaEventRecord(e0, st);
    if (e == cudaSuccess) e = launch(iters);
    if (e == cudaSuccess) e = cudaEventRecord(e1, st);
    if (e == cudaSuccess) e = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    if (sink) cudaFree(sink);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (e != cudaSuccess) return check_cuda(e, "tina_probe_peak");
    *tflops = flops / (ms * 1e-3) / 1e12;
    if (ms_out) *ms_out = ms;
    return TINA_OK;
}

}  // namespace tina
