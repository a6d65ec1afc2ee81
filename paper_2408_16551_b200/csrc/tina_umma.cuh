// tina_umma.cuh -- pieces shared by the tcgen05 kernels of libtina (tina_umma.cu: the dense contraction,
// tina_sym.cu: the column-paired dense contraction): tile geometry, warp roles, the barrier block, and the
// FIR producer (register sliding window, Eq. (20)) with its packed-FMA helpers.
#pragma once
#include "tina_common.cuh"
#include "tina_ptx.cuh"

#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>

namespace tina {

using namespace ptx;

constexpr int BM = 128;                  // frames per tile (UMMA M)
constexpr int KC = 64;                   // K elements per pipeline chunk (one 128-byte swizzle row)
constexpr int NSUB = 256;                // columns per MMA instruction / B ring entry
constexpr int NT_MAX = 512;              // accumulator columns per pass (all of TMEM)
constexpr int A_PART_BYTES = BM * KC * 2;        // 16 KB
constexpr int A_RING_BYTES = 128 * 1024;     // 4 slots of hi+lo tiles (8 of hi only)
constexpr int B_ENTRY_BYTES = NSUB * KC * 2;     // 32 KB
constexpr int B_RING_BYTES = 80 * 1024;      // 5 half-tiles of 16 KB with cta_group::2
constexpr int UMMA_THREADS = 512;
// Warp roles.  The SM's issue arbiter favours higher warp ids, so the latency-critical single-thread
// roles (TMA, MMA) sit at the top and the throughput-bound FIR producers at the bottom.
constexpr int PROD_WARP0 = 0, N_PROD_WARPS = 8, FPW = BM / N_PROD_WARPS;   // 16 frames per producer warp
constexpr int EPI_WARP0 = 8;                // 4 warps; warp % 4 selects the TMEM lane quarter
constexpr int TMA_WARP = 12, MMA_WARP = 13, ALLOC_WARP = 14, MMA_WARP2 = 15;
constexpr int UMMA_CG = 2;                  // CTAs per tcgen05 cta_group (2: CTA pair, M = 256 per MMA)
constexpr int KSPLIT_MAX = 1024;            // longest accumulation chain kept in TMEM (K elements)

struct SmemCtl {
    uint64_t a_full[8], a_empty[8];
    uint64_t b_full[8], b_empty[8];
    uint64_t t_full[2], t_empty[2];
    uint32_t tmem_base;
};
constexpr int FIR_PITCH = 132;               // staged row pitch (floats) of the Toeplitz-FIR epilogue (N = 128 columns)
constexpr int EPI_LD = 36;                  // padded row length (floats) of the epilogue transpose tiles
constexpr int EPI_STAGE_BYTES = 4608;        // per epilogue warp: one padded 32 x EPI_LD tile; the TMA path uses 4096-byte tiles at q * 4096
constexpr size_t UMMA_SMEM_BYTES = A_RING_BYTES + B_RING_BYTES + 4 * EPI_STAGE_BYTES + sizeof(SmemCtl);
static_assert(UMMA_SMEM_BYTES <= 232448, "exceeds the 227 KB shared memory opt-in limit");

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_fn();      // cuTensorMapEncodeTiled through the runtime's driver entry point (tina_umma.cu)

// Cached plan (tina_umma.cu): the Fourier matrix as bf16 hi (| lo) parts, K-major, + its TMA tensor map
// (box = 64 contraction elements x min(N, 256) / 2 rows).  sym: the column-paired P x P layout of tina_sym.cu.
struct Plan {
    __nv_bfloat16* tt = nullptr;
    CUtensorMap tmap;
    CUtensorMap tmap32;     // sym plans only: boxes of 32 contraction elements (64-byte rows, SWIZZLE_64B)
};
tina_status get_plan(int P, bool real, bool inverse, int parts, bool fp16, cudaStream_t st, const Plan** out, bool sym = false);

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
__device__ __forceinline__ void sts128(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d)
{
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
__device__ __forceinline__ float2 ldg_f2(const float* p)
{
    return __ldg(reinterpret_cast<const float2*>(p));
}

template <int MT>
struct FirRegs {
    static constexpr int WA = MT > 0 ? MT : 1;
    float2 tap[WA];
    float2 row[WA - 1 + FPW];
};

// Issue every global load of one chunk: MT tap pairs and the FPW + MT - 1 input rows the warp touches.
template <int MT, bool REAL, bool CHECK>
__device__ __forceinline__ void fir_load(FirRegs<MT>& rg, const float* __restrict__ window, int P, int M,
                                         long long K, long long nblk, const float* __restrict__ xc, int c0, long long f0,
                                         long long x_len = 0)
{
    // K here is the distance between consecutive rows (prm.x_row_stride); x_len != 0 (CHECK only): element
    // index row * K + c0 (+1) must stay below x_len, anything beyond reads as zero (overlapping FIR rows)
    constexpr int WA = FirRegs<MT>::WA;
    if (MT > 0) {
        const float* wp = window + (REAL ? c0 : (c0 >> 1));
#pragma unroll
        for (int m = 0; m < WA; ++m) {
            if (m < M) {
                if (REAL) rg.tap[m] = ldg_f2(wp);
                else { const float h = __ldg(wp); rg.tap[m] = make_float2(h, h); }
            } else rg.tap[m] = make_float2(0.f, 0.f);
            wp += P;
        }
    }
    const long long r0 = f0 + M - WA;                 // first row of the window of frame f0
    const float* p = xc + r0 * K;
#pragma unroll
    for (int j = 0; j < WA - 1 + FPW; ++j) {
        if (CHECK) {
            const long long r = r0 + j;
            float2 v = make_float2(0.f, 0.f);
            if (r >= 0 && r < nblk) {
                if (x_len == 0) v = ldg_f2(p);
                else {
                    const long long e = r * K + c0;
                    if (e + 1 < x_len) v = ldg_f2(p);
                    else if (e < x_len) v.x = __ldg(p);
                }
            }
            rg.row[j] = v;
        } else {
            rg.row[j] = ldg_f2(p);
        }
        p += K;
    }
}

// Polyphase MAC of the FPW frames held in registers, split into bf16 hi / lo, swizzled store.
// Frame i uses rows i .. i + WA - 1 (row i + WA - 1 - m pairs with tap m).  Four frames are
// advanced together so that four independent FMA chains are in flight.
template <int MT>
__device__ __forceinline__ void fir_compute_store(const FirRegs<MT>& rg, uint32_t slot, const uint32_t (&swz)[8], bool split,
                                                  uint32_t rslot = 0,   // rslot != 0: also write the sibling CTA's slot
                                                  bool fp16 = false)   // single-pass fp16 operands instead of bf16
{
    constexpr int WA = FirRegs<MT>::WA;
    constexpr int FG = 8;                  // frames advanced together (independent FMA chains in flight)
#pragma unroll
    for (int i0 = 0; i0 < FPW; i0 += FG) {
        float2 y[FG];
        if (MT > 0) {
#pragma unroll
            for (int g = 0; g < FG; ++g) y[g] = fmul2(rg.tap[0], rg.row[i0 + g + WA - 1]);
#pragma unroll
            for (int m = 1; m < WA; ++m)
#pragma unroll
                for (int g = 0; g < FG; ++g) y[g] = ffma2(rg.tap[m], rg.row[i0 + g + WA - 1 - m], y[g]);
        } else {
#pragma unroll
            for (int g = 0; g < FG; ++g) y[g] = rg.row[i0 + g];
        }
#pragma unroll
        for (int g = 0; g < FG; ++g) {
            const int i = i0 + g;
            uint32_t hb;
            if (fp16) { const __half2 hh = __floats2half2_rn(y[g].x, y[g].y); hb = *reinterpret_cast<const uint32_t*>(&hh); }
            else { const __nv_bfloat162 hi = __floats2bfloat162_rn(y[g].x, y[g].y); hb = *reinterpret_cast<const uint32_t*>(&hi); }
            const uint32_t addr = slot + swz[i & 7] + (uint32_t)i * 128u;
            sts32(addr, hb);
            const uint32_t raddr = rslot + swz[i & 7] + (uint32_t)i * 128u;
            if (rslot) sts32_cluster(raddr, hb);
            if (split) {
                const float lx = y[g].x - __uint_as_float(hb << 16);
                const float ly = y[g].y - __uint_as_float(hb & 0xffff0000u);
                const __nv_bfloat162 lo = __floats2bfloat162_rn(lx, ly);
                sts32(addr + A_PART_BYTES, *reinterpret_cast<const uint32_t*>(&lo));
                if (rslot) sts32_cluster(raddr + A_PART_BYTES, *reinterpret_cast<const uint32_t*>(&lo));
            }
        }
    }
}

// tcgen05.commit: arrive on `bar` in this CTA (cta_group::1) or in every CTA of `mask` (::2)
template <int CG>
__device__ __forceinline__ void commit_cg(uint32_t bar, uint16_t mask)
{
    if (CG == 1) umma_commit(bar); else umma_commit_mc(bar, mask);
}
// arrive on a barrier the pair's leader CTA waits on (remote arrive from the peer of a cta_group::2 pair)
template <int CG>
__device__ __forceinline__ void arrive_leader(uint32_t bar, uint32_t rank_in_pair, uint32_t leader)
{
    if (CG == 1 || rank_in_pair == 0) mbar_arrive(bar); else mbar_arrive_cluster(bar, leader);
}

}  // namespace tina
