// tina_ct.cu -- PFB with a FACTORISED Fourier stage on the tensor cores.
//
// The paper allows "either a Discrete or Fast Fourier Transform" after the subfilter stage
// (PAPER.md:233).  tina_pfb keeps the dense P x P contraction the method prescribes (Eq. (12)); this
// file is the two-stage Cooley-Tukey form of the same transform for P = 1024 = 32 x 32 (complex kind):
// with p = a + 32 b and k = kb + 32 ka,
//     G[f][a][kb]  = sum_b y[f][a + 32 b] W32^(b kb)                        (32-point DFTs, stage 1)
//     G'[f][a][kb] = G[f][a][kb] * W1024^(a kb)                             (twiddle)
//     X[f][kb + 32 ka] = sum_a G'[f][a][kb] W32^(a ka)                      (32-point DFTs, stage 2)
// Both stages are 128 x 64 x 64 real-block GEMMs on tcgen05 (bf16 hi / lo operands, ALL FOUR products
// lo*lo, lo*hi, hi*hi, hi*lo, fp32 accumulate in TMEM: two chained stages double the split error of one,
// and an input dominated by one branch -- a window with one huge tap -- does not average it away: measured
// 1.02e-5 with three products; the tensor pipe has slack here) against
// the SAME 64 x 64 matrix, with the subfilter stage (Eq. (20)) as producer of the first A tile and the
// twiddle + transpose done by the first epilogue straight into the second A tile: nothing round-trips
// through HBM, and the tensor work drops from 8 P^2 to 8 P (32 + 32) flops per frame, which makes the
// kernel HBM / FMA bound instead of tensor bound.  One CTA = 8 frames per iteration (two 128-row GEMM tiles); one shared-memory area serves as first and second A operand in turn.
#include "tina_common.cuh"
#include "tina_ptx.cuh"

#include <cuda_bf16.h>
#include <cstdlib>

namespace tina {

using namespace ptx;

constexpr int CT_P = 1024, CT_A = 32, CT_B = 32;      // p = a + CT_A * b
constexpr int CT_FR = 8;                              // frames per group: CT_NT GEMM tiles of 4 frames x 32 rows
constexpr int CT_NT = CT_FR / 4;
constexpr int CT_THREADS = 256;                       // 8 warps; two CTAs per SM overlap each other's phases
constexpr int CT_NW = CT_THREADS / 32;
constexpr int CT_BPW = CT_B / CT_NW;                  // b values (input columns per lane) per warp
constexpr int CT_TILE = 128 * 64 * 2;                 // one bf16 128 x 64 tile: 16 KB
static_assert(CT_NW == 4 * CT_NT, "one warp per (tile, TMEM lane quarter) in the epilogues");

struct CtSmem {
    // per tile hi | lo.  The same area is, in turn, the stage-1 A operand (written by the subfilter stage) and the
    // stage-2 A operand (written by epilogue 1 once the stage-1 MMAs have retired).
    uint8_t a[CT_NT * 2 * CT_TILE];
    uint8_t bm[2 * 64 * 64 * 2];                      // W32 block matrix hi | lo, K-major SWIZZLE_128B (64 rows)
    float2 tw[CT_A * CT_B];                           // W1024^(a kb), [kb][a]
    uint64_t bar[2];
    uint32_t tmem_base;
};

__device__ __forceinline__ uint32_t sw128_off(uint32_t row, uint32_t kbyte)   // byte offset in a K-major SW128 tile
{
    return row * 128u + ((((kbyte >> 4) ^ (row & 7u)) << 4) | (kbyte & 15u));
}

__device__ __forceinline__ void split_store(uint8_t* tile, uint32_t off, float vx, float vy)
{
    const __nv_bfloat162 hi = __floats2bfloat162_rn(vx, vy);
    const uint32_t hb = *reinterpret_cast<const uint32_t*>(&hi);
    const __nv_bfloat162 lo = __floats2bfloat162_rn(vx - __uint_as_float(hb << 16), vy - __uint_as_float(hb & 0xffff0000u));
    *reinterpret_cast<uint32_t*>(tile + off) = hb;
    *reinterpret_cast<uint32_t*>(tile + CT_TILE + off) = *reinterpret_cast<const uint32_t*>(&lo);
}

// (vx, vy) -> packed bf16 pairs: hi = round(v), lo = round(v - hi)
__device__ __forceinline__ void split_pack(float vx, float vy, uint32_t& hb, uint32_t& lb)
{
    const __nv_bfloat162 hi = __floats2bfloat162_rn(vx, vy);
    hb = *reinterpret_cast<const uint32_t*>(&hi);
    const __nv_bfloat162 lo = __floats2bfloat162_rn(vx - __uint_as_float(hb << 16), vy - __uint_as_float(hb & 0xffff0000u));
    lb = *reinterpret_cast<const uint32_t*>(&lo);
}

// d = (a, a) * b + c on a packed fp32 pair (fma.rn.f32x2, SASS FFMA2 with a broadcast scalar operand)
__device__ __forceinline__ float2 ffma2_bc(float a, float2 b, float2 c)
{
    float2 d;
    asm("{\n\t.reg .b64 ra, rb, rc, rd;\n\tmov.b64 ra, {%2, %2};\n\tmov.b64 rb, {%3, %4};\n\tmov.b64 rc, {%5, %6};\n\t"
        "fma.rn.f32x2 rd, ra, rb, rc;\n\tmov.b64 {%0, %1}, rd;\n\t}"
        : "=f"(d.x), "=f"(d.y) : "f"(a), "f"(b.x), "f"(b.y), "f"(c.x), "f"(c.y));
    return d;
}

// streaming load of an input sample: no reuse in L1, which is left to the window taps
__device__ __forceinline__ float2 ldg_stream(const float2* p)
{
    float2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
    return v;
}

template <int MT>
__global__ void __launch_bounds__(CT_THREADS, 2)
pfb_ct_kernel(const float2* __restrict__ x, long long stream_stride, const float* __restrict__ window,
              const __nv_bfloat16* __restrict__ w32, float2* __restrict__ out, long long F, long long NBLK, int M,
              int groups_per_stream, int total_groups)
{
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    CtSmem& sm = *reinterpret_cast<CtSmem*>(smem_raw);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

    // ---- one-time setup: W32 block matrix into the swizzled layout, twiddle table, barriers, TMEM
    for (int e = tid; e < 2 * 64 * 64; e += CT_THREADS) {
        const int part = e / 4096, n = (e % 4096) / 64, c = e % 64;
        *reinterpret_cast<__nv_bfloat16*>(sm.bm + part * 8192 + sw128_off(n, c * 2)) = w32[part * 4096 + n * 64 + c];
    }
    for (int e = tid; e < CT_A * CT_B; e += CT_THREADS) {
        const int kb = e / CT_A, a = e % CT_A;                          // [kb][a]: a lane reads consecutive a
        double sn, cs;
        sincospi(2.0 * (double)((a * kb) % CT_P) / (double)CT_P, &sn, &cs);
        sm.tw[e] = make_float2((float)cs, (float)-sn);
    }
    if (tid == 0) { mbar_init(smem_u32(&sm.bar[0]), 1); mbar_init(smem_u32(&sm.bar[1]), 1); fence_mbar_init(); }
    if (warp == 0) { tmem_alloc<1>(smem_u32(&sm.tmem_base), 256); tmem_relinquish<1>(); }
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = sm.tmem_base;
    const uint32_t idesc = idesc_bf16(128, 64);
    const uint64_t d_ah = smem_desc_sw128(smem_u32(sm.a)), d_al = smem_desc_sw128(smem_u32(sm.a + CT_TILE));
    const uint64_t d_bh = smem_desc_sw128(smem_u32(sm.bm)), d_bl = smem_desc_sw128(smem_u32(sm.bm + 8192));
    constexpr uint64_t TILE_DESC = (uint64_t)(2 * CT_TILE) >> 4;          // descriptor step from one tile to the next

    constexpr int WA = MT;
    const int et = warp >> 2, eq = warp & 3;                              // epilogue role: tile, TMEM lane quarter
    uint8_t* const etile = sm.a + et * 2 * CT_TILE;
    const uint32_t fir_off = lane * 128 + ((warp ^ (lane & 7)) << 4);
    // ---- the window taps of this thread's CT_BPW columns live in TMEM columns 128..255 (its own lane of its warp's lane
    //      quarter; 16 columns per input column, zero beyond M): tensor memory the accumulators leave unused serves as a
    //      per-thread constant store, so the subfilter stage re-reads no taps through L1 / L2.
    const uint32_t tap_addr = tmem + ((uint32_t)((warp & 3) * 32) << 16) + 128 + (warp >> 2) * 64;
#pragma unroll 1
    for (int cb = 0; cb < CT_BPW; ++cb) {
        uint32_t tv[16];
#pragma unroll
        for (int m = 0; m < 16; ++m)
            tv[m] = m < M ? __float_as_uint(__ldg(window + (long long)m * CT_P + lane + CT_A * (CT_BPW * warp + cb))) : 0u;
        tmem_st16(tap_addr + cb * 16, tv);
    }
    tmem_st_wait();
    static_assert(CT_BPW == 4, "one 16-byte swizzle chunk per warp");
    uint32_t it = 0;
    for (int g = blockIdx.x; g < total_groups; g += gridDim.x, ++it) {
        const int s = g / groups_per_stream;
        const long long f0 = (long long)(g % groups_per_stream) * CT_FR;
        const float2* xs = x + (long long)s * stream_stride;
        // ---- subfilter stage, Eq. (20): thread (warp w, lane a) owns p = a + 32 b for b = CT_BPW w .. CT_BPW w + CT_BPW - 1,
        //      one column at a time: WA - 1 + CT_FR rows and WA taps in registers, CT_FR outputs
        //      The shared-memory offset of (row (fl, a), K cell b) is fir_off + constants: b = 4 warp + cb puts the column in
        //      16-byte chunk `warp` of its row, and the 128-byte swizzle XORs the chunk with a & 7.
        const long long r0 = f0 + M - WA;
        const bool interior = r0 >= 0 && r0 + WA - 1 + CT_FR <= NBLK;      // every row of the group exists (uniform)
        const float2* xg = xs + r0 * CT_P + lane + CT_A * CT_BPW * warp;
        uint32_t hprev[CT_FR], lprev[CT_FR];                               // the even column's results wait for the odd one
#pragma unroll
        for (int cb = 0; cb < CT_BPW; ++cb) {
            uint32_t tv[16];
            float2 row[WA - 1 + CT_FR];
            tmem_ld16(tap_addr + cb * 16, tv);
            if (interior) {
#pragma unroll
                for (int j = 0; j < WA - 1 + CT_FR; ++j) row[j] = ldg_stream(xg + cb * CT_A + j * CT_P);
            } else {
#pragma unroll
                for (int j = 0; j < WA - 1 + CT_FR; ++j) {
                    const long long r = r0 + j;
                    row[j] = (r >= 0 && r < NBLK) ? ldg_stream(xg + cb * CT_A + j * CT_P) : make_float2(0.f, 0.f);
                }
            }
            tmem_ld_wait();
#pragma unroll
            for (int fl = 0; fl < CT_FR; ++fl) {
                const float t0 = __uint_as_float(tv[0]);
                float2 y = make_float2(t0 * row[fl + WA - 1].x, t0 * row[fl + WA - 1].y);
#pragma unroll
                for (int m = 1; m < WA; ++m) y = ffma2_bc(__uint_as_float(tv[m]), row[fl + WA - 1 - m], y);
                uint32_t hb, lb;
                split_pack(y.x, y.y, hb, lb);
                if (cb & 1) {                                              // K cells b - 1, b: one 8-byte store per part
                    uint8_t* const dst = sm.a + fir_off + (cb - 1) * 4 + (fl >> 2) * 2 * CT_TILE + (fl & 3) * 32 * 128;
                    *reinterpret_cast<uint2*>(dst) = make_uint2(hprev[fl], hb);
                    *reinterpret_cast<uint2*>(dst + CT_TILE) = make_uint2(lprev[fl], lb);
                } else {
                    hprev[fl] = hb;
                    lprev[fl] = lb;
                }
            }
        }
        fence_proxy_async();
        __syncthreads();
        // ---- stage 1: D1 = A1 * W32  (tile t -> TMEM columns 64 t .. 64 t + 63)
        if (warp == 0 && elect_one()) {
            tc_fence_after();
#pragma unroll
            for (int t = 0; t < CT_NT; ++t) {
#pragma unroll
                for (int k = 0; k < 4; ++k) umma_bf16<1>(tmem + 64 * t, d_al + t * TILE_DESC + 2 * k, d_bl + 2 * k, idesc, k > 0);   // lo x lo
#pragma unroll
                for (int k = 0; k < 4; ++k) umma_bf16<1>(tmem + 64 * t, d_al + t * TILE_DESC + 2 * k, d_bh + 2 * k, idesc, 1);
#pragma unroll
                for (int k = 0; k < 4; ++k) umma_bf16<1>(tmem + 64 * t, d_ah + t * TILE_DESC + 2 * k, d_bh + 2 * k, idesc, 1);
#pragma unroll
                for (int k = 0; k < 4; ++k) umma_bf16<1>(tmem + 64 * t, d_ah + t * TILE_DESC + 2 * k, d_bl + 2 * k, idesc, 1);
            }
            umma_commit(smem_u32(&sm.bar[0]));
        }
        mbar_wait(smem_u32(&sm.bar[0]), it & 1u);
        tc_fence_after();
        // ---- epilogue 1: twiddle, split, transposed write into A2 (over A1: its MMAs have retired): row (fl, kb), K cell a.
        //      Warp (et, eq) reads TMEM lanes 32 eq .. +31 (rows (fl = eq, a = lane)) of tile et.
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            uint32_t v[32];
            tmem_ld32(tmem + ((uint32_t)(eq * 32) << 16) + 64 * et + 32 * h, v);
            tmem_ld_wait();
#pragma unroll
            for (int q = 0; q < 16; ++q) {
                const int kb = 16 * h + q;
                const float gr = __uint_as_float(v[2 * q]), gi = __uint_as_float(v[2 * q + 1]);
                const float2 w = sm.tw[kb * CT_A + lane];
                split_store(etile, sw128_off(eq * 32 + kb, lane * 4), gr * w.x - gi * w.y, gr * w.y + gi * w.x);
            }
        }
        fence_proxy_async();
        tc_fence_before();
        __syncthreads();
        // ---- stage 2: D2 = A2 * W32  (over D1: every warp has read its part)
        if (warp == 0 && elect_one()) {
            tc_fence_after();
#pragma unroll
            for (int t = 0; t < CT_NT; ++t) {
#pragma unroll
                for (int k = 0; k < 4; ++k) umma_bf16<1>(tmem + 64 * t, d_al + t * TILE_DESC + 2 * k, d_bl + 2 * k, idesc, k > 0);   // lo x lo
#pragma unroll
                for (int k = 0; k < 4; ++k) umma_bf16<1>(tmem + 64 * t, d_al + t * TILE_DESC + 2 * k, d_bh + 2 * k, idesc, 1);
#pragma unroll
                for (int k = 0; k < 4; ++k) umma_bf16<1>(tmem + 64 * t, d_ah + t * TILE_DESC + 2 * k, d_bh + 2 * k, idesc, 1);
#pragma unroll
                for (int k = 0; k < 4; ++k) umma_bf16<1>(tmem + 64 * t, d_ah + t * TILE_DESC + 2 * k, d_bl + 2 * k, idesc, 1);
            }
            umma_commit(smem_u32(&sm.bar[1]));
        }
        mbar_wait(smem_u32(&sm.bar[1]), it & 1u);
        tc_fence_after();
        // ---- epilogue 2: row (fl, kb) holds X[f][kb + 32 ka] for all ka: for a fixed ka the 32 lanes of a warp hold 32
        //      consecutive channels, so the accumulators go straight to global memory, 256 contiguous bytes per store.
        {
            const long long f = f0 + et * 4 + eq;
            float2* const orow = out + ((long long)s * F + f) * CT_P + lane;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                uint32_t v[32];
                tmem_ld32(tmem + ((uint32_t)(eq * 32) << 16) + 64 * et + 32 * h, v);
                tmem_ld_wait();
                if (f < F) {
#pragma unroll
                    for (int q = 0; q < 16; ++q)
                        orow[(16 * h + q) * 32] = make_float2(__uint_as_float(v[2 * q]), __uint_as_float(v[2 * q + 1]));
                }
            }
        }
        tc_fence_before();
        // no barrier here: the next group's subfilter stage only writes the A area (its MMAs have retired), and the next
        // MMA into these TMEM columns is issued behind the barrier that ends that stage
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc<1>(tmem, 256);
}

// ---------------------------------------------------------------------------------------------------------------
// Warp-specialised variant: one CTA per SM, 20 warps.  Warps 0-7 (two warpgroups, 144 registers) only run the subfilter
// stage and keep TWO columns of loads in flight; warps 8-15 (80 registers) only run the two epilogues; warp 16 (32
// registers) issues the MMAs.  setmaxnreg moves registers inside the CTA's launch allocation (96 x 640 = 61440), so
// 256 x 144 + 256 x 80 + 128 x 32 must not exceed it.  Two operand slots (2 x 64 KB) and two accumulator slots (2 x 128 TMEM columns) form a ring, so the loads and
// FMAs of group i + 1 overlap the MMAs and epilogues of group i inside the CTA.  Same arithmetic as pfb_ct_kernel.
constexpr int WS_THREADS = 640, WS_PROD = 256, WS_EPI = 256;
constexpr int WS_SLOTS = 2;
constexpr int WS_SLOT_BYTES = CT_NT * 2 * CT_TILE;        // 64 KB

struct WsSmem {
    uint8_t a[WS_SLOTS][WS_SLOT_BYTES];
    uint8_t bm[2 * 64 * 64 * 2];
    float2 tw[CT_A * CT_B];
    uint64_t a1_full[WS_SLOTS], d1_full[WS_SLOTS], a2_full[WS_SLOTS], d2_full[WS_SLOTS], d_free[WS_SLOTS];
    uint32_t tmem_base;
};

template <int R> __device__ __forceinline__ void setmaxnreg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" :: "n"(R)); }
template <int R> __device__ __forceinline__ void setmaxnreg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" :: "n"(R)); }

template <int MT>
__global__ void __maxnreg__(96)
pfb_ctws_kernel(const float2* __restrict__ x, long long stream_stride, const float* __restrict__ window,
                const __nv_bfloat16* __restrict__ w32, float2* __restrict__ out, long long F, long long NBLK, int M,
                int groups_per_stream, int total_groups)
{
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    WsSmem& sm = *reinterpret_cast<WsSmem*>(smem_raw);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

    for (int e = tid; e < 2 * 64 * 64; e += WS_THREADS) {
        const int part = e / 4096, n = (e % 4096) / 64, c = e % 64;
        *reinterpret_cast<__nv_bfloat16*>(sm.bm + part * 8192 + sw128_off(n, c * 2)) = w32[part * 4096 + n * 64 + c];
    }
    for (int e = tid; e < CT_A * CT_B; e += WS_THREADS) {
        const int kb = e / CT_A, a = e % CT_A;
        double sn, cs;
        sincospi(2.0 * (double)((a * kb) % CT_P) / (double)CT_P, &sn, &cs);
        sm.tw[e] = make_float2((float)cs, (float)-sn);
    }
    if (tid == 0) {
        for (int s = 0; s < WS_SLOTS; ++s) {
            mbar_init(smem_u32(&sm.a1_full[s]), WS_PROD);
            mbar_init(smem_u32(&sm.d1_full[s]), 1);
            mbar_init(smem_u32(&sm.a2_full[s]), WS_EPI);
            mbar_init(smem_u32(&sm.d2_full[s]), 1);
            mbar_init(smem_u32(&sm.d_free[s]), WS_EPI);
        }
        fence_mbar_init();
    }
    if (warp == 0) { tmem_alloc<1>(smem_u32(&sm.tmem_base), 512); tmem_relinquish<1>(); }
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = sm.tmem_base;
    const int n_groups = ((int)blockIdx.x < total_groups) ? (total_groups - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
    constexpr int WA = MT, NR = WA - 1 + CT_FR;

    if (warp < 8) {
        // ================================================================== producers: subfilter stage
        setmaxnreg_inc<144>();
        const uint32_t fir_off = lane * 128 + ((warp ^ (lane & 7)) << 4);
        const uint32_t tap_addr = tmem + ((uint32_t)((warp & 3) * 32) << 16) + 256 + (warp >> 2) * 64;
#pragma unroll 1
        for (int cb = 0; cb < CT_BPW; ++cb) {
            uint32_t tv[16];
#pragma unroll
            for (int m = 0; m < 16; ++m)
                tv[m] = m < M ? __float_as_uint(__ldg(window + (long long)m * CT_P + lane + CT_A * (CT_BPW * warp + cb))) : 0u;
            tmem_st16(tap_addr + cb * 16, tv);
        }
        tmem_st_wait();
        auto load_col = [&](int gg, int cb, float2 (&row)[NR]) {
            const long long r0 = (long long)(gg % groups_per_stream) * CT_FR + M - WA;
            const float2* xg = x + (long long)(gg / groups_per_stream) * stream_stride + r0 * CT_P + lane + CT_A * (CT_BPW * warp + cb);
            if (r0 >= 0 && r0 + NR <= NBLK) {
#pragma unroll
                for (int j = 0; j < NR; ++j) row[j] = ldg_stream(xg + j * CT_P);
            } else {
#pragma unroll
                for (int j = 0; j < NR; ++j) row[j] = (r0 + j >= 0 && r0 + j < NBLK) ? ldg_stream(xg + j * CT_P) : make_float2(0.f, 0.f);
            }
        };
        float2 rows[2][NR];
        if (n_groups > 0) load_col(blockIdx.x, 0, rows[0]);
#pragma unroll 1
        for (int i = 0; i < n_groups; ++i) {
            const int g = (int)blockIdx.x + i * (int)gridDim.x, slot = i & 1;
            uint8_t* const abase = sm.a[slot];
            uint32_t hprev[CT_FR], lprev[CT_FR];
#pragma unroll
            for (int cb = 0; cb < CT_BPW; ++cb) {
                uint32_t tv[16];
                tmem_ld16(tap_addr + cb * 16, tv);
                // the next column (or column 0 of the next group) is requested before this one is computed
                if (cb + 1 < CT_BPW) load_col(g, cb + 1, rows[(cb + 1) & 1]);
                else if (i + 1 < n_groups) load_col(g + (int)gridDim.x, 0, rows[0]);
                float2 (&row)[NR] = rows[cb & 1];
                tmem_ld_wait();
                // the slot's previous contents (stage-2 operand of group i - 2) must have been consumed
                if (cb == 1 && i >= WS_SLOTS) mbar_wait(smem_u32(&sm.d2_full[slot]), ((i >> 1) - 1) & 1u);
#pragma unroll
                for (int fl = 0; fl < CT_FR; ++fl) {
                    const float t0 = __uint_as_float(tv[0]);
                    float2 y = make_float2(t0 * row[fl + WA - 1].x, t0 * row[fl + WA - 1].y);
#pragma unroll
                    for (int m = 1; m < WA; ++m) y = ffma2_bc(__uint_as_float(tv[m]), row[fl + WA - 1 - m], y);
                    uint32_t hb, lb;
                    split_pack(y.x, y.y, hb, lb);
                    if (cb & 1) {
                        uint8_t* const dst = abase + fir_off + (cb - 1) * 4 + (fl >> 2) * 2 * CT_TILE + (fl & 3) * 32 * 128;
                        *reinterpret_cast<uint2*>(dst) = make_uint2(hprev[fl], hb);
                        *reinterpret_cast<uint2*>(dst + CT_TILE) = make_uint2(lprev[fl], lb);
                    } else {
                        hprev[fl] = hb;
                        lprev[fl] = lb;
                    }
                }
            }
            fence_proxy_async();
            mbar_arrive(smem_u32(&sm.a1_full[slot]));
        }
    } else if (warp < 16) {
        // ================================================================== epilogue warps
        setmaxnreg_dec<80>();
        const int e = warp - 8, et = e >> 2, eq = e & 3;
        auto epi2 = [&](int i) {
            const int g = (int)blockIdx.x + i * (int)gridDim.x, slot = i & 1;
            const int s = g / groups_per_stream;
            const long long f = (long long)(g % groups_per_stream) * CT_FR + et * 4 + eq;
            mbar_wait(smem_u32(&sm.d2_full[slot]), (i >> 1) & 1u);
            tc_fence_after();
            float2* const orow = out + ((long long)s * F + f) * CT_P + lane;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                uint32_t v[32];
                tmem_ld32(tmem + ((uint32_t)(eq * 32) << 16) + 128 * slot + 64 * et + 32 * h, v);
                tmem_ld_wait();
                if (f < F) {
#pragma unroll
                    for (int q = 0; q < 16; ++q)
                        orow[(16 * h + q) * 32] = make_float2(__uint_as_float(v[2 * q]), __uint_as_float(v[2 * q + 1]));
                }
            }
            tc_fence_before();
            mbar_arrive(smem_u32(&sm.d_free[slot]));
        };
#pragma unroll 1
        for (int i = 0; i < n_groups; ++i) {
            const int slot = i & 1;
            uint8_t* const etile = sm.a[slot] + et * 2 * CT_TILE;
            mbar_wait(smem_u32(&sm.d1_full[slot]), (i >> 1) & 1u);
            tc_fence_after();
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                uint32_t v[32];
                tmem_ld32(tmem + ((uint32_t)(eq * 32) << 16) + 128 * slot + 64 * et + 32 * h, v);
                tmem_ld_wait();
#pragma unroll
                for (int q = 0; q < 16; ++q) {
                    const int kb = 16 * h + q;
                    const float gr = __uint_as_float(v[2 * q]), gi = __uint_as_float(v[2 * q + 1]);
                    const float2 w = sm.tw[kb * CT_A + lane];
                    split_store(etile, sw128_off(eq * 32 + kb, lane * 4), gr * w.x - gi * w.y, gr * w.y + gi * w.x);
                }
            }
            fence_proxy_async();
            tc_fence_before();
            mbar_arrive(smem_u32(&sm.a2_full[slot]));
            if (i >= 1) epi2(i - 1);                    // while the stage-2 MMAs of group i run
        }
        if (n_groups > 0) epi2(n_groups - 1);
    } else {
        // ================================================================== MMA issuer (warp 16; warps 17-19 idle)
        setmaxnreg_dec<32>();
        if (warp == 16 && elect_one()) {
            const uint32_t idesc = idesc_bf16(128, 64);
            const uint64_t d_bh = smem_desc_sw128(smem_u32(sm.bm)), d_bl = smem_desc_sw128(smem_u32(sm.bm + 8192));
            constexpr uint64_t TILE_DESC = (uint64_t)(2 * CT_TILE) >> 4, PART_DESC = (uint64_t)CT_TILE >> 4;
            auto stage = [&](int slot, uint64_t bar) {
                const uint64_t d_ah = smem_desc_sw128(smem_u32(sm.a[slot]));
#pragma unroll
                for (int t = 0; t < CT_NT; ++t) {
                    const uint32_t dcol = tmem + 128 * slot + 64 * t;
                    const uint64_t da = d_ah + t * TILE_DESC;
#pragma unroll
                    for (int k = 0; k < 4; ++k) umma_bf16<1>(dcol, da + PART_DESC + 2 * k, d_bl + 2 * k, idesc, k > 0);   // lo x lo
#pragma unroll
                    for (int k = 0; k < 4; ++k) umma_bf16<1>(dcol, da + PART_DESC + 2 * k, d_bh + 2 * k, idesc, 1);
#pragma unroll
                    for (int k = 0; k < 4; ++k) umma_bf16<1>(dcol, da + 2 * k, d_bh + 2 * k, idesc, 1);
#pragma unroll
                    for (int k = 0; k < 4; ++k) umma_bf16<1>(dcol, da + 2 * k, d_bl + 2 * k, idesc, 1);
                }
                umma_commit((uint32_t)bar);
            };
#pragma unroll 1
            for (int i = 0; i <= n_groups; ++i) {
                if (i < n_groups) {
                    const int slot = i & 1;
                    mbar_wait(smem_u32(&sm.a1_full[slot]), (i >> 1) & 1u);
                    if (i >= WS_SLOTS) mbar_wait(smem_u32(&sm.d_free[slot]), ((i >> 1) - 1) & 1u);   // accumulators drained
                    tc_fence_after();
                    stage(slot, smem_u32(&sm.d1_full[slot]));
                }
                if (i >= 1) {
                    const int slot = (i - 1) & 1;
                    mbar_wait(smem_u32(&sm.a2_full[slot]), ((i - 1) >> 1) & 1u);
                    tc_fence_after();
                    stage(slot, smem_u32(&sm.d2_full[slot]));
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc<1>(tmem, 512);
}

}  // namespace tina

namespace tina {

// defined in tina_umma.cu: the cached bf16 hi | lo block matrix of a P-point complex DFT ([2][2P][2P], row n = output)
const __nv_bfloat16* umma_twiddle_plan(int P, bool real, bool inverse, cudaStream_t st, tina_status* status);

tina_status ct_pfb(const void* x, int S, long long n_samples, int M, const float* window, void* out, cudaStream_t st)
{
    const long long NBLK = n_samples / CT_P, F = NBLK - M + 1;
    tina_status ps = TINA_OK;
    const __nv_bfloat16* w32 = umma_twiddle_plan(32, false, false, st, &ps);
    if (!w32) return ps;
    const long long gps = (F + CT_FR - 1) / CT_FR;
    if (gps * S > 0x7fffffffLL) return fail(TINA_ERR_UNSUPPORTED, "tina_pfb_fft: too many frames");
    DevCtx* ctx = nullptr;
    if ((ps = dev_ctx(&ctx)) != TINA_OK) return ps;
    const int n_sm = ctx->n_sm;
    const int total = (int)(gps * S);
    if (!options().ct_no_ws) {                              // warp-specialised variant: one 640-thread CTA per SM
        const void* kw = M <= 4 ? (const void*)pfb_ctws_kernel<4> : M <= 8 ? (const void*)pfb_ctws_kernel<8> : (const void*)pfb_ctws_kernel<16>;
        if ((ps = ensure_smem(ctx, kw, (int)sizeof(WsSmem) + 1024, "pfb_ctws_kernel setup")) != TINA_OK) return ps;
        const int grid = total < n_sm ? total : n_sm;
        const size_t smem = sizeof(WsSmem) + 1024;
        const float2* xf = static_cast<const float2*>(x);
        float2* of = static_cast<float2*>(out);
        if (M <= 4) pfb_ctws_kernel<4><<<grid, WS_THREADS, smem, st>>>(xf, n_samples, window, w32, of, F, NBLK, M, (int)gps, total);
        else if (M <= 8) pfb_ctws_kernel<8><<<grid, WS_THREADS, smem, st>>>(xf, n_samples, window, w32, of, F, NBLK, M, (int)gps, total);
        else pfb_ctws_kernel<16><<<grid, WS_THREADS, smem, st>>>(xf, n_samples, window, w32, of, F, NBLK, M, (int)gps, total);
        count_launch();
        g_last_path = kPathUmma; note_kernel("pfb_ctws_kernel");
        return check_cuda(cudaGetLastError(), "pfb_ctws_kernel launch");
    }
    {
        const void* kc = M <= 4 ? (const void*)pfb_ct_kernel<4> : M <= 8 ? (const void*)pfb_ct_kernel<8> : (const void*)pfb_ct_kernel<16>;
        if ((ps = ensure_smem(ctx, kc, (int)sizeof(CtSmem) + 1024, "pfb_ct_kernel setup")) != TINA_OK) return ps;
    }
    const int per_sm = 2;                                   // 256 threads, 89 KB shared memory, 128 TMEM columns per CTA
    const int grid = total < n_sm * per_sm ? total : n_sm * per_sm;
    const size_t smem = sizeof(CtSmem) + 1024;
    const float2* xf = static_cast<const float2*>(x);
    float2* of = static_cast<float2*>(out);
    if (M <= 4) pfb_ct_kernel<4><<<grid, CT_THREADS, smem, st>>>(xf, n_samples, window, w32, of, F, NBLK, M, (int)gps, total);
    else if (M <= 8) pfb_ct_kernel<8><<<grid, CT_THREADS, smem, st>>>(xf, n_samples, window, w32, of, F, NBLK, M, (int)gps, total);
    else pfb_ct_kernel<16><<<grid, CT_THREADS, smem, st>>>(xf, n_samples, window, w32, of, F, NBLK, M, (int)gps, total);
    count_launch();
    g_last_path = kPathUmma; note_kernel("pfb_ct_kernel");
    return check_cuda(cudaGetLastError(), "pfb_ct_kernel launch");
}

}  // namespace tina
