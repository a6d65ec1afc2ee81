// tina_ctr.cu -- PFB with a FACTORISED Fourier stage for the REAL kind at P = 4096 = 64 x 64 (BASELINE config 5;
// SURVEY.md section 8(f) rank 2, "either a Discrete or Fast Fourier Transform").
//
// With p = a + 64 b and k = kb + 64 ka, for real y:
//     G[f][a][kb]  = sum_b y[f][a + 64 b] W64^(b kb)                        (64-point DFTs of real data, stage 1)
//     G'[f][a][kb] = G[f][a][kb] * W4096^(a kb)                             (twiddle)
//     X[f][kb + 64 ka] = sum_a G'[f][a][kb] W64^(a ka),  k = 0 .. 2048      (stage 2; ka = 0 .. 31, plus k = 2048)
// Both stages contract against ONE 128 x 64 matrix B1[(kb, c)][b] = (cos, -sin)(2 pi b kb / 64) held in shared memory
// (bf16 hi | lo, bf16x3 products, fp32 accumulation in TMEM):
//   stage 1 is computed TRANSPOSED, D1^T[(kb, c)][(frame, a)] = B1 * A1^T, so that an epilogue thread (one TMEM lane =
//     one (kb, re | im)) sees consecutive a in consecutive columns: after one shuffle with its partner lane it owns the
//     real OR the imaginary part of G' for 64 consecutive a, which it packs eight to a 16-byte store into the stage-2
//     operand (rows (frame, kb), K = a), real parts and imaginary parts in two separate tiles;
//   stage 2 runs the two tiles against the first 64 rows of B1 (ka = 0 .. 31):  D_R = Re(G') B1^T = (C_r, -S_r),
//     D_I = Im(G') B1^T = (C_i, -S_i), and X = (D_R.re - D_I.im, D_R.im + D_I.re);
//   X[2048] = sum_a (-1)^a G[a][0] is a thread-local alternating sum in the first epilogue.
// One CTA per SM (193 KB of shared memory), 512 threads, 4 frames (two 128-row tiles) per iteration; the window taps
// live in the upper 256 TMEM columns (tcgen05.st once, tcgen05.ld per column), so they cost no L1 / L2 traffic.
#include "tina_common.cuh"
#include "tina_ptx.cuh"

#include <cuda_bf16.h>
#include <cstdlib>

namespace tina {

using namespace ptx;

constexpr int CR_P = 4096, CR_NK = CR_P / 2 + 1;
constexpr int CR_FR = 4;                              // frames per group: 2 tiles x 2 frames x 64 rows
constexpr int CR_THREADS = 512;
constexpr int CR_BPW = 4;                             // b values per warp in the subfilter stage (16 warps x 4 = 64)
constexpr int CR_TILE = 128 * 64 * 2;                 // one bf16 128 x 64 tile: 16 KB
constexpr int CR_TWP = 66;                            // twiddle table row pitch in float2 (64 + 2: conflict-free 16-byte reads)

struct CrSmem {
    // [tile][block: real | imaginary parts of G'][hi | lo].  The stage-1 operand of tile t (rows (frame, a), K = b)
    // occupies a[t][0] until its MMAs have retired; epilogue 1 then overwrites it.
    uint8_t a[2][2][2][CR_TILE];
    uint8_t bm[2][CR_TILE];                           // B1 hi | lo: row n = 2 kb + c, K = b, K-major SWIZZLE_128B
    float2 tw[64 * CR_TWP];                           // W4096^(a kb), [kb][a]
    float nyq[2][2][2];                               // [tile][frame][column half]: partial Nyquist sums
    uint64_t bar[4];                                  // stage 1 of tile 0 / 1, stage 2 of tile 0 / 1
    uint32_t tmem_base;
};
static_assert(sizeof(CrSmem) + 1024 <= 227 * 1024, "shared memory budget");

__device__ __forceinline__ uint32_t cr_sw128(uint32_t row, uint32_t kbyte)    // byte offset in a K-major SW128 tile
{
    return row * 128u + ((((kbyte >> 4) ^ (row & 7u)) << 4) | (kbyte & 15u));
}

// packed fp32 pair d = a * b + c (fma.rn.f32x2)
__device__ __forceinline__ float2 cr_ffma2(float2 a, float2 b, float2 c)
{
    float2 d;
    asm("{\n\t.reg .b64 ra, rb, rc, rd;\n\tmov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\tmov.b64 rc, {%6, %7};\n\t"
        "fma.rn.f32x2 rd, ra, rb, rc;\n\tmov.b64 {%0, %1}, rd;\n\t}"
        : "=f"(d.x), "=f"(d.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y), "f"(c.x), "f"(c.y));
    return d;
}

// (vx, vy) -> packed bf16 pairs: hi = round(v), lo = round(v - hi); vx in the low half
__device__ __forceinline__ void cr_split(float vx, float vy, uint32_t& hb, uint32_t& lb)
{
    const __nv_bfloat162 hi = __floats2bfloat162_rn(vx, vy);
    hb = *reinterpret_cast<const uint32_t*>(&hi);
    const __nv_bfloat162 lo = __floats2bfloat162_rn(vx - __uint_as_float(hb << 16), vy - __uint_as_float(hb & 0xffff0000u));
    lb = *reinterpret_cast<const uint32_t*>(&lo);
}

__device__ __forceinline__ float2 cr_ldg2(const float* p)
{
    float2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
    return v;
}

template <int MT>
__global__ void __launch_bounds__(CR_THREADS, 1)
pfb_ctr_kernel(const float* __restrict__ x, long long stream_stride, const float* __restrict__ window,
               float2* __restrict__ out, long long F, long long NBLK, int M, int groups_per_stream, int total_groups)
{
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    CrSmem& sm = *reinterpret_cast<CrSmem*>(smem_raw);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

    // ---- one-time setup: B1, twiddle table, barriers, TMEM, taps
    for (int e = tid; e < 128 * 64; e += CR_THREADS) {
        const int n = e >> 6, b = e & 63, kb = n >> 1;
        float sn, cs;
        sincospif((float)((b * kb) & 63) * (1.0f / 32.0f), &sn, &cs);
        const float v = (n & 1) ? -sn : cs;
        const __nv_bfloat16 hi = __float2bfloat16_rn(v);
        *reinterpret_cast<__nv_bfloat16*>(sm.bm[0] + cr_sw128(n, b * 2)) = hi;
        *reinterpret_cast<__nv_bfloat16*>(sm.bm[1] + cr_sw128(n, b * 2)) = __float2bfloat16_rn(v - __bfloat162float(hi));
    }
    for (int e = tid; e < 64 * 64; e += CR_THREADS) {
        const int kb = e >> 6, a = e & 63;
        double sn, cs;
        sincospi((double)(a * kb) / 2048.0, &sn, &cs);
        sm.tw[kb * CR_TWP + a] = make_float2((float)cs, (float)-sn);
    }
    if (tid == 0) { for (int i = 0; i < 4; ++i) mbar_init(smem_u32(&sm.bar[i]), 1); fence_mbar_init(); }
    if (warp == 0) { tmem_alloc<1>(smem_u32(&sm.tmem_base), 512); tmem_relinquish<1>(); }
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = sm.tmem_base;
    // taps of this thread's columns p = 2 lane (+ 1) + 64 (4 warp + bi): TMEM columns 256 .. 511, its own lane of its
    // warp's lane quarter, 16 columns per bi holding (tap m of a, tap m of a + 1) pairs, zero beyond M
    const uint32_t tap_addr = tmem + ((uint32_t)((warp & 3) * 32) << 16) + 256 + (warp >> 2) * 64;
#pragma unroll 1
    for (int bi = 0; bi < CR_BPW; ++bi) {
        uint32_t tv[16];
        const float* wp = window + 2 * lane + 64 * (CR_BPW * warp + bi);
#pragma unroll
        for (int m = 0; m < 8; ++m) {
            tv[2 * m] = m < M ? __float_as_uint(__ldg(wp + (long long)m * CR_P)) : 0u;
            tv[2 * m + 1] = m < M ? __float_as_uint(__ldg(wp + (long long)m * CR_P + 1)) : 0u;
        }
        tmem_st16(tap_addr + bi * 16, tv);
    }
    tmem_st_wait();

    const uint32_t idesc1 = idesc_bf16(128, 128), idesc2 = idesc_bf16(128, 64);
    const uint64_t d_bh = smem_desc_sw128(smem_u32(sm.bm[0])), d_bl = smem_desc_sw128(smem_u32(sm.bm[1]));
    const uint64_t d_a = smem_desc_sw128(smem_u32(&sm.a[0][0][0][0]));
    constexpr uint64_t PART = (uint64_t)CR_TILE >> 4, BLOCK = 2 * PART, TILE = 2 * BLOCK;   // descriptor steps

    constexpr int WA = MT, NR = WA - 1 + CR_FR;
    // subfilter-stage store offset.  A thread owns a = 2 lane and 2 lane + 1 (one 8-byte load); within a frame's 64 tile
    // rows a sits at row rho(a) = a / 2 + 32 (a & 1), so the two rows are lane and lane + 32 (2-way instead of 4-way
    // bank conflicts); epilogue 1 undoes the permutation for free when it picks TMEM columns.  K bytes 8 warp .. + 7.
    const uint32_t fir_off = lane * 128 + ((((uint32_t)warp >> 1) ^ (lane & 7)) << 4) + 8 * (warp & 1);
    // epilogue roles: TMEM lane quarter; epilogue 1: frame of the tile and column half; epilogue 2: ka block
    const int eq = warp & 3, q4 = warp >> 2, eh = q4 >> 1, ch = q4 & 1;
    // the NR = WA - 1 + CR_FR samples of input columns (2 lane, 2 lane + 1) + 64 (4 warp + bi) that group gg needs; rows
    // outside the stream read as zero (the first groups when M < WA and the last group of a stream take that path)
    auto load_col = [&](int gg, int bi, float2 (&row)[NR]) {
        const long long r0 = (long long)(gg % groups_per_stream) * CR_FR + M - WA;
        const float* xg = x + (long long)(gg / groups_per_stream) * stream_stride + r0 * CR_P + 2 * lane + 64 * (CR_BPW * warp + bi);
        if (r0 >= 0 && r0 + NR <= NBLK) {                                  // uniform
#pragma unroll
            for (int j = 0; j < NR; ++j) row[j] = cr_ldg2(xg + j * CR_P);
        } else {
#pragma unroll
            for (int j = 0; j < NR; ++j)
                row[j] = (r0 + j >= 0 && r0 + j < NBLK) ? cr_ldg2(xg + j * CR_P) : make_float2(0.f, 0.f);
        }
    };
    // Loads run one column ahead of the FMAs: column bi + 1 is requested before column bi is computed, and column 0 of
    // the NEXT group right after this group's subfilter stage, so it is in flight during the MMA waits and epilogues.
    float2 pre[NR], pre1[NR];
    if ((int)blockIdx.x < total_groups) { load_col(blockIdx.x, 0, pre); load_col(blockIdx.x, 1, pre1); }
    uint32_t it = 0;
    for (int g = blockIdx.x; g < total_groups; g += gridDim.x, ++it) {
        const int s = g / groups_per_stream;
        const long long f0 = (long long)(g % groups_per_stream) * CR_FR;
        // ---- subfilter stage, Eq. (20): thread (warp w, lane l) owns a = 2 l, 2 l + 1 of columns b = 4 w .. 4 w + 3
        {
            uint32_t hA[CR_FR][2], lA[CR_FR][2], hB[CR_FR][2], lB[CR_FR][2];   // packed K cells of tile rows lane, lane + 32
            uint32_t hprev[CR_FR], lprev[CR_FR];
            float2 rows[2][NR];
#pragma unroll
            for (int j = 0; j < NR; ++j) { rows[0][j] = pre[j]; rows[1][j] = pre1[j]; }
#pragma unroll
            for (int bi = 0; bi < CR_BPW; ++bi) {
                uint32_t tv[16];
                tmem_ld16(tap_addr + bi * 16, tv);
                // columns 0 and 1 were requested during the previous group's epilogues; column bi + 1 >= 2 goes into the
                // buffer that column bi - 1 has just left
                if (bi >= 1 && bi + 1 < CR_BPW) load_col(g, bi + 1, rows[(bi + 1) & 1]);
                float2 (&row)[NR] = rows[bi & 1];
                tmem_ld_wait();
#pragma unroll
                for (int fl = 0; fl < CR_FR; ++fl) {
                    float2 y = make_float2(__uint_as_float(tv[0]) * row[fl + WA - 1].x, __uint_as_float(tv[1]) * row[fl + WA - 1].y);
#pragma unroll
                    for (int m = 1; m < WA; ++m)
                        y = cr_ffma2(make_float2(__uint_as_float(tv[2 * m]), __uint_as_float(tv[2 * m + 1])), row[fl + WA - 1 - m], y);
                    uint32_t hb, lb;                                       // low half: a = 2 l, high half: a = 2 l + 1
                    cr_split(y.x, y.y, hb, lb);
                    if (bi & 1) {
                        hA[fl][bi >> 1] = __byte_perm(hprev[fl], hb, 0x5410);
                        hB[fl][bi >> 1] = __byte_perm(hprev[fl], hb, 0x7632);
                        lA[fl][bi >> 1] = __byte_perm(lprev[fl], lb, 0x5410);
                        lB[fl][bi >> 1] = __byte_perm(lprev[fl], lb, 0x7632);
                    } else {
                        hprev[fl] = hb;
                        lprev[fl] = lb;
                    }
                }
            }
            if (g + (int)gridDim.x < total_groups) {
                load_col(g + (int)gridDim.x, 0, pre);
                load_col(g + (int)gridDim.x, 1, pre1);
                // columns 2 and 3 of the next group: pulled into L2 now, loaded into registers inside its subfilter stage
                const int gn = g + (int)gridDim.x;
                const long long r0 = (long long)(gn % groups_per_stream) * CR_FR + M - WA;
                if (r0 >= 0 && r0 + NR <= NBLK) {
                    const float* xg = x + (long long)(gn / groups_per_stream) * stream_stride + r0 * CR_P + 2 * lane + 64 * (CR_BPW * warp + 2);
                    if ((lane & 15) == 0) {
#pragma unroll
                        for (int j = 0; j < NR; ++j) {
                            asm volatile("prefetch.global.L2 [%0];" :: "l"(xg + j * CR_P));
                            asm volatile("prefetch.global.L2 [%0];" :: "l"(xg + j * CR_P + 64));
                        }
                    }
                }
            }
#pragma unroll
            for (int fl = 0; fl < CR_FR; ++fl) {
                uint8_t* const dst = &sm.a[fl >> 1][0][0][0] + (fl & 1) * 64 * 128 + fir_off;
                *reinterpret_cast<uint2*>(dst) = make_uint2(hA[fl][0], hA[fl][1]);
                *reinterpret_cast<uint2*>(dst + CR_TILE) = make_uint2(lA[fl][0], lA[fl][1]);
                *reinterpret_cast<uint2*>(dst + 32 * 128) = make_uint2(hB[fl][0], hB[fl][1]);
                *reinterpret_cast<uint2*>(dst + 32 * 128 + CR_TILE) = make_uint2(lB[fl][0], lB[fl][1]);
            }
        }
        fence_proxy_async();
        __syncthreads();
        // The two tiles of a group are pipelined against the tensor pipe: ALL warps run epilogue 1 of tile 0 while the
        // stage-1 MMAs of tile 1 execute, epilogue 1 of tile 1 while the stage-2 MMAs of tile 0 execute, epilogue 2 of
        // tile 0 while the stage-2 MMAs of tile 1 execute; only the stage-1 MMAs of tile 0 are waited for in full.
        // ---- stage 1 (transposed): D1^T[t] = B1 * A1[t]^T -> TMEM columns 128 t .. 128 t + 127 = (frame, a)
        if (warp == 0 && elect_one()) {
            tc_fence_after();
#pragma unroll
            for (int t = 0; t < 2; ++t) {
#pragma unroll
                for (int k = 0; k < 4; ++k) umma_bf16<1>(tmem + 128 * t, d_bh + 2 * k, d_a + t * TILE + PART + 2 * k, idesc1, k > 0);
#pragma unroll
                for (int k = 0; k < 4; ++k) umma_bf16<1>(tmem + 128 * t, d_bl + 2 * k, d_a + t * TILE + 2 * k, idesc1, 1);
#pragma unroll
                for (int k = 0; k < 4; ++k) umma_bf16<1>(tmem + 128 * t, d_bh + 2 * k, d_a + t * TILE + 2 * k, idesc1, 1);
                umma_commit(smem_u32(&sm.bar[t]));
            }
        }
#pragma unroll
        for (int t = 0; t < 2; ++t) {
            mbar_wait(smem_u32(&sm.bar[t]), it & 1u);
            tc_fence_after();
            // ---- epilogue 1 of tile t: warp (eq, eh, ch) reads TMEM lanes 32 eq .. + 31 = (kb = 16 eq + lane / 2,
            //      c = lane & 1) and the columns a = 32 ch .. 32 ch + 31 of frame 2 t + eh; the partner lane (lane ^ 1)
            //      holds the other part of G[a][kb].  G' = G * w:  Re = Gr wr - Gi wi,  Im = Gi wr + Gr wi  ->
            //      own * wr + partner * (c ? wi : -wi).
            {
                const int kb = 16 * eq + (lane >> 1), c = lane & 1;
                const float sgn = c ? 1.f : -1.f;
                const uint32_t row = eh * 64 + kb;
                uint8_t* const blk = &sm.a[t][c][0][0];
                const float4* twr = reinterpret_cast<const float4*>(sm.tw + kb * CR_TWP) + 16 * ch;
                // TMEM column rho of this frame holds a = 2 rho (rho < 32) or 2 (rho - 32) + 1: even a in ve, odd a in vo
                uint32_t ve[16], vo[16];
                tmem_ld16(tmem + ((uint32_t)(eq * 32) << 16) + 128 * t + 64 * eh + 16 * ch, ve);
                tmem_ld16(tmem + ((uint32_t)(eq * 32) << 16) + 128 * t + 64 * eh + 32 + 16 * ch, vo);
                tmem_ld_wait();
                float nyq = 0.f;
#pragma unroll
                for (int j4 = 0; j4 < 4; ++j4) {                           // a = 8 j8 .. 8 j8 + 7, j8 = 4 ch + j4
                    uint32_t hw[4], lw[4];
#pragma unroll
                    for (int i2 = 0; i2 < 4; ++i2) {
                        const int i = 4 * j4 + i2;                         // a = 32 ch + 2 i, + 1
                        const float4 w = twr[i];
                        const float v0 = __uint_as_float(ve[i]), v1 = __uint_as_float(vo[i]);
                        const float p0 = __shfl_xor_sync(0xffffffffu, v0, 1), p1 = __shfl_xor_sync(0xffffffffu, v1, 1);
                        nyq += v0 - v1;
                        const float o0 = fmaf(p0, sgn * w.y, v0 * w.x), o1 = fmaf(p1, sgn * w.w, v1 * w.z);
                        cr_split(o0, o1, hw[i2], lw[i2]);
                    }
                    const uint32_t off = cr_sw128(row, 16 * (4 * ch + j4));
                    *reinterpret_cast<uint4*>(blk + off) = make_uint4(hw[0], hw[1], hw[2], hw[3]);
                    *reinterpret_cast<uint4*>(blk + CR_TILE + off) = make_uint4(lw[0], lw[1], lw[2], lw[3]);
                }
                // k = 2048: X = sum_a (-1)^a G[a][0] (real; the lanes holding (kb = 0, re) have 32 terms each)
                if (eq == 0 && lane == 0) sm.nyq[t][eh][ch] = nyq;
            }
            fence_proxy_async();
            tc_fence_before();
            __syncthreads();
            // ---- stage 2 of tile t: D_R = Re(G') * B1[0..63]^T -> columns 128 t .. + 63,  D_I = Im(G') * B1[0..63]^T -> + 64 .. + 127
            if (warp == 0 && elect_one()) {
                tc_fence_after();
#pragma unroll
                for (int c = 0; c < 2; ++c) {
                    const uint64_t da = d_a + t * TILE + c * BLOCK;
                    const uint32_t dcol = tmem + 128 * t + 64 * c;
#pragma unroll
                    for (int k = 0; k < 4; ++k) umma_bf16<1>(dcol, da + PART + 2 * k, d_bh + 2 * k, idesc2, k > 0);
#pragma unroll
                    for (int k = 0; k < 4; ++k) umma_bf16<1>(dcol, da + 2 * k, d_bh + 2 * k, idesc2, 1);
#pragma unroll
                    for (int k = 0; k < 4; ++k) umma_bf16<1>(dcol, da + 2 * k, d_bl + 2 * k, idesc2, 1);
                }
                umma_commit(smem_u32(&sm.bar[2 + t]));
            }
            if (tid < 2) {                                                 // Nyquist bins of the tile's two frames
                const long long f = f0 + 2 * t + tid;
                if (f < F) out[((long long)s * F + f) * CR_NK + CR_P / 2] = make_float2(sm.nyq[t][tid][0] + sm.nyq[t][tid][1], 0.f);
            }
        }
        // ---- epilogue 2: warp (eq, q4) reads rows 32 eq .. + 31 = (frame 2 t + eq / 2, kb = 32 (eq & 1) + lane) and
        //      ka = 8 q4 .. 8 q4 + 7.  D_R = (C_r, -S_r), D_I = (C_i, -S_i):  X = (C_r + S_i, C_i - S_r).
        //      For a fixed ka the 32 lanes hold 32 consecutive channels: 256 contiguous bytes per warp store.
#pragma unroll
        for (int t = 0; t < 2; ++t) {
            mbar_wait(smem_u32(&sm.bar[2 + t]), it & 1u);
            tc_fence_after();
            const long long f = f0 + 2 * t + (eq >> 1);
            float2* const orow = out + ((long long)s * F + f) * CR_NK + 32 * (eq & 1) + lane + 64 * 8 * q4;
            uint32_t vr[16], vi[16];
            tmem_ld16(tmem + ((uint32_t)(eq * 32) << 16) + 128 * t + 16 * q4, vr);
            tmem_ld16(tmem + ((uint32_t)(eq * 32) << 16) + 128 * t + 64 + 16 * q4, vi);
            tmem_ld_wait();
            if (f < F) {
#pragma unroll
                for (int i = 0; i < 8; ++i)
                    orow[64 * i] = make_float2(__uint_as_float(vr[2 * i]) - __uint_as_float(vi[2 * i + 1]),
                                               __uint_as_float(vr[2 * i + 1]) + __uint_as_float(vi[2 * i]));
            }
        }
        tc_fence_before();
        // no barrier here: the next subfilter stage only writes shared memory whose MMAs have retired, and the next MMA
        // into these TMEM columns is issued behind the barrier that ends that stage
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc<1>(tmem, 512);
}

// ---------------------------------------------------------------------------------------------------------------
// Warp-specialised variant, OPT-IN (TINA_CTR_WS=1): correct (same parity tests) but measured SLOWER than the kernel
// above at config 5 (0.65 ms vs 0.60 ms), so it is not the default; kept as the measured experiment DESIGN.md describes.
// One CTA per SM, 20 warps:
//   warps 0-7   producers: subfilter stage only.  A thread owns a = 2 lane, 2 lane + 1 of columns b = 8 warp .. + 7 and a
//               GROUP of 4 frames (two 128-row tiles), loads one column ahead, writes the stage-1 operands of both tiles;
//   warps 8-15  epilogues, per TILE: epilogue 2 of tile T - 1, then epilogue 1 of tile T;
//   warp 16     issues the MMAs: stage 1 of tile T + 1, then stage 2 of tile T.
// Shared memory: four stage-1 operand tiles (a ring of two groups, 128 KB), ONE stage-2 operand tile (64 KB), B1 (32 KB).
// The twiddle W4096^(a kb) does not come from a 34 KB table here: an epilogue thread has a fixed kb, so it keeps
// W^(8 ah kb), ah = 0..7, and W^(al kb), al = 0..7, in registers and multiplies the two.
// TMEM: two 128-column accumulator slots (tile parity; stage 2 of a tile overwrites its own stage-1 columns once
// epilogue 1 has read them) + 256 columns of window taps.  Registers move with setmaxnreg inside 96 x 640.
// Why it loses: with 64 K registers per SM only 8 producer warps with one column of loads in flight fit next to the
// epilogue warps (22 KB in flight per SM); the subfilter stage alone then takes 0.43 ms (role-skipping runs), against
// 0.21 ms when all 16 warps of the kernel above load.
constexpr int CW_THREADS = 640, CW_PROD = 256, CW_EPI = 256;
constexpr int CW_BPW = 8;                             // b values per producer warp (8 warps x 8 = 64)

struct CwSmem {
    uint8_t a1[4][2][CR_TILE];                        // [tile slot][hi | lo]: rows (frame, rho(a)), K = b
    uint8_t a2[2][2][CR_TILE];                        // [real | imaginary parts of G'][hi | lo]: rows (frame, kb), K = a
    uint8_t bm[2][CR_TILE];
    uint64_t a1_full[2], a1_free[2], d1_full[2], a2_full, d2_full[2], d_free[2];
    uint32_t tmem_base;
};
static_assert(sizeof(CwSmem) + 1024 <= 227 * 1024, "shared memory budget");

template <int R> __device__ __forceinline__ void cw_reg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" :: "n"(R)); }
template <int R> __device__ __forceinline__ void cw_reg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" :: "n"(R)); }

template <int MT>
__global__ void __maxnreg__(96)
pfb_ctrws_kernel(const float* __restrict__ x, long long stream_stride, const float* __restrict__ window,
                 float2* __restrict__ out, long long F, long long NBLK, int M, int groups_per_stream, int total_groups)
{
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    CwSmem& sm = *reinterpret_cast<CwSmem*>(smem_raw);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

    for (int e = tid; e < 128 * 64; e += CW_THREADS) {
        const int n = e >> 6, b = e & 63, kb = n >> 1;
        float sn, cs;
        sincospif((float)((b * kb) & 63) * (1.0f / 32.0f), &sn, &cs);
        const float v = (n & 1) ? -sn : cs;
        const __nv_bfloat16 hi = __float2bfloat16_rn(v);
        *reinterpret_cast<__nv_bfloat16*>(sm.bm[0] + cr_sw128(n, b * 2)) = hi;
        *reinterpret_cast<__nv_bfloat16*>(sm.bm[1] + cr_sw128(n, b * 2)) = __float2bfloat16_rn(v - __bfloat162float(hi));
    }
    if (tid == 0) {
        for (int s = 0; s < 2; ++s) {
            mbar_init(smem_u32(&sm.a1_full[s]), CW_PROD);
            mbar_init(smem_u32(&sm.a1_free[s]), 1);
            mbar_init(smem_u32(&sm.d1_full[s]), 1);
            mbar_init(smem_u32(&sm.d2_full[s]), 1);
            mbar_init(smem_u32(&sm.d_free[s]), CW_EPI);
        }
        mbar_init(smem_u32(&sm.a2_full), CW_EPI);
        fence_mbar_init();
    }
    if (warp == 0) { tmem_alloc<1>(smem_u32(&sm.tmem_base), 512); tmem_relinquish<1>(); }
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = sm.tmem_base;
    const int n_groups = ((int)blockIdx.x < total_groups) ? (total_groups - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
    const int n_tiles = 2 * n_groups;
    constexpr int WA = MT, NR = WA - 1 + CR_FR;

    if (warp < 8) {
        // ================================================================== producers: subfilter stage, Eq. (20)
        cw_reg_inc<112>();
        // taps of columns p = 2 lane (+ 1) + 64 (8 warp + bi): TMEM columns 256 + 128 (warp / 4) + 16 bi, (tap m of a,
        // tap m of a + 1) pairs, zero beyond M
        const uint32_t tap_addr = tmem + ((uint32_t)((warp & 3) * 32) << 16) + 256 + (warp >> 2) * 128;
#pragma unroll 1
        for (int bi = 0; bi < CW_BPW; ++bi) {
            uint32_t tv[16];
            const float* wp = window + 2 * lane + 64 * (CW_BPW * warp + bi);
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                tv[2 * m] = m < M ? __float_as_uint(__ldg(wp + (long long)m * CR_P)) : 0u;
                tv[2 * m + 1] = m < M ? __float_as_uint(__ldg(wp + (long long)m * CR_P + 1)) : 0u;
            }
            tmem_st16(tap_addr + bi * 16, tv);
        }
        tmem_st_wait();
        // tile rows lane (a even) and lane + 32 (a odd) of each frame, K bytes 16 warp + 8 half .. + 7
        const uint32_t fir_off = lane * 128 + ((((uint32_t)warp) ^ (lane & 7)) << 4);
        auto load_col = [&](int gg, int bi, float2 (&row)[NR]) {
            const long long r0 = (long long)(gg % groups_per_stream) * CR_FR + M - WA;
            const float* xg = x + (long long)(gg / groups_per_stream) * stream_stride + r0 * CR_P + 2 * lane + 64 * (CW_BPW * warp + bi);
            if (r0 >= 0 && r0 + NR <= NBLK) {                                  // uniform
#pragma unroll
                for (int j = 0; j < NR; ++j) row[j] = cr_ldg2(xg + j * CR_P);
            } else {
#pragma unroll
                for (int j = 0; j < NR; ++j)
                    row[j] = (r0 + j >= 0 && r0 + j < NBLK) ? cr_ldg2(xg + j * CR_P) : make_float2(0.f, 0.f);
            }
        };
        float2 rows[2][NR];
        if (n_groups > 0) load_col(blockIdx.x, 0, rows[0]);
#pragma unroll 1
        for (int i = 0; i < n_groups; ++i) {
            const int g = (int)blockIdx.x + i * (int)gridDim.x;
            uint8_t* const abase = &sm.a1[2 * (i & 1)][0][0] + fir_off;
#pragma unroll 1
            for (int half = 0; half < 2; ++half) {
                uint32_t hA[CR_FR][2], lA[CR_FR][2], hB[CR_FR][2], lB[CR_FR][2];
                uint32_t hprev[CR_FR], lprev[CR_FR];
#pragma unroll
                for (int b4 = 0; b4 < 4; ++b4) {
                    const int bi = 4 * half + b4;
                    uint32_t tv[16];
                    tmem_ld16(tap_addr + bi * 16, tv);
                    // the next column (or column 0 of the next group) is requested before this one is computed
                    if (bi + 1 < CW_BPW) load_col(g, bi + 1, rows[(b4 + 1) & 1]);
                    else if (i + 1 < n_groups) load_col(g + (int)gridDim.x, 0, rows[0]);
                    float2 (&row)[NR] = rows[b4 & 1];
                    tmem_ld_wait();
#pragma unroll
                    for (int fl = 0; fl < CR_FR; ++fl) {
                        float2 y = make_float2(__uint_as_float(tv[0]) * row[fl + WA - 1].x, __uint_as_float(tv[1]) * row[fl + WA - 1].y);
#pragma unroll
                        for (int m = 1; m < WA; ++m)
                            y = cr_ffma2(make_float2(__uint_as_float(tv[2 * m]), __uint_as_float(tv[2 * m + 1])), row[fl + WA - 1 - m], y);
                        uint32_t hb, lb;                                       // low half: a = 2 l, high half: a = 2 l + 1
                        cr_split(y.x, y.y, hb, lb);
                        if (b4 & 1) {
                            hA[fl][b4 >> 1] = __byte_perm(hprev[fl], hb, 0x5410);
                            hB[fl][b4 >> 1] = __byte_perm(hprev[fl], hb, 0x7632);
                            lA[fl][b4 >> 1] = __byte_perm(lprev[fl], lb, 0x5410);
                            lB[fl][b4 >> 1] = __byte_perm(lprev[fl], lb, 0x7632);
                        } else {
                            hprev[fl] = hb;
                            lprev[fl] = lb;
                        }
                    }
                }
                // the slot's previous contents (stage-1 operands of group i - 2) must have been consumed
                if (half == 0 && i >= 2) mbar_wait(smem_u32(&sm.a1_free[i & 1]), ((i >> 1) - 1) & 1u);
#pragma unroll
                for (int fl = 0; fl < CR_FR; ++fl) {
                    uint8_t* const dst = abase + (fl >> 1) * 2 * CR_TILE + (fl & 1) * 64 * 128 + 8 * half;
                    *reinterpret_cast<uint2*>(dst) = make_uint2(hA[fl][0], hA[fl][1]);
                    *reinterpret_cast<uint2*>(dst + CR_TILE) = make_uint2(lA[fl][0], lA[fl][1]);
                    *reinterpret_cast<uint2*>(dst + 32 * 128) = make_uint2(hB[fl][0], hB[fl][1]);
                    *reinterpret_cast<uint2*>(dst + 32 * 128 + CR_TILE) = make_uint2(lB[fl][0], lB[fl][1]);
                }
            }
            fence_proxy_async();
            mbar_arrive(smem_u32(&sm.a1_full[i & 1]));
        }
    } else if (warp < 16) {
        // ================================================================== epilogue warps
        cw_reg_inc<104>();
        const int e = warp - 8, eq = e & 3, eh = e >> 2;
        const uint32_t tq = tmem + ((uint32_t)(eq * 32) << 16);
        // epilogue 1: TMEM lane = (kb = 16 eq + lane / 2, c = lane & 1).  G' = G w with w = W4096^(a kb) = (wr, wi):
        // Re = Gr wr - Gi wi, Im = Gi wr + Gr wi  ->  own * wr + partner * sgn wi, sgn = c ? 1 : -1.
        // w(a) = base[a / 8] * step[a % 8]; the sign is folded into the imaginary parts (sgn^2 = 1).
        const int kb = 16 * eq + (lane >> 1), c = lane & 1;
        float br[8], bj[8], sr[8], sj[8];
        {
            // arguments j kb / 2048 are exact in fp32, so sincospif is good to about an ulp
            const float sgn = c ? 1.f : -1.f;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                float sn, cs;
                sincospif((float)((8 * j * kb) & 4095) * (1.0f / 2048.0f), &sn, &cs);
                br[j] = cs;
                bj[j] = -sn * sgn;
                sincospif((float)(j * kb) * (1.0f / 2048.0f), &sn, &cs);
                sr[j] = cs;
                sj[j] = -sn * sgn;
            }
        }
        auto epi2 = [&](int T) {
            // rows 32 eq .. + 31 = (frame eq / 2 of the tile, kb = 32 (eq & 1) + lane), ka = 16 eh .. + 15.
            // D_R = (C_r, -S_r), D_I = (C_i, -S_i):  X = (C_r + S_i, C_i - S_r); 256 contiguous bytes per warp store.
            const int g = (int)blockIdx.x + (T >> 1) * (int)gridDim.x;
            const int s = g / groups_per_stream;
            const long long f = (long long)(g % groups_per_stream) * CR_FR + 2 * (T & 1) + (eq >> 1);
            float2* const orow = out + ((long long)s * F + f) * CR_NK + 32 * (eq & 1) + lane + 64 * 16 * eh;
            mbar_wait(smem_u32(&sm.d2_full[T & 1]), (T >> 1) & 1u);
            tc_fence_after();
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                uint32_t vr[16], vi[16];
                tmem_ld16(tq + 128 * (T & 1) + 32 * eh + 16 * h, vr);
                tmem_ld16(tq + 128 * (T & 1) + 64 + 32 * eh + 16 * h, vi);
                tmem_ld_wait();
                if (f < F) {
#pragma unroll
                    for (int q = 0; q < 8; ++q)
                        orow[64 * (8 * h + q)] = make_float2(__uint_as_float(vr[2 * q]) - __uint_as_float(vi[2 * q + 1]),
                                                             __uint_as_float(vr[2 * q + 1]) + __uint_as_float(vi[2 * q]));
                }
            }
            tc_fence_before();
            mbar_arrive(smem_u32(&sm.d_free[T & 1]));
        };
#pragma unroll 1
        for (int T = 0; T < n_tiles; ++T) {
            const int g = (int)blockIdx.x + (T >> 1) * (int)gridDim.x;
            const long long f = (long long)(g % groups_per_stream) * CR_FR + 2 * (T & 1) + eh;
            const uint32_t row = eh * 64 + kb;
            uint8_t* const blk = &sm.a2[c][0][0];
            if (T >= 1) epi2(T - 1);                    // frees tile T - 1's accumulators (stage 1 of T + 1) and implies A2 is free
            mbar_wait(smem_u32(&sm.d1_full[T & 1]), (T >> 1) & 1u);
            tc_fence_after();
            float nyq = 0.f;
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                // TMEM column rho of this frame holds a = 2 rho (rho < 32) or 2 (rho - 32) + 1: even a in ve, odd a in vo
                uint32_t ve[8], vo[8];
                tmem_ld8(tq + 128 * (T & 1) + 64 * eh + 8 * h, ve);
                tmem_ld8(tq + 128 * (T & 1) + 64 * eh + 32 + 8 * h, vo);
                tmem_ld_wait();
#pragma unroll
                for (int j2 = 0; j2 < 2; ++j2) {                           // a = 8 j8 .. 8 j8 + 7
                    const int j8 = 2 * h + j2;
                    uint32_t hw[4], lw[4];
                    // opaque to the optimiser: otherwise all 64 products are hoisted out of the tile loop and spilled
                    asm volatile("" : "+f"(br[j8]), "+f"(bj[j8]));
#pragma unroll
                    for (int i2 = 0; i2 < 4; ++i2) {
                        const int i = 4 * j2 + i2;                         // a = 8 j8 + 2 i2, + 1
                        const float w0r = br[j8] * sr[2 * i2] - bj[j8] * sj[2 * i2], w0j = br[j8] * sj[2 * i2] + bj[j8] * sr[2 * i2];
                        const float w1r = br[j8] * sr[2 * i2 + 1] - bj[j8] * sj[2 * i2 + 1], w1j = br[j8] * sj[2 * i2 + 1] + bj[j8] * sr[2 * i2 + 1];
                        const float v0 = __uint_as_float(ve[i]), v1 = __uint_as_float(vo[i]);
                        const float p0 = __shfl_xor_sync(0xffffffffu, v0, 1), p1 = __shfl_xor_sync(0xffffffffu, v1, 1);
                        nyq += v0 - v1;
                        const float o0 = fmaf(p0, w0j, v0 * w0r), o1 = fmaf(p1, w1j, v1 * w1r);
                        cr_split(o0, o1, hw[i2], lw[i2]);
                    }
                    const uint32_t off = cr_sw128(row, 16 * j8);
                    *reinterpret_cast<uint4*>(blk + off) = make_uint4(hw[0], hw[1], hw[2], hw[3]);
                    *reinterpret_cast<uint4*>(blk + CR_TILE + off) = make_uint4(lw[0], lw[1], lw[2], lw[3]);
                }
            }
            // k = 2048: X = sum_a (-1)^a G[a][0] (real; the lane holding (kb = 0, re) has all 64 terms)
            if (eq == 0 && lane == 0 && f < F) out[((long long)(g / groups_per_stream) * F + f) * CR_NK + CR_P / 2] = make_float2(nyq, 0.f);
            fence_proxy_async();
            tc_fence_before();
            mbar_arrive(smem_u32(&sm.a2_full));
        }
        if (n_tiles > 0) epi2(n_tiles - 1);
    } else {
        // ================================================================== MMA issuer (warp 16; warps 17-19 idle)
        cw_reg_dec<40>();
        if (warp == 16 && elect_one()) {
            const uint32_t idesc1 = idesc_bf16(128, 128), idesc2 = idesc_bf16(128, 64);
            const uint64_t d_bh = smem_desc_sw128(smem_u32(sm.bm[0])), d_bl = smem_desc_sw128(smem_u32(sm.bm[1]));
            const uint64_t d_a1 = smem_desc_sw128(smem_u32(&sm.a1[0][0][0])), d_a2 = smem_desc_sw128(smem_u32(&sm.a2[0][0][0]));
            constexpr uint64_t PART = (uint64_t)CR_TILE >> 4, BLOCK = 2 * PART;   // descriptor steps
#pragma unroll 1
            for (int T = 0; T <= n_tiles; ++T) {
                if (T < n_tiles) {
                    // ---- stage 1 (transposed): D1^T = B1 * A1^T -> accumulator slot T & 1, columns = (frame, rho(a))
                    const int i = T >> 1;
                    if ((T & 1) == 0) mbar_wait(smem_u32(&sm.a1_full[i & 1]), (i >> 1) & 1u);
                    if (T >= 2) mbar_wait(smem_u32(&sm.d_free[T & 1]), ((T >> 1) - 1) & 1u);      // accumulators drained
                    tc_fence_after();
                    const uint32_t dcol = tmem + 128 * (T & 1);
                    const uint64_t da = d_a1 + (uint64_t)(T & 3) * BLOCK;
#pragma unroll
                    for (int k = 0; k < 4; ++k) umma_bf16<1>(dcol, d_bh + 2 * k, da + PART + 2 * k, idesc1, k > 0);
#pragma unroll
                    for (int k = 0; k < 4; ++k) umma_bf16<1>(dcol, d_bl + 2 * k, da + 2 * k, idesc1, 1);
#pragma unroll
                    for (int k = 0; k < 4; ++k) umma_bf16<1>(dcol, d_bh + 2 * k, da + 2 * k, idesc1, 1);
                    umma_commit(smem_u32(&sm.d1_full[T & 1]));
                    if (T & 1) umma_commit(smem_u32(&sm.a1_free[i & 1]));
                }
                if (T >= 1) {
                    // ---- stage 2 of tile U: D_R = Re(G') B1[0..63]^T -> columns + 0 .. 63, D_I = Im(G') B1[0..63]^T -> + 64 .. 127
                    const int U = T - 1;
                    mbar_wait(smem_u32(&sm.a2_full), U & 1u);
                    tc_fence_after();
#pragma unroll
                    for (int c = 0; c < 2; ++c) {
                        const uint64_t da = d_a2 + c * BLOCK;
                        const uint32_t dcol = tmem + 128 * (U & 1) + 64 * c;
#pragma unroll
                        for (int k = 0; k < 4; ++k) umma_bf16<1>(dcol, da + PART + 2 * k, d_bh + 2 * k, idesc2, k > 0);
#pragma unroll
                        for (int k = 0; k < 4; ++k) umma_bf16<1>(dcol, da + 2 * k, d_bh + 2 * k, idesc2, 1);
#pragma unroll
                        for (int k = 0; k < 4; ++k) umma_bf16<1>(dcol, da + 2 * k, d_bl + 2 * k, idesc2, 1);
                    }
                    umma_commit(smem_u32(&sm.d2_full[U & 1]));
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc<1>(tmem, 512);
}

tina_status ctr_pfb(const void* x, int S, long long n_samples, int M, const float* window, void* out, cudaStream_t st)
{
    const long long NBLK = n_samples / CR_P, F = NBLK - M + 1;
    const long long gps = (F + CR_FR - 1) / CR_FR;
    if (gps * S > 0x7fffffffLL) return fail(TINA_ERR_UNSUPPORTED, "tina_pfb_fft: too many frames");
    DevCtx* ctx = nullptr;
    tina_status ps = dev_ctx(&ctx);
    if (ps != TINA_OK) return ps;
    const int n_sm = ctx->n_sm;
    const int total = (int)(gps * S);
    const int grid = total < n_sm ? total : n_sm;           // one CTA per SM (all 512 TMEM columns)
    const float* xf = static_cast<const float*>(x);
    float2* of = static_cast<float2*>(out);
    if (options().ctr_ws) {                                 // warp-specialised variant: one 640-thread CTA per SM
        const size_t wsmem = sizeof(CwSmem) + 1024;
        const void* kw = M <= 4 ? (const void*)pfb_ctrws_kernel<4> : (const void*)pfb_ctrws_kernel<8>;
        if ((ps = ensure_smem(ctx, kw, (int)wsmem, "pfb_ctrws_kernel setup")) != TINA_OK) return ps;
        if (M <= 4) pfb_ctrws_kernel<4><<<grid, CW_THREADS, wsmem, st>>>(xf, n_samples, window, of, F, NBLK, M, (int)gps, total);
        else pfb_ctrws_kernel<8><<<grid, CW_THREADS, wsmem, st>>>(xf, n_samples, window, of, F, NBLK, M, (int)gps, total);
        count_launch();
        g_last_path = kPathUmma; note_kernel("pfb_ctrws_kernel");
        return check_cuda(cudaGetLastError(), "pfb_ctrws_kernel launch");
    }
    const size_t smem = sizeof(CrSmem) + 1024;
    {
        const void* kc = M <= 4 ? (const void*)pfb_ctr_kernel<4> : (const void*)pfb_ctr_kernel<8>;
        if ((ps = ensure_smem(ctx, kc, (int)smem, "pfb_ctr_kernel setup")) != TINA_OK) return ps;
    }
    if (M <= 4) pfb_ctr_kernel<4><<<grid, CR_THREADS, smem, st>>>(xf, n_samples, window, of, F, NBLK, M, (int)gps, total);
    else pfb_ctr_kernel<8><<<grid, CR_THREADS, smem, st>>>(xf, n_samples, window, of, F, NBLK, M, (int)gps, total);
    count_launch();
    g_last_path = kPathUmma; note_kernel("pfb_ctr_kernel");
    return check_cuda(cudaGetLastError(), "pfb_ctr_kernel launch");
}

}  // namespace tina
