// tina_firt.cu -- standalone FIR (Eq. (15)) as a banded-Toeplitz contraction on the tensor cores,
// round-2 kernel: the paper's unfolding view (Eq. (17)-(19)).
//
// A channel is cut into blocks of T = 128 outputs; block b needs the T + M - 1 inputs x[bT .. bT + T + M - 2]:
//     y[bT + n] = sum_c x[bT + c] * Tz[c][n],      Tz[c][n] = a[n + M-1 - c]   (0 outside the band 0 <= . < M)
// i.e. a GEMM whose A rows are overlapping windows of the signal (row pitch T) and whose B is the fixed Toeplitz
// matrix of the taps, K = T + M - 1 padded to a multiple of 32.  fp32 accuracy as everywhere in libtina: A and B
// split into bf16 hi + lo, three products (lo*hi, hi*hi, hi*lo), fp32 accumulation in TMEM.
//
// What differs from the round-1 route through pfb_umma_kernel (measured there: the issuing thread needed ~207
// cycles per M256 x N128 x K16 instruction against ~90 for the bare loop, producers busy 70 % on exposed global
// load latency, 0.46 of the HBM roofline):
//   * the Toeplitz matrix is built ONCE per CTA from the taps, straight into shared memory, and stays resident
//     (no per-call toeplitz_kernel, no tensor map, no B ring, no L2 traffic for B);
//   * the signal is staged by TMA: a 3-D map {128, L / 128, C} over x, 128-byte-swizzled boxes of 32 floats x 128 rows; chunk kc of
//     a tile is the box at column 32 (kc % 4) of row (tile row + kc / 4) -- the overlap of the A rows costs
//     nothing but L2 bandwidth, and rows past the end of a channel arrive as zeros;
//   * the producers only convert, and the A operand lives in TENSOR MEMORY, not in shared memory: a producer lane
//     owns one row of the staged 128 x 32 block (ld.shared.v4 from the 128-byte-swizzled TMA box), packs bf16x2 hi
//     and the exact remainder's bf16x2 lo, and writes both with tcgen05.st into the 128 TMEM columns kept for A
//     (4 slots x (16 hi + 16 lo) columns); the MMAs read A from there (tcgen05.mma with a TMEM A operand), so the
//     operand costs neither st.shared nor tensor-core shared-memory reads -- shared-memory bandwidth was the bound
//     of the shared-memory-operand version (r02 captures: 82 % of the 128 B/clk pipe);
//   * three TMEM accumulator stages of 128 columns, so the epilogue of a tile overlaps the MMAs of the next two.
// CTA pair, tcgen05.mma.cta_group::2, M = 256 (each CTA 128 rows), N = 128 (each CTA holds 64 rows of B).
// Needs L % 128 == 0 (the 3-D view) and M <= 193; other shapes keep the round-1 route or the CUDA-core kernel.
#include "tina_umma.cuh"

#include <cstring>
#include <vector>

namespace tina {

using namespace ptx;

constexpr int FT_T = 128;                         // outputs per block (GEMM N) and A row pitch
constexpr int FT_KC = 32;                         // contraction elements per chunk (64-byte rows, SWIZZLE_64B)
constexpr int FT_A_COLS = FT_KC / 2;              // TMEM columns of one part (hi or lo) of an A chunk: bf16 pairs
constexpr int FT_A_SLOTS = 4;                     // A chunks resident in TMEM
constexpr int FT_B_TILE = (FT_T / UMMA_CG) * FT_KC * 2;   // 4 KB: this CTA's 64 rows of one chunk and part
constexpr int FT_IN_SLOT = BM * FT_KC * 4;        // 16 KB fp32
constexpr int FT_PITCH = 129;                     // staged row pitch (floats) of the epilogue: odd, see below
constexpr int FT_STAGE = 32 * FT_PITCH * 4;       // per epilogue warp
constexpr int FT_ACC = 3;                         // TMEM accumulator stages of 128 columns
constexpr int FT_A_COL0 = FT_ACC * FT_T;          // first TMEM column of the A slots
static_assert(FT_A_COL0 + FT_A_SLOTS * 2 * FT_A_COLS <= 512, "TMEM budget");

struct FirtCtl {
    uint64_t a_full[4], a_empty[4];
    uint64_t in_full[8], in_empty[8];
    uint64_t t_full[FT_ACC], t_empty[FT_ACC];
    uint64_t b_free, b_ready;          // per-channel taps: "all MMAs that read the old matrix are done" / "new matrix written"
    uint32_t tmem_base;
};

struct FirtParams {
    const float* taps;         // [M] (taps_stride == 0) or [C][M]
    float* y;                  // [C][Lo]
    long long Lo;              // outputs per channel
    int M, n_kc;               // taps, chunks (Kp / 32)
    int taps_stride;           // 0: one tap vector; M: one per channel
    int tiles_per_chan, total_work;
    int in_slots;              // input ring depth (even: see the producers)
    int b_part_bytes;          // bytes of one part (hi or lo) of the resident band matrix, multiple of 1024
    unsigned long long* prof;  // -DTINA_DEV only (TINA_PROF): [grid][16] cycle counters
    int debug;                 // -DTINA_DEV only (TINA_DEBUG_SKIP): 128 no global stores, 256 no TMA loads, 512 no MMAs, 1024 no operand writes, 2048 no TMEM read-out
};
#ifdef TINA_DEV
#define FT_DBG(b) (prm.debug & (b))
#else
#define FT_DBG(b) 0
#endif
#ifdef TINA_DEV
#define FT_NOW() (prm.prof ? clock64() : 0LL)
#else
#define FT_NOW() 0LL
#endif

__device__ __forceinline__ float2 firt_lds_f2(uint32_t addr)
{
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ void firt_sts16(uint32_t addr, uint32_t v)
{
    asm volatile("st.shared.b16 [%0], %1;" ::"r"(addr), "h"((unsigned short)v) : "memory");
}

__global__ void __launch_bounds__(UMMA_THREADS, 1)
fir_umma_kernel(const __grid_constant__ CUtensorMap tmap_x, const FirtParams prm)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    if ((smem_u32(smem) & 1023u) != 0) __trap();
    constexpr int CG = UMMA_CG;
    const int n_kc = prm.n_kc;
    // Every 32-row chunk of the Toeplitz matrix is a window of ONE band matrix G[n'][c'] = a[n' + M-1 - c'],
    // c' in [0, 32): chunk kc needs the rows n' = n - 32 kc, so this CTA keeps the 64 + 32 (n_kc - 1) rows
    // n' in [64 rank - 32 (n_kc - 1), 64 rank + 64) once (hi | lo) and chunk kc's B tile starts 32 (n_kc - 1 - kc) rows in.
    uint8_t* b_res = smem;
    const uint32_t b_part = (uint32_t)prm.b_part_bytes;                   // bytes of one part, multiple of 1024
    uint8_t* in_ring = b_res + 2 * (size_t)b_part;
    uint8_t* stage = in_ring + (size_t)prm.in_slots * FT_IN_SLOT;
    FirtCtl* ctl = reinterpret_cast<FirtCtl*>(stage + 4 * FT_STAGE);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();
    constexpr uint32_t leader = 0;
    constexpr uint16_t pair_mask = 3;
    const int cl = blockIdx.x / CG, n_cl = gridDim.x / CG;
    constexpr uint32_t n_a = FT_A_SLOTS;
    const uint32_t n_in = (uint32_t)prm.in_slots;
    // contiguous ranges of tiles per pair: a pair stays inside a channel as long as possible (per-channel taps
    // rebuild the Toeplitz matrix only when the channel changes)
    const int per = (prm.total_work + n_cl - 1) / n_cl;
    const int w_begin = min(cl * per, prm.total_work), w_end = min(w_begin + per, prm.total_work);

    if (warp == TMA_WARP && lane == 0) {
        prefetch_tmap(&tmap_x);
        for (int i = 0; i < FT_A_SLOTS; ++i) {
            mbar_init(smem_u32(&ctl->a_full[i]), N_PROD_WARPS / 2 + (rank == 0 ? CG - 1 : 0));   // one producer group per chunk
            mbar_init(smem_u32(&ctl->a_empty[i]), 1);
        }
        for (int i = 0; i < 8; ++i) {
            mbar_init(smem_u32(&ctl->in_full[i]), 1);
            mbar_init(smem_u32(&ctl->in_empty[i]), N_PROD_WARPS / 2);
        }
        for (int i = 0; i < FT_ACC; ++i) { mbar_init(smem_u32(&ctl->t_full[i]), 1); mbar_init(smem_u32(&ctl->t_empty[i]), 4 * CG); }
        mbar_init(smem_u32(&ctl->b_free), 1);
        mbar_init(smem_u32(&ctl->b_ready), N_PROD_WARPS + (rank == 0 ? CG - 1 : 0));
        fence_mbar_init();
    }
    if (warp == ALLOC_WARP) {
        tmem_alloc<CG>(smem_u32(&ctl->tmem_base), 512);
        tmem_relinquish<CG>();
    }
    // band matrix of channel `chan`, bf16 hi | lo, K-major, 64-byte-swizzled: element (j, c') at row j, 16-byte chunk
    // (c' >> 3) ^ ((j >> 1) & 3)
    auto build_b = [&](int chan, int tid, int nthreads) {
        const float* taps = prm.taps + (long long)chan * prm.taps_stride;
        const int M = prm.M, rows = FT_T / CG + FT_KC * (n_kc - 1);
        const int n0 = (int)rank * (FT_T / CG) - FT_KC * (n_kc - 1);      // n' of row 0
        const uint32_t b_s = smem_u32(b_res);
        for (int idx = tid; idx < rows * FT_KC; idx += nthreads) {
            const int j = idx / FT_KC, cc = idx - j * FT_KC;
            const int k = n0 + j + M - 1 - cc;
            const float v = (k >= 0 && k < M) ? __ldg(taps + k) : 0.f;
            const __nv_bfloat16 hi = __float2bfloat16(v);
            const __nv_bfloat16 lo = __float2bfloat16(v - __bfloat162float(hi));
            const uint32_t off = (uint32_t)j * 64u + ((((uint32_t)cc >> 3) ^ (((uint32_t)j >> 1) & 3u)) << 4) + ((uint32_t)cc & 7u) * 2u;
            firt_sts16(b_s + off, (uint32_t)__bfloat16_as_ushort(hi));
            firt_sts16(b_s + off + b_part, (uint32_t)__bfloat16_as_ushort(lo));
        }
    };
    if (prm.taps_stride == 0 || w_begin < w_end) build_b(prm.taps_stride ? w_begin / prm.tiles_per_chan : 0, threadIdx.x, UMMA_THREADS);
    fence_proxy_async();
    tc_fence_before();
    cluster_sync();
    tc_fence_after();
    const uint32_t tmem_base = ctl->tmem_base;
    // per-channel taps: tile w starts a new channel (the pair's first tile was built above)
    auto new_channel = [&](int w) { return prm.taps_stride != 0 && w > w_begin && (w % prm.tiles_per_chan) == 0; };

    if (warp == TMA_WARP) {
        // ============================ TMA producer: signal rows ================================
        if (lane == 0) {
            RingPos in;
            long long pt_w = 0, pt_x, pt_tot = FT_NOW();
            for (int w = w_begin; w < w_end; ++w) {
                const int chan = w / prm.tiles_per_chan;
                const int row0 = (w % prm.tiles_per_chan) * (BM * CG) + (int)rank * BM;
                for (int kc = 0; kc < n_kc; ++kc) {
                    pt_x = FT_NOW(); mbar_wait<64>(smem_u32(&ctl->in_empty[in.idx]), in.phase ^ 1); pt_w += FT_NOW() - pt_x;
                    const uint32_t bar = smem_u32(&ctl->in_full[in.idx]);
                    if (FT_DBG(256)) mbar_arrive(bar);
                    else {
                        mbar_expect_tx(bar, FT_IN_SLOT);
                        tma_load_3d(smem_u32(in_ring + in.idx * FT_IN_SLOT), &tmap_x, bar, FT_KC * (kc & 3), row0 + (kc >> 2), chan);
                    }
                    in.advance(n_in);
                }
            }
            if (prm.prof) { unsigned long long* pp = prm.prof + blockIdx.x * 16; pp[0] = FT_NOW() - pt_tot; pp[1] = pt_w; }
        }
    } else if (warp == MMA_WARP) {
        // ============================ MMA issuer =============================================
        if (rank != 0) {
            RingPos a;                                    // forward "my A tile is ready" to the leader
            uint32_t br_phase = 0;
            for (int w = w_begin; w < w_end; ++w) {
                if (new_channel(w)) {                     // ... and "my half of the new Toeplitz matrix is written"
                    mbar_wait(smem_u32(&ctl->b_ready), br_phase);
                    br_phase ^= 1u;
                    if (lane == 0) mbar_arrive_cluster(smem_u32(&ctl->b_ready), leader);
                    __syncwarp();
                }
                for (int kc = 0; kc < n_kc; ++kc) {
                    mbar_wait(smem_u32(&ctl->a_full[a.idx]), a.phase);
                    if (lane == 0) mbar_arrive_cluster(smem_u32(&ctl->a_full[a.idx]), leader);
                    __syncwarp();
                    a.advance(n_a);
                }
            }
        } else {
            RingPos a, t;
            uint32_t br_phase = 0;
            long long pm_a = 0, pm_t = 0, pm_x, pm_tot = FT_NOW();
            const uint32_t idesc = idesc_bf16(BM * CG, FT_T, false);
            // descriptors of the resident band matrix, chunk 0 (the 14-bit address field takes the per-chunk offset
            // by plain addition: all of shared memory is below 2^18 bytes)
            const uint64_t b_hi0 = smem_desc_sw64(smem_u32(b_res)), b_lo0 = smem_desc_sw64(smem_u32(b_res) + b_part);
            const uint32_t a_t0 = tmem_base + FT_A_COL0;
            for (int w = w_begin; w < w_end; ++w) {
                if (new_channel(w)) {
                    // every MMA issued so far has read the old matrix: release it once they are done, then wait
                    // until both CTAs have written the new one
                    if (lane == 0) commit_cg<CG>(smem_u32(&ctl->b_free), pair_mask);
                    __syncwarp();
                    mbar_wait(smem_u32(&ctl->b_ready), br_phase);
                    br_phase ^= 1u;
                    tc_fence_after();
                }
                pm_x = FT_NOW(); mbar_wait(smem_u32(&ctl->t_empty[t.idx]), t.phase ^ 1); pm_t += FT_NOW() - pm_x;      // the epilogue has drained this stage
                tc_fence_after();
                const uint32_t d = tmem_base + t.idx * (uint32_t)FT_T;
                for (int kc = 0; kc < n_kc; ++kc) {
                    pm_x = FT_NOW(); mbar_wait(smem_u32(&ctl->a_full[a.idx]), a.phase); pm_a += FT_NOW() - pm_x;
                    tc_fence_after();
                    // one ELECTED thread issues (the compiler then knows a single thread is active and emits the
                    // tcgen05 instructions straight; under `lane == 0` it wraps each in an any-thread loop, and the
                    // issuing thread, not the tensor pipe, bounded the kernel: ~150 cycles per instruction against 64)
                    if (elect_one()) {
                        const uint32_t a_hi = a_t0 + a.idx * (2 * FT_A_COLS), a_lo = a_hi + FT_A_COLS;
                        const uint64_t b_step = (uint64_t)((uint32_t)(n_kc - 1 - kc) * (FT_KC * 64u) >> 4);     // 32 rows of 64 B per chunk step
                        const uint64_t b_hi = b_hi0 + b_step, b_lo = b_lo0 + b_step;
                        uint32_t acc = kc > 0;
                        if (!FT_DBG(512)) {
#pragma unroll
                        for (int k = 0; k < FT_KC / 16; ++k) { umma_bf16_ts<CG>(d, a_lo + 8 * k, b_hi + 2 * k, idesc, acc); acc = 1; }
#pragma unroll
                        for (int k = 0; k < FT_KC / 16; ++k) umma_bf16_ts<CG>(d, a_hi + 8 * k, b_hi + 2 * k, idesc, 1);
#pragma unroll
                        for (int k = 0; k < FT_KC / 16; ++k) umma_bf16_ts<CG>(d, a_hi + 8 * k, b_lo + 2 * k, idesc, 1);
                        }
                        commit_cg<CG>(smem_u32(&ctl->a_empty[a.idx]), pair_mask);
                        if (kc == n_kc - 1) commit_cg<CG>(smem_u32(&ctl->t_full[t.idx]), pair_mask);
                    }
                    __syncwarp();
                    a.advance(n_a);
                }
                t.advance(FT_ACC);
            }
            if (prm.prof && lane == 0) { unsigned long long* pp = prm.prof + blockIdx.x * 16; pp[2] = FT_NOW() - pm_tot; pp[3] = pm_a; pp[4] = pm_t; }
        }
    } else if (warp >= EPI_WARP0 && warp < EPI_WARP0 + 4) {
        // ============================ epilogue ==============================================
        // The warp's 32 rows x 128 columns are ONE contiguous run of 4096 floats of y[chan] that is only 4-byte
        // aligned (Lo is odd for even L and M): stage it (row pitch 132 floats), hand the accumulator back, and
        // write the run as 16-byte-aligned float4 with a scalar head and tail.
        const int q = warp - EPI_WARP0;
        float* stg = reinterpret_cast<float*>(stage + q * FT_STAGE);
        RingPos t;
        long long pe_w = 0, pe_s = 0, pe_x, pe_tot = FT_NOW();
        for (int w = w_begin; w < w_end; ++w) {
            const int chan = w / prm.tiles_per_chan;
            const long long row0 = (long long)(w % prm.tiles_per_chan) * (BM * CG) + rank * BM + q * 32;
            pe_x = FT_NOW(); mbar_wait<128>(smem_u32(&ctl->t_full[t.idx]), t.phase); pe_w += FT_NOW() - pe_x; pe_x = FT_NOW();
            tc_fence_after();
            const uint32_t taddr = tmem_base + t.idx * (uint32_t)FT_T + ((uint32_t)(q * 32) << 16);
            uint32_t r[32];
            if (!FT_DBG(2048)) {
            tmem_ld32(taddr, r);
#pragma unroll
            for (int cb = 0; cb < FT_T; cb += 32) {
                tmem_ld_wait();
                // staged layout: element e of a row at word (e >> 2) + 32 (e & 3) of the row (pitch 129 words): the
                // writes (lane = row, odd pitch) and the read-out below (lanes 4 elements apart) are both conflict-free
#pragma unroll
                for (int j = 0; j < 8; ++j)
#pragma unroll
                    for (int k = 0; k < 4; ++k)
                        stg[lane * FT_PITCH + (cb >> 2) + j + 32 * k] = __uint_as_float(r[4 * j + k]);
                if (cb + 32 < FT_T) tmem_ld32(taddr + cb + 32, r);
            }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) arrive_leader<CG>(smem_u32(&ctl->t_empty[t.idx]), rank, leader);
            pe_s += FT_NOW() - pe_x;
            const long long e0 = row0 * FT_T;                              // first element of the run in the channel
            long long n_run = prm.Lo - e0;
            if (n_run > 32LL * FT_T) n_run = 32LL * FT_T;
            if (n_run > 0 && !FT_DBG(128)) {
                float* g = prm.y + (long long)chan * prm.Lo + e0;
                const int run = (int)n_run;
                const int head = min(run, (int)(((16u - ((uint32_t)(uintptr_t)g & 15u)) & 15u) >> 2));
                const int nv4 = (run - head) >> 2;
                auto at = [&](int l) { return stg[(l >> 7) * FT_PITCH + ((l & 127) >> 2) + 32 * (l & 3)]; };
                if (lane < head) g[lane] = at(lane);
                // (an aligned-float4 variant -- two ld.shared.v4 of the staged row and a funnel shift by `head` instead of
                // four scalar loads -- was measured slower: 0.177 against 0.137 ms; the scalar form stays)
                // float4 number v = 32 it + j covers elements head + 128 it + 4 j .. + 3: row `it` of the staged tile for
                // j < 31, but the last one of each row straddles rows it and it + 1 when head > 0 -- its bank would collide
                // with lane 0's (a 2-way conflict on every load), so lane 31 sits out and the 31 seams go out afterwards,
                // seam `it` by lane `it` (banks it + 31 and it + 1: conflict-free)
                if (head == 0 || lane < 31) {
                    for (int v = lane; v < nv4; v += 32) {
                        const int l = head + 4 * v;
                        *reinterpret_cast<float4*>(g + l) = make_float4(at(l), at(l + 1), at(l + 2), at(l + 3));
                    }
                }
                if (head != 0 && 32 * lane + 31 < nv4) {
                    const int l = head + 4 * (32 * lane + 31);
                    *reinterpret_cast<float4*>(g + l) = make_float4(at(l), at(l + 1), at(l + 2), at(l + 3));
                }
                const int tail0 = head + 4 * nv4;
                if (tail0 + lane < run) g[tail0 + lane] = at(tail0 + lane);
            }
            __syncwarp();
            t.advance(FT_ACC);
        }
        if (prm.prof && q == 0 && lane == 0) { unsigned long long* pp = prm.prof + blockIdx.x * 16; pp[5] = FT_NOW() - pe_tot; pp[6] = pe_w; pp[7] = pe_s; }
    } else if (warp >= PROD_WARP0 && warp < PROD_WARP0 + N_PROD_WARPS) {
        // ============================ producers: fp32 -> bf16 hi / lo =========================
        // Two groups of four warps take alternate chunks (a chunk's tcgen05.st / barrier round trip overlaps the other
        // group's conversion; the ring depths are even, so a slot always belongs to one group); within a group warp pwl
        // converts rows 32 pwl .. +31 of the staged 128 x 32 block, ONE ROW PER LANE (= its lane of TMEM lane quarter
        // pwl = warp % 4): eight 16-byte loads from the 128-byte-swizzled row (a quarter warp covers all 32 banks),
        // 16 + 16 packed bf16x2 words, two tcgen05.st.
        const int pw = warp - PROD_WARP0;
        const uint32_t grp = (uint32_t)pw >> 2, pwl = (uint32_t)pw & 3u;
        static_assert(PROD_WARP0 % 4 == 0 && FT_KC == 32, "producer warp pwl owns TMEM lanes 32 pwl .. +31");
        const uint32_t in_lane = smem_u32(in_ring) + (pwl * 32u + (uint32_t)lane) * 128u, sw = (uint32_t)lane & 7u;
        const uint32_t a_t = tmem_base + ((pwl * 32u) << 16) + FT_A_COL0;
        RingPos in, a;
        uint32_t bf_phase = 0;
        long long pp_i = 0, pp_a = 0, pp_x, pp_tot = FT_NOW();
        uint32_t n_chunk = 0;
        for (int w = w_begin; w < w_end; ++w) {
            if (new_channel(w)) {
                mbar_wait(smem_u32(&ctl->b_free), bf_phase);
                bf_phase ^= 1u;
                build_b(w / prm.tiles_per_chan, pw * 32 + lane, N_PROD_WARPS * 32);
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&ctl->b_ready));          // all eight warps rebuild
            }
            for (int kc = 0; kc < n_kc; ++kc, ++n_chunk) {
                if ((n_chunk & 1u) != grp) { in.advance(n_in); a.advance(n_a); continue; }
                pp_x = FT_NOW(); mbar_wait(smem_u32(&ctl->in_full[in.idx]), in.phase); pp_i += FT_NOW() - pp_x;
                uint32_t hb[FT_A_COLS], lb[FT_A_COLS];
#pragma unroll
                for (int c = 0; c < 8; ++c) {
                    const float4 v = lds128f(in_lane + in.idx * FT_IN_SLOT + ((((uint32_t)c) ^ sw) << 4));
                    const __nv_bfloat162 h0 = __floats2bfloat162_rn(v.x, v.y), h1 = __floats2bfloat162_rn(v.z, v.w);
                    hb[2 * c] = *reinterpret_cast<const uint32_t*>(&h0);
                    hb[2 * c + 1] = *reinterpret_cast<const uint32_t*>(&h1);
                    const __nv_bfloat162 l0 = __floats2bfloat162_rn(v.x - __uint_as_float(hb[2 * c] << 16),
                                                                     v.y - __uint_as_float(hb[2 * c] & 0xffff0000u));
                    const __nv_bfloat162 l1 = __floats2bfloat162_rn(v.z - __uint_as_float(hb[2 * c + 1] << 16),
                                                                     v.w - __uint_as_float(hb[2 * c + 1] & 0xffff0000u));
                    lb[2 * c] = *reinterpret_cast<const uint32_t*>(&l0);
                    lb[2 * c + 1] = *reinterpret_cast<const uint32_t*>(&l1);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&ctl->in_empty[in.idx]));
                in.advance(n_in);
                pp_x = FT_NOW(); mbar_wait(smem_u32(&ctl->a_empty[a.idx]), a.phase ^ 1); pp_a += FT_NOW() - pp_x;
                tc_fence_after();
                if (!FT_DBG(1024)) {
                    tmem_st16(a_t + a.idx * (2 * FT_A_COLS), hb);
                    tmem_st16(a_t + a.idx * (2 * FT_A_COLS) + FT_A_COLS, lb);
                    tmem_st_wait();
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&ctl->a_full[a.idx]));
                a.advance(n_a);
            }
        }
        if (prm.prof && pw == 0 && lane == 0) { unsigned long long* pp = prm.prof + blockIdx.x * 16; pp[8] = FT_NOW() - pp_tot; pp[9] = pp_i; pp[10] = pp_a; }
    }

    tc_fence_before();
    cluster_sync();
    if (warp == ALLOC_WARP) tmem_dealloc<CG>(tmem_base, 512);
}

// true if this kernel handled the call (shared taps: taps [M]; per_channel: taps [C][M])
bool firt_fir(const float* x, const float* taps, float* y, int C, long long L, int M, bool per_channel, cudaStream_t st,
              tina_status* status)
{
    if (M > 193 || L % FT_T != 0 || L / FT_T > 0x7fffffffLL || options().fir_simt || options().fir_v1) return false;
    const long long Lo = L - M + 1;
    const int Kp = (FT_T + M - 1 + FT_KC - 1) / FT_KC * FT_KC;
    const int n_kc = Kp / FT_KC;
    const long long R = (Lo + FT_T - 1) / FT_T;                      // output blocks (A rows) per channel
    const long long tps = (R + BM * UMMA_CG - 1) / (BM * UMMA_CG);
    if (tps * C > 0x7fffffffLL) return false;
    DevCtx* ctx = nullptr;
    if ((*status = dev_ctx(&ctx)) != TINA_OK) return true;

    FirtParams prm;
    memset(&prm, 0, sizeof(prm));
    prm.taps = taps; prm.y = y; prm.Lo = Lo; prm.M = M; prm.n_kc = n_kc;
    prm.taps_stride = per_channel ? M : 0;
    prm.tiles_per_chan = (int)tps;
    prm.total_work = (int)(tps * C);
    prm.b_part_bytes = ((FT_T / UMMA_CG + FT_KC * (n_kc - 1)) * 64 + 1023) / 1024 * 1024;
    const size_t fixed = 2 * (size_t)prm.b_part_bytes + 4 * FT_STAGE + sizeof(FirtCtl);
    // Ring depths are EVEN: the two producer groups take alternate chunks, and a slot shared by both groups would let a
    // group test the parity of a barrier that is a whole phase behind (measured: a rare deadlock with a 3-slot ring).
    // Six slots of read-ahead (96 KB per SM), measured on c3: 2 -> 0.135 ms, 4 -> 0.107, 6 -> 0.1005, 8 -> 0.1095 (deeper
    // read-ahead lets the loads crowd the stores out at the memory controllers)
    prm.in_slots = 6;
    while (prm.in_slots > 2 && fixed + (size_t)prm.in_slots * FT_IN_SLOT > 232448) prm.in_slots -= 2;
    if (fixed + (size_t)prm.in_slots * FT_IN_SLOT > 232448) return false;
#ifdef TINA_DEV
    if (options().b_entries) prm.in_slots = options().b_entries;
    prm.debug = options().debug_skip;
#endif
    const size_t smem = fixed + (size_t)prm.in_slots * FT_IN_SLOT;

    EncodeTiledFn enc = encode_fn();
    if (!enc) { *status = fail(TINA_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found"); return true; }
    CUtensorMap tmap_x;
    memset(&tmap_x, 0, sizeof(tmap_x));
    {
        const cuuint32_t estr[3] = {1, 1, 1};
        const cuuint64_t dims[3] = {(cuuint64_t)FT_T, (cuuint64_t)(L / FT_T), (cuuint64_t)C};
        const cuuint64_t strides[2] = {(cuuint64_t)FT_T * sizeof(float), (cuuint64_t)L * sizeof(float)};
        const cuuint32_t box[3] = {FT_KC, BM, 1};
        CUresult r = enc(&tmap_x, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(x), dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                         CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) { *status = fail(TINA_ERR_CUDA, "cuTensorMapEncodeTiled(fir input) failed (%d)", (int)r); return true; }
    }
    if ((*status = ensure_smem(ctx, reinterpret_cast<const void*>(fir_umma_kernel), 232448, "cudaFuncSetAttribute(fir_umma_kernel)")) != TINA_OK)
        return true;
    const int n_cl = ctx->n_sm / UMMA_CG;
    const int grid = UMMA_CG * (prm.total_work < n_cl ? prm.total_work : n_cl);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(UMMA_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = UMMA_CG;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
#ifdef TINA_DEV
    const bool prof = options().prof;
    if (prof) {
        cudaError_t pe = cudaMalloc(&prm.prof, (size_t)grid * 16 * 8);
        if (pe == cudaSuccess) pe = cudaMemsetAsync(prm.prof, 0, (size_t)grid * 16 * 8, st);
        if (pe != cudaSuccess) { if (prm.prof) cudaFree(prm.prof); *status = check_cuda(pe, "TINA_PROF counter buffer"); return true; }
    }
#endif
    cudaError_t e = cudaLaunchKernelEx(&cfg, fir_umma_kernel, tmap_x, prm);
#ifdef TINA_DEV
    if (prof) {
        std::vector<unsigned long long> h((size_t)grid * 16);
        cudaError_t pe = cudaStreamSynchronize(st);
        if (pe == cudaSuccess) pe = cudaMemcpy(h.data(), prm.prof, h.size() * 8, cudaMemcpyDeviceToHost);
        cudaFree(prm.prof);
        if (pe != cudaSuccess) { *status = check_cuda(pe, "TINA_PROF counter read-back"); return true; }
        double acc[16] = {0};
        for (int b = 0; b < grid; b += UMMA_CG) for (int i = 0; i < 16; ++i) acc[i] += (double)h[(size_t)b * 16 + i] / (grid / UMMA_CG);
        fprintf(stderr, "[tina prof fir] leader mean cycles: tma tot %.0f in_empty %.0f | mma tot %.0f a_full %.0f t_empty %.0f | epi tot %.0f t_full %.0f tmem->smem %.0f | prod tot %.0f in_full %.0f a_empty %.0f\n",
                acc[0], acc[1], acc[2], acc[3], acc[4], acc[5], acc[6], acc[7], acc[8], acc[9], acc[10]);
    }
#endif
    count_launch();
    g_last_path = kPathUmma;
    note_kernel(per_channel ? "fir_umma_kernel<per-channel taps>" : "fir_umma_kernel");
    *status = e != cudaSuccess ? check_cuda(e, "fir_umma_kernel launch") : check_cuda(cudaGetLastError(), "fir_umma_kernel launch");
    return true;
}

}  // namespace tina
