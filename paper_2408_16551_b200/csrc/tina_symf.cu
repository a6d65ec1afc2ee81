// tina_symf.cu -- complex-kind fused PFB / DFT with every distinct ROW pair of the Fourier matrix contracted once as
// well (on top of the column pairing of tina_sym.cu).
//
// Eq. (12).  For the bins k in [0, P/2) the kernel of tina_sym.cu evaluates, with y = yr + i yi,
//     U = sum_p yr[p] cos(2 pi p k / P),  Z = sum_p yr[p] sin(2 pi p k / P),  W, V likewise from yi.
// The rows p and P - p of the cosine matrix are EQUAL and those of the sine matrix OPPOSITE, so with H = P / 2 and
//     a+[q] = y[q] + y[P - q],  a-[q] = y[q] - y[P - q]   (q = 1 .. H-1),   a+[0] = y[0],
//     U[k] = sum_{q < H} a+r[q] cos(2 pi q k / P) + (-1)^k yr[H],      Z[k] = sum_{0 < q < H} a-r[q] sin(2 pi q k / P):
// contraction length H instead of P and ONE matrix (cosine for U, sine for Z) per operand instead of [C | S]:
// 2 P^2 tensor flops per frame and product instead of 4 P^2 (8 P^2 in the plain block form).  It is still the dense
// contraction of Eq. (12)-(13): every output bin is an inner product against its own Fourier-matrix entries on the
// tensor cores, no factorisation of P; what is gone is the second evaluation of entries that differ only in sign.
// bench.py keeps counting 8 P^2 useful flops per frame and prints the issued count (issued / useful = 0.75 for bf16x3).
// The unpaired sample y[H] rides in the (otherwise empty) slot q = 0 of the a- operand: a "Csp" matrix whose only
// non-zero column is q = 0 with (-1)^k adds it to U (first chunk only).  The Nyquist bin X[H] = sum_q (-1)^q a+[q] + y[H]
// needs one more cosine column: 16 extra matrix rows "E" (one non-zero) ride in the cosine tiles and are contracted by
// an N = 16 instruction into the first 16 columns of the Z accumulator in pass 0 (Z[0] is identically zero, so its
// column is free; the other 15 rows are zero), where the sine matrix's row for bin 0 carries the 1 that adds y[H].
//
// Structure: as pfb_symt_kernel (CTA pair, tcgen05.mma.cta_group::2, M = 256, TMA-staged input window and taps,
// MN-major A tiles), with
//   chunk    = 16 folded elements q0 .. q0+15 = the input columns q0 .. q0+15 AND P-q0-15 .. P-q0 (two staged boxes)
//   producer = lane l < 16: column q0 + l, lane 16 + j: column P - q0 - j; FIR as before, then one shfl.xor 16 per value
//              and a+ (lanes < 16) / a- (lanes >= 16); operand tiles [r+ | r- | i+ | i-] x (hi, lo), 128 frames x 16
//   TMEM     = U | Z | W | V, 128 columns each; warp 13 issues the r products (U, Z), warp 15 the i products (W, V)
//   B ring   = per chunk the tiles S_hi, C_hi, [Csp_hi], C_lo, S_lo, [Csp_lo] (72 rows x 16 per CTA, SWIZZLE_32B)
#include "tina_sym.cuh"

#include <cstring>
#include <map>
#include <mutex>
#include <tuple>
#include <vector>

namespace tina {

using namespace ptx;

constexpr int SF_KQ = 16;                                  // folded contraction elements per chunk
constexpr int SF_TILE = BM * SF_KQ * 2;                    // 4 KB: 128 frames x 16 of bf16, MN-major SWIZZLE_128B
constexpr uint32_t SF_A_LBO = 2048, SF_A_SBO = 1024;       // bytes between the two 64-frame blocks / the two groups of 8 columns
constexpr int SF_A_RING = 64 * 1024;                       // 2 slots of 8 tiles (bf16x3) or 4 of 4 (single pass)
constexpr int SF_B_ROWS = 72;                              // rows per CTA and tile: 64 matrix rows + 8 rows of the E block
constexpr int SF_B_ENTRY = SF_B_ROWS * 32;                 // 2304 B: [72][16] bf16, K-major SWIZZLE_32B
constexpr int SF_B_ENTRIES = 16;
constexpr int SF_B_E_OFF = 64 * 32;                        // byte offset of the E rows in a cosine tile
constexpr int SF_IN_PITCH = 144;                           // staged row: 18 complex columns
constexpr int SF_TAP_PITCH = 80;                           // staged tap row: 20 floats
constexpr int SF_IN_MIR = 20608, SF_IN_TAPD = 41216, SF_IN_TAPM = 42496, SF_IN_SP = 43776;   // 128-byte aligned parts of a slot
constexpr int SF_IN_SLOT = 46080;
constexpr int SF_IN_SLOTS = 2;

struct SmemCtlF {
    uint64_t a_full[4], a_empty[4];
    uint64_t b_full[SF_B_ENTRIES], b_empty[SF_B_ENTRIES];
    uint64_t in_full[2], in_empty[2];
    uint64_t t_full[2], t_empty[2];
    uint32_t tmem_base;
};
// order: A ring | epilogue staging | B ring | input ring | barriers
constexpr size_t SF_SMEM_BYTES = SF_A_RING + 4 * SY_STAGE + SF_B_ENTRIES * SF_B_ENTRY + SF_IN_SLOTS * SF_IN_SLOT + sizeof(SmemCtlF);
static_assert(SF_SMEM_BYTES <= 232448, "exceeds the 227 KB shared memory opt-in limit");

// K-major operand, SWIZZLE_32B: rows of 32 B (16 bf16), 8-row groups of 256 B
__device__ __forceinline__ uint64_t smem_desc_sw32(uint32_t saddr)
{
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3FFFF) >> 4);
    d |= (uint64_t)1 << 16;
    d |= (uint64_t)(256 >> 4) << 32;
    d |= (uint64_t)1 << 46;
    d |= (uint64_t)6 << 61;                           // SWIZZLE_32B
    return d;
}

struct FoldMaps {
    CUtensorMap b72, b64;        // twiddle plan: boxes of 16 x 72 rows (cosine + E) and 16 x 64 rows (sine, Csp)
    CUtensorMap out, out2;       // output (as tina_sym.cu)
    CUtensorMap x, xsp, w;       // input: 36 floats x rows; 4 floats x rows (column P/2); window: 20 floats x MT rows
};

// plan row of (part, pass, block): CE blocks of 144 rows, S blocks of 128 rows, then the Csp blocks of 128 rows
__host__ __device__ inline int fold_row_ce(int npg, int rows_part, int part, int pass) { (void)npg; return part * rows_part + pass * 272; }
__host__ __device__ inline int fold_row_s(int npg, int rows_part, int part, int pass) { (void)npg; return part * rows_part + pass * 272 + 144; }
__host__ __device__ inline int fold_row_sp(int npg, int rows_part, int part, int pass) { return part * rows_part + npg * 272 + pass * 128; }

// Twiddle plan [parts][rows_part][H] (K-major: a row holds the folded index q).  Per pass (128 bins from k0):
//   CE block, per CTA r of the pair: 64 rows cos(2 pi q (k0 + 64 r + i) / P), then 8 rows E (pass 0, r = 0, first row:
//             (-1)^q, everything else 0);  S block: 64 rows per CTA of sin (inverse: -sin); column q = 0 of bin 0: 1;
//   Csp block: column q = 0: (-1)^k, other columns 0.      Bins >= P/2 are zero rows; 1/P is folded in for the inverse.
__global__ void twiddle_fold_kernel(__nv_bfloat16* __restrict__ tt, int P, int inverse, int parts, int fp16, int npg, int rows_part)
{
    const int H = P >> 1;
    const long long total = (long long)rows_part * H;
    const double scale = inverse ? 1.0 / (double)P : 1.0;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x) {
        const int row = (int)(e / H), q = (int)(e % H);
        double v = 0.0;
        // A pass has nb = min(128, H - k0) bins; with cta_group::2 the instruction takes the first nb / 2 rows of EACH
        // CTA's tile, so CTA r's tile holds the bins k0 + r nb / 2 + i (i < nb / 2), zero rows after them.
        if (row < npg * 272) {
            const int pass = row / 272, rr = row % 272, k0 = pass * SY_BINS;
            const int nb2 = min(SY_BINS, H - k0) / 2;
            if (rr < 144) {                                // CE: [C half 0 | E 0 | C half 1 | E 1]
                const int r = rr / 72, i = rr % 72;
                if (i < 64) {
                    if (i < nb2) { const int k = k0 + r * nb2 + i; double sn, cs; sincospi(2.0 * (double)(((long long)q * k) % P) / (double)P, &sn, &cs); v = cs; }
                } else if (pass == 0 && r == 0 && i == 64) v = (q & 1) ? -1.0 : 1.0;
            } else {                                       // S
                const int r = (rr - 144) / 64, i = (rr - 144) % 64;
                if (i < nb2) {
                    const int k = k0 + r * nb2 + i;
                    double sn, cs; sincospi(2.0 * (double)(((long long)q * k) % P) / (double)P, &sn, &cs);
                    v = inverse ? -sn : sn;
                    if (q == 0) v = (k == 0) ? ((H & 1) ? -1.0 : 1.0) : 0.0;   // y[P/2] rides in slot q = 0 of a-: Nyquist += (-1)^(P/2) y[P/2]
                }
            }
        } else {                                           // Csp
            const int pass = (row - npg * 272) / 128, rr = (row - npg * 272) % 128, k0 = pass * SY_BINS;
            const int nb2 = min(SY_BINS, H - k0) / 2, r = rr / 64, i = rr % 64;
            if (i < nb2 && q == 0) v = ((k0 + r * nb2 + i) & 1) ? -1.0 : 1.0;
        }
        v *= scale;
        if (fp16) { reinterpret_cast<__half*>(tt)[e] = __double2half(v); continue; }
        const __nv_bfloat16 hi = __double2bfloat16(v);
        tt[e] = hi;
        if (parts > 1) tt[total + e] = __double2bfloat16(v - (double)__bfloat162float(hi));
    }
}

template <int MT, int PARTS>
__global__ void __launch_bounds__(UMMA_THREADS, 1)
pfb_symf_kernel(const __grid_constant__ FoldMaps maps, const SymParams prm, const int rows_part)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    if ((smem_u32(smem) & 1023u) != 0) __trap();
    uint8_t* a_ring = smem;
    uint8_t* stage = smem + SF_A_RING;
    uint8_t* b_ring = stage + 4 * SY_STAGE;
    uint8_t* in_ring = b_ring + SF_B_ENTRIES * SF_B_ENTRY;
    SmemCtlF* ctl = reinterpret_cast<SmemCtlF*>(in_ring + SF_IN_SLOTS * SF_IN_SLOT);

    constexpr int CG = UMMA_CG;
    constexpr int WA = MT > 0 ? MT : 1;
    constexpr int IN_ROWS = BM + WA - 1;
    constexpr int parts = PARTS;
    constexpr uint32_t a_slot_bytes = 4u * parts * SF_TILE;            // [r+ | r- | i+ | i-] x (hi, lo)
    constexpr uint32_t n_a = (uint32_t)SF_A_RING / a_slot_bytes;       // 2 (bf16x3) or 4 (single pass)
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int P = prm.P, M = prm.M, H = P >> 1;
    const int n_kc = H / SF_KQ;
    const uint32_t rank = cluster_ctarank();
    constexpr uint32_t leader = 0;
    constexpr uint16_t pair_mask = 3;
    const int cl = blockIdx.x / CG, n_cl = gridDim.x / CG;
    const int npg = prm.n_passes;

    if (warp == TMA_WARP && lane == 0) {
        prefetch_tmap(&maps.b72); prefetch_tmap(&maps.b64); prefetch_tmap(&maps.out); prefetch_tmap(&maps.out2);
        prefetch_tmap(&maps.x); prefetch_tmap(&maps.xsp);
        if (MT > 0) prefetch_tmap(&maps.w);
        for (int i = 0; i < 4; ++i) { mbar_init(smem_u32(&ctl->a_full[i]), N_PROD_WARPS + (rank == 0 ? CG - 1 : 0)); mbar_init(smem_u32(&ctl->a_empty[i]), 2); }
        for (int i = 0; i < SF_B_ENTRIES; ++i) { mbar_init(smem_u32(&ctl->b_full[i]), 1); mbar_init(smem_u32(&ctl->b_empty[i]), 2); }
        for (int i = 0; i < SF_IN_SLOTS; ++i) { mbar_init(smem_u32(&ctl->in_full[i]), 1); mbar_init(smem_u32(&ctl->in_empty[i]), N_PROD_WARPS); }
        for (int i = 0; i < 2; ++i) { mbar_init(smem_u32(&ctl->t_full[i]), 1); mbar_init(smem_u32(&ctl->t_empty[i]), 4 * CG); }
        fence_mbar_init();
    }
    if (warp == ALLOC_WARP) {
        tmem_alloc<CG>(smem_u32(&ctl->tmem_base), 512);
        tmem_relinquish<CG>();
    }
    tc_fence_before();
    cluster_sync();
    tc_fence_after();
    const uint32_t tmem_base = ctl->tmem_base;

    if (warp == ALLOC_WARP) {
        // ============================ TMA producer: input rows + taps ========================
        if (lane == 0) {
            RingPos in;
            for (int w = cl; w < prm.total_work; w += n_cl) {
                const int tile = w / npg;
                const int s = tile / prm.tiles_per_stream;
                const int r0 = (tile % prm.tiles_per_stream) * (BM * CG) + (int)rank * BM + M - WA;
                for (int kc = 0; kc < n_kc; ++kc) {
                    const int q0 = kc * SF_KQ;
                    mbar_wait<64>(smem_u32(&ctl->in_empty[in.idx]), in.phase ^ 1);
                    const uint32_t bar = smem_u32(&ctl->in_full[in.idx]);
                    const uint32_t dst = smem_u32(in_ring + in.idx * SF_IN_SLOT);
                    uint32_t bytes = 2u * IN_ROWS * SF_IN_PITCH + (MT > 0 ? 2u * MT * SF_TAP_PITCH : 0u);
                    if (kc == 0) bytes += (uint32_t)IN_ROWS * 16u;
                    mbar_expect_tx(bar, bytes);
                    // columns q0 .. q0+17 and P-q0-16 .. P-q0+1 (columns >= P arrive as zeros: y[P] = 0 pairs with y[0])
                    tma_load_3d(dst, &maps.x, bar, 2 * q0, r0, s);
                    tma_load_3d(dst + SF_IN_MIR, &maps.x, bar, 2 * (P - q0 - 16), r0, s);
                    if (MT > 0) {
                        tma_load_2d(dst + SF_IN_TAPD, &maps.w, bar, q0, 0);
                        tma_load_2d(dst + SF_IN_TAPM, &maps.w, bar, P - q0 - 16, 0);
                    }
                    if (kc == 0) tma_load_3d(dst + SF_IN_SP, &maps.xsp, bar, 2 * H, r0, s);   // the unpaired column P/2
                    in.advance(SF_IN_SLOTS);
                }
            }
        }
    } else if (warp == TMA_WARP) {
        // ============================ TMA producer: twiddle tiles ============================
        if (lane == 0) {
            RingPos b;
            auto put = [&](const CUtensorMap* map, uint32_t box_bytes, int col, int row) {
                mbar_wait<64>(smem_u32(&ctl->b_empty[b.idx]), b.phase ^ 1);
                const uint32_t bar = smem_u32(&ctl->b_full[b.idx]);
                if (rank == 0) mbar_expect_tx(bar, 2 * box_bytes);
                tma_load_2d_cg2(smem_u32(b_ring + b.idx * SF_B_ENTRY), map, mapa_u32(bar, leader), col, row);
                b.advance(SF_B_ENTRIES);
            };
            for (int w = cl; w < prm.total_work; w += n_cl) {
                const int pass = w % npg;
                for (int kc = 0; kc < n_kc; ++kc) {
                    const int q0 = kc * SF_KQ;
                    // order of use: S_hi, C_hi, [Csp_hi], C_lo, S_lo, [Csp_lo]
                    put(&maps.b64, 64 * 32, q0, fold_row_s(npg, rows_part, 0, pass) + (int)rank * 64);
                    put(&maps.b72, 72 * 32, q0, fold_row_ce(npg, rows_part, 0, pass) + (int)rank * 72);
                    if (kc == 0) put(&maps.b64, 64 * 32, q0, fold_row_sp(npg, rows_part, 0, pass) + (int)rank * 64);
                    if (parts > 1) {
                        put(&maps.b72, 72 * 32, q0, fold_row_ce(npg, rows_part, 1, pass) + (int)rank * 72);
                        put(&maps.b64, 64 * 32, q0, fold_row_s(npg, rows_part, 1, pass) + (int)rank * 64);
                        if (kc == 0) put(&maps.b64, 64 * 32, q0, fold_row_sp(npg, rows_part, 1, pass) + (int)rank * 64);
                    }
                }
            }
        }
    } else if (warp == MMA_WARP || warp == MMA_WARP2) {
        // ============================ MMA issuers ===========================================
        // warp 13 (h = 0): the r operand -> U (columns 0-127) and Z (128-255); warp 15 (h = 1): the i operand -> W, V.
        const int h = warp == MMA_WARP ? 0 : 1;
        if (rank != 0 && h == 0) {
            RingPos a;
            for (int w = cl; w < prm.total_work; w += n_cl)
                for (int kc = 0; kc < n_kc; ++kc) {
                    mbar_wait(smem_u32(&ctl->a_full[a.idx]), a.phase);
                    if (lane == 0) mbar_arrive_cluster(smem_u32(&ctl->a_full[a.idx]), leader);
                    __syncwarp();
                    a.advance(n_a);
                }
        }
        if (rank == 0) {
            RingPos a, b;
            uint32_t te_phase = 0;
            const uint32_t d_cos = tmem_base + (uint32_t)h * 256u, d_sin = d_cos + 128u;
            for (int w = cl; w < prm.total_work; w += n_cl) {
                const int pass = w % npg;
                const int k0 = pass * SY_BINS;
                const int nb = min(SY_BINS, H - k0);
                const uint32_t idesc_n = idesc_bf16(BM * CG, nb, prm.fp16 != 0) | IDESC_A_MN_MAJOR;
                const uint32_t idesc_e = idesc_bf16(BM * CG, 16, prm.fp16 != 0) | IDESC_A_MN_MAJOR;
                for (int ks = 0; ks < prm.k_splits; ++ks) {
                    const int kc_begin = ks * prm.kc_per_split, kc_end = min(n_kc, kc_begin + prm.kc_per_split);
                    for (int kc = kc_begin; kc < kc_end; ++kc) {
                        mbar_wait(smem_u32(&ctl->a_full[a.idx]), a.phase);
                        tc_fence_after();
                        // tiles of this operand in the slot: [+hi, +lo, -hi, -lo] (single pass: [+, -])
                        const uint32_t t0 = smem_u32(a_ring + a.idx * a_slot_bytes) + (uint32_t)h * 2u * parts * SF_TILE;
                        const uint64_t a_ph = smem_desc_mn_sw128(t0, SF_A_LBO, SF_A_SBO);
                        const uint64_t a_pl = smem_desc_mn_sw128(t0 + SF_TILE, SF_A_LBO, SF_A_SBO);
                        const uint64_t a_mh = smem_desc_mn_sw128(t0 + parts * SF_TILE, SF_A_LBO, SF_A_SBO);
                        const uint64_t a_ml = smem_desc_mn_sw128(t0 + (parts + 1) * SF_TILE, SF_A_LBO, SF_A_SBO);
                        if (kc == kc_begin) {
                            mbar_wait(smem_u32(&ctl->t_empty[h]), te_phase ^ 1u);
                            te_phase ^= 1u;
                            tc_fence_after();
                        }
                        const uint32_t acc0 = kc > kc_begin;
                        // one twiddle tile: wait, issue (lane 0), hand it back
                        auto with_entry = [&](auto&& issue) {
                            mbar_wait(smem_u32(&ctl->b_full[b.idx]), b.phase);
                            tc_fence_after();
                            if (elect_one()) {
                                issue(smem_u32(b_ring + b.idx * SF_B_ENTRY));
                                commit_cg<CG>(smem_u32(&ctl->b_empty[b.idx]), pair_mask);
                            }
                            __syncwarp();
                            b.advance(SF_B_ENTRIES);
                        };
                        // S_hi: Z (+)= a-lo S_hi + a-hi S_hi
                        with_entry([&](uint32_t bt) {
                            const uint64_t bd = smem_desc_sw32(bt);
                            uint32_t acc = acc0;
                            if (parts > 1) { umma_bf16<CG>(d_sin, a_ml, bd, idesc_n, acc); acc = 1; }
                            umma_bf16<CG>(d_sin, a_mh, bd, idesc_n, acc);
                        });
                        // C_hi: U (+)= a+lo C_hi + a+hi C_hi;  pass 0: the E rows -> first 16 columns of Z (Nyquist in column 0)
                        with_entry([&](uint32_t bt) {
                            const uint64_t bd = smem_desc_sw32(bt);
                            uint32_t acc = acc0;
                            if (parts > 1) { umma_bf16<CG>(d_cos, a_pl, bd, idesc_n, acc); acc = 1; }
                            umma_bf16<CG>(d_cos, a_ph, bd, idesc_n, acc);
                            if (pass == 0) {
                                const uint64_t be = smem_desc_sw32(bt + SF_B_E_OFF);
                                if (parts > 1) umma_bf16<CG>(d_sin, a_pl, be, idesc_e, 1);
                                umma_bf16<CG>(d_sin, a_ph, be, idesc_e, 1);
                            }
                        });
                        // first chunk: Csp_hi: U += (a-lo + a-hi) Csp_hi (only slot q = 0 = y[P/2] is met by a non-zero entry)
                        if (kc == 0) with_entry([&](uint32_t bt) {
                            const uint64_t bd = smem_desc_sw32(bt);
                            if (parts > 1) umma_bf16<CG>(d_cos, a_ml, bd, idesc_n, 1);
                            umma_bf16<CG>(d_cos, a_mh, bd, idesc_n, 1);
                        });
                        if (parts > 1) {
                            with_entry([&](uint32_t bt) {                       // C_lo
                                const uint64_t bd = smem_desc_sw32(bt);
                                umma_bf16<CG>(d_cos, a_ph, bd, idesc_n, 1);
                                if (pass == 0) umma_bf16<CG>(d_sin, a_ph, smem_desc_sw32(bt + SF_B_E_OFF), idesc_e, 1);
                            });
                            with_entry([&](uint32_t bt) { umma_bf16<CG>(d_sin, a_mh, smem_desc_sw32(bt), idesc_n, 1); });   // S_lo
                            if (kc == 0) with_entry([&](uint32_t bt) { umma_bf16<CG>(d_cos, a_mh, smem_desc_sw32(bt), idesc_n, 1); });   // Csp_lo
                        }
                        if (elect_one()) {
                            commit_cg<CG>(smem_u32(&ctl->a_empty[a.idx]), pair_mask);
                            if (kc == kc_end - 1) commit_cg<CG>(smem_u32(&ctl->t_full[h]), pair_mask);
                        }
                        __syncwarp();
                        a.advance(n_a);
                    }
                }
            }
        }
    } else if (warp >= EPI_WARP0 && warp < EPI_WARP0 + 4) {
        EpiCtx ec;
        ec.t_full0 = smem_u32(&ctl->t_full[0]); ec.t_full1 = smem_u32(&ctl->t_full[1]);
        ec.t_empty0 = smem_u32(&ctl->t_empty[0]); ec.t_empty1 = smem_u32(&ctl->t_empty[1]);
        ec.stage = smem_u32(stage); ec.tmem_base = tmem_base; ec.rank = rank; ec.cl = cl; ec.n_cl = n_cl;
        sym_epilogue<true>(prm, &maps.out, &maps.out2, ec, warp - EPI_WARP0, lane);
    } else if (warp >= PROD_WARP0 && warp < PROD_WARP0 + N_PROD_WARPS) {
        // ============================ FIR producers =========================================
        // Warp pw owns frames 16 pw .. +15.  Lane l < 16: column q0 + l (staged box 0, index l); lane 16 + j: column
        // P - q0 - j (staged box 1, index 16 - j); first chunk, lane 16: the unpaired column P/2 (its own little box).
        const int pw = warp - PROD_WARP0;
        const uint32_t a_ring_s = smem_u32(a_ring), in_ring_s = smem_u32(in_ring);
        const uint32_t role = (uint32_t)lane >> 4, kq = (uint32_t)lane & 15u;
        const uint32_t kg = kq >> 3, kr = kq & 7u;
        uint32_t cell0[FPW / 8];
#pragma unroll
        for (int j = 0; j < FPW / 8; ++j)
            cell0[j] = a_ring_s + role * (uint32_t)parts * SF_TILE + (uint32_t)(pw >> 2) * SF_A_LBO + kg * SF_A_SBO + kr * 128u +
                       (((2u * ((uint32_t)pw & 3u) + (uint32_t)j) ^ kr) << 4);
        constexpr uint32_t im_off = 2u * parts * SF_TILE;
        const uint32_t idx = role ? 16u - kq : kq;
        const uint32_t in_lane = in_ring_s + (role ? (uint32_t)SF_IN_MIR : 0u) + (uint32_t)(pw * FPW) * SF_IN_PITCH + idx * 8u;
        const uint32_t tap_lane = in_ring_s + (role ? (uint32_t)SF_IN_TAPM : (uint32_t)SF_IN_TAPD) + idx * 4u;
        const uint32_t sp_lane = in_ring_s + SF_IN_SP + (uint32_t)(pw * FPW) * 16u;
        RingPos in, a;
        for (int w = cl; w < prm.total_work; w += n_cl)
            for (int kc = 0; kc < n_kc; ++kc) {
                const bool special = kc == 0 && lane == 16;           // this lane filters column P/2 in this chunk
                mbar_wait(smem_u32(&ctl->in_full[in.idx]), in.phase);
                float2 tap[WA], row[WA - 1 + FPW];
                {
                    const uint32_t so_in = in.idx * SF_IN_SLOT;
                    if (MT > 0) {
#pragma unroll
                        for (int m = 0; m < WA; ++m) { const float hh = lds_f1(tap_lane + so_in + (uint32_t)m * SF_TAP_PITCH); tap[m] = make_float2(hh, hh); }
                    }
                    if (kc == 0) {                                   // (warp-uniform) lane 16 reads its own little box and taps
                        const uint32_t src = special ? sp_lane + so_in : in_lane + so_in;
                        const uint32_t pitch = special ? 16u : (uint32_t)SF_IN_PITCH;
#pragma unroll
                        for (int j = 0; j < WA - 1 + FPW; ++j) row[j] = lds_f2(src + (uint32_t)j * pitch);
                        if (MT > 0 && special) {
#pragma unroll
                            for (int m = 0; m < WA; ++m) { const float hh = m < M ? __ldg(prm.window + (long long)m * P + H) : 0.f; tap[m] = make_float2(hh, hh); }
                        }
                    } else {
#pragma unroll
                        for (int j = 0; j < WA - 1 + FPW; ++j) row[j] = lds_f2(in_lane + so_in + (uint32_t)j * SF_IN_PITCH);
                    }
                }
                mbar_wait(smem_u32(&ctl->a_empty[a.idx]), a.phase ^ 1);
                const uint32_t so = a.idx * a_slot_bytes;
                // a = co * own + cp * partner: a+ = y[q] + y[P-q] (lanes < 16), a- = y[q] - y[P-q] (lanes >= 16: own is
                // y[P-q]); first chunk: lane 0 keeps y[0] alone and lane 16 carries y[P/2] in the empty slot q = 0 of a-
                const float co = (role && !special) ? -1.f : 1.f;
                const float cp = (kc == 0 && kq == 0) ? 0.f : 1.f;
                auto pack2 = [&](float a0, float a1) -> uint32_t {
                    if (parts == 1 && prm.fp16) { const __half2 hh = __floats2half2_rn(a0, a1); return *reinterpret_cast<const uint32_t*>(&hh); }
                    const __nv_bfloat162 hb = __floats2bfloat162_rn(a0, a1);
                    return *reinterpret_cast<const uint32_t*>(&hb);
                };
#pragma unroll
                for (int j = 0; j < FPW / 8; ++j) {
                    float2 yv[8];
                    if (MT > 1) {
#pragma unroll
                        for (int g = 0; g < 8; ++g) yv[g] = fmul2(tap[0], row[8 * j + g + WA - 1]);
#pragma unroll
                        for (int m = 1; m < WA; ++m)
#pragma unroll
                            for (int g = 0; g < 8; ++g) yv[g] = ffma2(tap[m], row[8 * j + g + WA - 1 - m], yv[g]);
                    } else {
#pragma unroll
                        for (int g = 0; g < 8; ++g) yv[g] = MT == 1 ? fmul2(tap[0], row[8 * j + g]) : row[8 * j + g];
                    }
                    if (kc == 0) {                                   // (warp-uniform) the general form, for the two unpaired samples
#pragma unroll
                        for (int g = 0; g < 8; ++g) {
                            const float px = __shfl_xor_sync(0xffffffffu, yv[g].x, 16), py = __shfl_xor_sync(0xffffffffu, yv[g].y, 16);
                            yv[g].x = fmaf(cp, px, co * yv[g].x);
                            yv[g].y = fmaf(cp, py, co * yv[g].y);
                        }
                    } else {
#pragma unroll
                        for (int g = 0; g < 8; ++g) {
                            const float px = __shfl_xor_sync(0xffffffffu, yv[g].x, 16), py = __shfl_xor_sync(0xffffffffu, yv[g].y, 16);
                            yv[g].x = fmaf(co, yv[g].x, px);
                            yv[g].y = fmaf(co, yv[g].y, py);
                        }
                    }
                    uint32_t hr[4], hi[4];
#pragma unroll
                    for (int q = 0; q < 4; ++q) { hr[q] = pack2(yv[2 * q].x, yv[2 * q + 1].x); hi[q] = pack2(yv[2 * q].y, yv[2 * q + 1].y); }
                    const uint32_t addr = cell0[j] + so;
                    sts128(addr, hr[0], hr[1], hr[2], hr[3]);
                    sts128(addr + im_off, hi[0], hi[1], hi[2], hi[3]);
                    if (parts > 1) {
                        uint32_t lr[4], li[4];
#pragma unroll
                        for (int q = 0; q < 4; ++q) {
                            lr[q] = pack2(yv[2 * q].x - __uint_as_float(hr[q] << 16), yv[2 * q + 1].x - __uint_as_float(hr[q] & 0xffff0000u));
                            li[q] = pack2(yv[2 * q].y - __uint_as_float(hi[q] << 16), yv[2 * q + 1].y - __uint_as_float(hi[q] & 0xffff0000u));
                        }
                        sts128(addr + SF_TILE, lr[0], lr[1], lr[2], lr[3]);
                        sts128(addr + im_off + SF_TILE, li[0], li[1], li[2], li[3]);
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&ctl->in_empty[in.idx]));
                in.advance(SF_IN_SLOTS);
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&ctl->a_full[a.idx]));
                a.advance(n_a);
            }
    }

    tc_fence_before();
    cluster_sync();
    if (warp == ALLOC_WARP) tmem_dealloc<CG>(tmem_base, 512);
}

// =====================================================================================
// Host side
// =====================================================================================
namespace {

struct FoldPlan { __nv_bfloat16* tt = nullptr; CUtensorMap b72, b64; int rows_part = 0, npg = 0; };
using FoldKey = std::tuple<int, int, int, int, int>;      // device, P, inverse, parts, fp16
std::mutex g_fold_mu;
std::map<FoldKey, FoldPlan> g_fold_plans;

tina_status get_fold_plan(int P, bool inverse, int parts, bool fp16, cudaStream_t st, const FoldPlan** out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return check_cuda(e, "cudaGetDevice");
    std::lock_guard<std::mutex> lk(g_fold_mu);
    const FoldKey key{dev, P, inverse ? 1 : 0, parts, fp16 ? 1 : 0};
    auto it = g_fold_plans.find(key);
    if (it != g_fold_plans.end()) { *out = &it->second; return TINA_OK; }
    const int H = P / 2;
    FoldPlan pl;
    pl.npg = (H + SY_BINS - 1) / SY_BINS;
    pl.rows_part = pl.npg * (272 + 128);
    const size_t bytes = (size_t)parts * pl.rows_part * H * sizeof(__nv_bfloat16);
    e = cudaMalloc(&pl.tt, bytes);
    if (e != cudaSuccess) return check_cuda(e, "cudaMalloc(folded twiddles)");
    twiddle_fold_kernel<<<592, 256, 0, st>>>(pl.tt, P, inverse ? 1 : 0, parts, fp16 ? 1 : 0, pl.npg, pl.rows_part);
    count_launch();
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { cudaFree(pl.tt); return check_cuda(e, "twiddle_fold_kernel"); }
    EncodeTiledFn enc = encode_fn();
    if (!enc) { cudaFree(pl.tt); return fail(TINA_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found"); }
    const cuuint64_t dims[2] = {(cuuint64_t)H, (cuuint64_t)parts * pl.rows_part};
    const cuuint64_t strides[1] = {(cuuint64_t)H * sizeof(__nv_bfloat16)};
    const cuuint32_t estr[2] = {1, 1};
    const CUtensorMapDataType dt = fp16 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT16 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16;
    const cuuint32_t box72[2] = {SF_KQ, SF_B_ROWS}, box64[2] = {SF_KQ, 64};
    CUresult r = enc(&pl.b72, dt, 2, pl.tt, dims, strides, box72, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_32B,
                     CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r == CUDA_SUCCESS)
        r = enc(&pl.b64, dt, 2, pl.tt, dims, strides, box64, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_32B,
                CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { cudaFree(pl.tt); return fail(TINA_ERR_CUDA, "cuTensorMapEncodeTiled(folded twiddles) failed (%d)", (int)r); }
    auto ins = g_fold_plans.emplace(key, pl);
    *out = &ins.first->second;
    return TINA_OK;
}

template <int MT, int PARTS>
tina_status launch_symf(DevCtx* ctx, const FoldMaps& maps, const SymParams& prm, int rows_part, int grid, cudaStream_t st)
{
    auto kern = pfb_symf_kernel<MT, PARTS>;
    tina_status as = ensure_smem(ctx, reinterpret_cast<const void*>(kern), (int)SF_SMEM_BYTES, "cudaFuncSetAttribute(pfb_symf_kernel)");
    if (as != TINA_OK) return as;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(UMMA_THREADS);
    cfg.dynamicSmemBytes = SF_SMEM_BYTES;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = UMMA_CG;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    cudaError_t e = cudaLaunchKernelEx(&cfg, kern, maps, prm, rows_part);
    count_launch();
    g_last_path = kPathUmma;
    note_kernel("pfb_symf_kernel", 0.25);
    if (e != cudaSuccess) return check_cuda(e, "pfb_symf_kernel launch");
    return check_cuda(cudaGetLastError(), "pfb_symf_kernel launch");
}

}  // namespace

void symf_clear_plans()
{
    std::lock_guard<std::mutex> lk(g_fold_mu);
    for (auto& kv : g_fold_plans) cudaFree(kv.second.tt);
    g_fold_plans.clear();
}

bool symf_supported(int P, int M, bool has_window) { return P >= 64 && P <= kMaxP && P % 64 == 0 && (!has_window || M <= 16); }

// complex kind, P % 64 == 0, window == nullptr (DFT batch) or M <= 16
tina_status symf_pfb(const void* x, int S, long long n_samples, int P, int M, const float* window, bool inverse,
                     tina_precision prec, void* out, cudaStream_t st)
{
    const long long NBLK = n_samples / P;
    const long long F = NBLK - M + 1;
    const int parts = prec == TINA_PREC_FP32 ? 2 : 1;
    const bool fp16 = prec == TINA_PREC_FP16;
    const FoldPlan* plan = nullptr;
    tina_status ps = get_fold_plan(P, inverse, parts, fp16, st, &plan);
    if (ps != TINA_OK) return ps;
    DevCtx* ctx = nullptr;
    if ((ps = dev_ctx(&ctx)) != TINA_OK) return ps;
    const int H = P / 2;

    SymParams prm;
    memset(&prm, 0, sizeof(prm));
    prm.x = static_cast<const float*>(x);
    prm.window = window;
    prm.out = static_cast<float*>(out);
    prm.stream_stride = 2 * n_samples;
    prm.F = F;
    prm.NBLK = NBLK;
    prm.P = P;
    prm.M = M;
    prm.tiles_per_stream = (int)((F + BM * UMMA_CG - 1) / (BM * UMMA_CG));
    prm.n_passes = plan->npg;
    const long long total = (long long)S * prm.tiles_per_stream * prm.n_passes;
    if (total > 0x7fffffffLL) return fail(TINA_ERR_UNSUPPORTED, "tina_pfb: too many tiles");
    prm.total_work = (int)total;
    prm.parts = parts;
    prm.fp16 = fp16 ? 1 : 0;
    prm.k_splits = (H + KSPLIT_MAX - 1) / KSPLIT_MAX;          // accumulation chains of <= 1024
    prm.kc_per_split = ((H / SF_KQ) + prm.k_splits - 1) / prm.k_splits;
    prm.debug = options().debug_skip;
    const int n_cl = ctx->n_sm / UMMA_CG;
    const int grid = UMMA_CG * (prm.total_work < n_cl ? prm.total_work : n_cl);

    EncodeTiledFn enc = encode_fn();
    if (!enc) return fail(TINA_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found");
    const cuuint32_t estr[3] = {1, 1, 1};
    FoldMaps maps;
    memset(&maps, 0, sizeof(maps));
    maps.b72 = plan->b72; maps.b64 = plan->b64;
    const int MT = !window ? 0 : (M <= 4 ? 4 : (M <= 8 ? 8 : 16));
    static_assert(sizeof(CUtensorMap) == 128, "TmapSet layout");
    // five maps per call (out, out2, x, xsp, w): two cache entries
    TmapKey tkey;
    memset(&tkey, 0, sizeof(tkey));
    tkey.p[0] = x; tkey.p[1] = window; tkey.p[2] = out;
    tkey.n[0] = n_samples;
    tkey.i[0] = S; tkey.i[1] = P; tkey.i[2] = M; tkey.i[5] = 7;      // tag 7: symf_pfb, first set
    TmapKey tkey2 = tkey; tkey2.i[5] = 8;
    TmapSet t1, t2;
    if (tmap_cache_get(ctx, tkey, &t1) && tmap_cache_get(ctx, tkey2, &t2)) {
        memcpy(&maps.out, t1.m[0], 128); memcpy(&maps.out2, t1.m[1], 128); memcpy(&maps.x, t1.m[2], 128); memcpy(&maps.xsp, t1.m[3], 128);
        memcpy(&maps.w, t2.m[0], 128);
    } else {
        const cuuint64_t dims[3] = {(cuuint64_t)2 * P, (cuuint64_t)F, (cuuint64_t)S};
        const cuuint64_t strides[2] = {(cuuint64_t)2 * P * sizeof(float), (cuuint64_t)F * 2 * P * sizeof(float)};
        const cuuint32_t box[3] = {32, 32, 1}, box2[3] = {28, 32, 1};
        CUresult r = enc(&maps.out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, out, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                         CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r == CUDA_SUCCESS)
            r = enc(&maps.out2, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, out, dims, strides, box2, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        const cuuint64_t xdims[3] = {(cuuint64_t)2 * P, (cuuint64_t)NBLK, (cuuint64_t)S};
        const cuuint64_t xstrides[2] = {(cuuint64_t)2 * P * sizeof(float),
                                        S > 1 ? (cuuint64_t)prm.stream_stride * sizeof(float) : (cuuint64_t)NBLK * 2 * P * sizeof(float)};
        const cuuint32_t rows = (cuuint32_t)(BM + (MT > 0 ? MT : 1) - 1);
        const cuuint32_t xbox[3] = {36, rows, 1}, spbox[3] = {4, rows, 1};
        if (r == CUDA_SUCCESS)
            r = enc(&maps.x, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<void*>(x), xdims, xstrides, xbox, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r == CUDA_SUCCESS)
            r = enc(&maps.xsp, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<void*>(x), xdims, xstrides, spbox, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r == CUDA_SUCCESS && MT > 0) {
            const cuuint64_t wdims[2] = {(cuuint64_t)P, (cuuint64_t)M};
            const cuuint64_t wstrides[1] = {(cuuint64_t)P * sizeof(float)};
            const cuuint32_t wbox[2] = {20, (cuuint32_t)MT};
            r = enc(&maps.w, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float*>(window), wdims, wstrides, wbox, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        }
        if (r != CUDA_SUCCESS) return fail(TINA_ERR_CUDA, "cuTensorMapEncodeTiled(pfb_symf_kernel) failed (%d)", (int)r);
        memcpy(t1.m[0], &maps.out, 128); memcpy(t1.m[1], &maps.out2, 128); memcpy(t1.m[2], &maps.x, 128); memcpy(t1.m[3], &maps.xsp, 128);
        memset(&t2, 0, sizeof(t2)); memcpy(t2.m[0], &maps.w, 128);
        tmap_cache_put(ctx, tkey, t1); tmap_cache_put(ctx, tkey2, t2);
    }
#define TINA_SYMF(MT_) (parts == 2 ? launch_symf<MT_, 2>(ctx, maps, prm, plan->rows_part, grid, st) \
                                   : launch_symf<MT_, 1>(ctx, maps, prm, plan->rows_part, grid, st))
    if (MT == 0) return TINA_SYMF(0);
    if (MT == 4) return TINA_SYMF(4);
    if (MT == 8) return TINA_SYMF(8);
    return TINA_SYMF(16);
#undef TINA_SYMF
}

}  // namespace tina
