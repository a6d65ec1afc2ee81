// tina_sym.cu -- the fused PFB / DFT kernel for the COMPLEX kind with every distinct column pair of the
// Fourier matrix contracted once.
//
// Eq. (12) for a complex frame y = yr + i yi and the bins k and P-k:
//     X[k]   = sum_p y[p] (c - i s),   X[P-k] = sum_p y[p] (c + i s),   c = cos(2 pi p k / P), s = sin(2 pi p k / P)
// The two bins share the four real sums
//     U = sum_p yr c,   V = sum_p yi s,   W = sum_p yi c,   Z = sum_p yr s
//     X[k] = (U + V) + i (W - Z),        X[P-k] = (U - V) + i (W + Z)
// so the dense contraction against the P x P Fourier matrix needs the real products  yr * [C | S]  and
// yi * [C | S]  for k in [0, P/2) only: 4 P^2 tensor flops per frame and pass instead of the 8 P^2 of the real
// 2P x 2P block form (tina_umma.cu), half the twiddle bytes, and contraction length P instead of 2P (one
// accumulation chain at P = 1024).  It is still the dense contraction of Eq. (12)-(13) -- no factorisation of P;
// bench.py keeps counting 8 P^2 useful flops and reports the issued count.  Bin 0 has s = 0, so its sine column
// carries (-1)^p instead and delivers the unpaired Nyquist bin X[P/2].
//
// Structure (same roles as tina_umma.cu; CTA pair, tcgen05.mma.cta_group::2, M = 256):
//   A slot   = [yr hi | yr lo | yi hi | yi lo], 128 frames x 64 contraction elements each (bf16, K-major
//              SWIZZLE_128B): the FIR producers de-interleave the complex samples with 16-bit stores
//   B entry  = 64 contraction elements x 256 matrix rows (128 bins x (cos, sin)), half per CTA, hi / lo
//   TMEM     = D1 (columns 0-255) = yr * [C|S] = (U, Z) per bin,  D2 (columns 256-511) = yi * [C|S] = (W, V)
//   MMA      = warp 13 issues the yr products into D1, warp 15 the yi products into D2, against the SAME B entry
//   epilogue = tcgen05.ld of 16 bins from D1 and D2, the +- combine in registers, a forward 32 x 32 staging
//              tile (bins k ..) and a mirrored one (the aligned group of bins P-k-16 .., in reverse), both stored by TMA
#include "tina_sym.cuh"

#include <cstring>
#include <vector>

namespace tina {

using namespace ptx;

// Polyphase MAC of the FPW frames held in registers (as fir_compute_store), the complex result DE-INTERLEAVED:
// real parts into the yr tiles, imaginary parts into the yi tiles, each split into bf16 hi / lo.
// `cell` = byte offset (in a 16 KB tile) of this lane's 2-byte cell in row 0 of the warp's slab for each swizzle
// phase; tile order in the slot: [yr hi | yr lo | yi hi | yi lo] (single pass: [yr | yi]).
template <int MT, bool SPLIT>
__device__ __forceinline__ void fir_compute_store_sym(const FirRegs<MT>& rg, const uint32_t (&cell)[8], bool fp16)
{
    // cell[j]: shared-memory address of this lane's 2-byte cell in row 0 of the warp's slab of the yr hi tile, for
    // swizzle phase j (slot base, sub-step and lane already folded in): everything below is an immediate offset
    constexpr int WA = FirRegs<MT>::WA;
    constexpr int FG = 8;
    constexpr uint32_t im_off = SPLIT ? 2u * A_PART_BYTES : (uint32_t)A_PART_BYTES;
    constexpr bool split = SPLIT;
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
            if (!SPLIT && fp16) { const __half2 hh = __floats2half2_rn(y[g].x, y[g].y); hb = *reinterpret_cast<const uint32_t*>(&hh); }
            else { const __nv_bfloat162 hi = __floats2bfloat162_rn(y[g].x, y[g].y); hb = *reinterpret_cast<const uint32_t*>(&hi); }
            const uint32_t addr = cell[i & 7] + (uint32_t)i * 128u;
            sts16(addr, hb);
            sts16(addr + im_off, hb >> 16);
            if (split) {
                const float lx = y[g].x - __uint_as_float(hb << 16);
                const float ly = y[g].y - __uint_as_float(hb & 0xffff0000u);
                const __nv_bfloat162 lo = __floats2bfloat162_rn(lx, ly);
                const uint32_t lb = *reinterpret_cast<const uint32_t*>(&lo);
                sts16(addr + A_PART_BYTES, lb);
                sts16(addr + im_off + A_PART_BYTES, lb >> 16);
            }
        }
    }
}

template <int MT, int PARTS>
__global__ void __launch_bounds__(UMMA_THREADS, 1)
pfb_sym_kernel(const __grid_constant__ CUtensorMap tmap_b, const __grid_constant__ CUtensorMap tmap_out,
               const __grid_constant__ CUtensorMap tmap_out2, const SymParams prm)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    if ((smem_u32(smem) & 1023u) != 0) __trap();                // the swizzled tiles need 1024-byte alignment
    uint8_t* a_ring = smem;
    uint8_t* b_ring = smem + SY_A_RING;
    uint8_t* stage = b_ring + SY_B_ENTRIES * SY_B_ENTRY;
    SmemCtl* ctl = reinterpret_cast<SmemCtl*>(stage + 4 * SY_STAGE);

    constexpr int CG = UMMA_CG;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    constexpr int parts = PARTS;                                      // 2: bf16x3 (hi + lo tiles), 1: single pass
    constexpr uint32_t a_slot_bytes = 2u * parts * A_PART_BYTES;
    const uint32_t n_a = (uint32_t)SY_A_RING / a_slot_bytes;            // 2 (bf16x3) or 4 (single pass)
    const int P = prm.P;
    const int n_kc = P / KC;
    const int half = P >> 1;                                           // bins 0 .. P/2 - 1 are contracted
    const uint32_t rank = cluster_ctarank();                           // rank in the CTA pair; 0 = leader
    constexpr uint32_t leader = 0;
    constexpr uint16_t pair_mask = 3;
    const int cl = blockIdx.x / CG, n_cl = gridDim.x / CG;
    const int npg = prm.n_passes;
    const uint32_t b_box_bytes = (uint32_t)(P < NSUB ? P : NSUB) / CG * KC * 2;   // bytes one TMA box delivers

    if (warp == TMA_WARP && lane == 0) {
        prefetch_tmap(&tmap_b);
        prefetch_tmap(&tmap_out);
        prefetch_tmap(&tmap_out2);
        for (int i = 0; i < 8; ++i) { mbar_init(smem_u32(&ctl->a_full[i]), N_PROD_WARPS + (rank == 0 ? CG - 1 : 0)); mbar_init(smem_u32(&ctl->a_empty[i]), 2); }
        for (int i = 0; i < SY_B_ENTRIES; ++i) { mbar_init(smem_u32(&ctl->b_full[i]), 1); mbar_init(smem_u32(&ctl->b_empty[i]), 2); }
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

    if (warp == TMA_WARP) {
        // ============================ TMA producer: [C|S] tiles, hi then lo per chunk ===============
        if (lane == 0) {
            RingPos b;
            for (int w = cl; w < prm.total_work; w += n_cl) {
                const int k0 = (w % npg) * SY_BINS;
                const int nw = 2 * min(SY_BINS, half - k0);               // matrix rows of this pass
                for (int kc = 0; kc < n_kc; ++kc)
                    for (int part = 0; part < parts; ++part) {
                        mbar_wait<64>(smem_u32(&ctl->b_empty[b.idx]), b.phase ^ 1);
                        const uint32_t bar = smem_u32(&ctl->b_full[b.idx]);
                        const uint32_t dst = smem_u32(b_ring + b.idx * SY_B_ENTRY);
                        const int row = part * P + 2 * k0 + (int)rank * (nw / CG);
                        if (rank == 0) mbar_expect_tx(bar, 2 * b_box_bytes);
                        tma_load_2d_cg2(dst, &tmap_b, mapa_u32(bar, leader), kc * KC, row);
                        b.advance(SY_B_ENTRIES);
                    }
            }
        }
    } else if (warp == MMA_WARP || warp == MMA_WARP2) {
        // ============================ MMA issuers ===========================================
        // warp 13 (h = 0): yr tiles -> D1;  warp 15 (h = 1): yi tiles -> D2.  Both consume the same B entries
        // (b_empty takes one commit from each) and the same A slot (a_empty likewise).  Only the leader CTA
        // issues; the peer's warp 13 forwards "my A tile is ready" to the leader's barrier.
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
            const uint32_t d = tmem_base + (uint32_t)h * 256u;
            long long pm_a = 0, pm_b = 0, pm_t = 0, pm_x, pm_tot = SY_NOW();
            for (int w = cl; w < prm.total_work; w += n_cl) {
                const int k0 = (w % npg) * SY_BINS;
                const int nw = 2 * min(SY_BINS, half - k0);
                const uint32_t idesc = idesc_bf16(BM * CG, nw, prm.fp16 != 0);
                for (int ks = 0; ks < prm.k_splits; ++ks) {
                    const int kc_begin = ks * prm.kc_per_split, kc_end = min(n_kc, kc_begin + prm.kc_per_split);
                    for (int kc = kc_begin; kc < kc_end; ++kc) {
                        pm_x = SY_NOW(); mbar_wait(smem_u32(&ctl->a_full[a.idx]), a.phase); pm_a += SY_NOW() - pm_x;
                        tc_fence_after();
                        const uint32_t a_hi = smem_u32(a_ring + a.idx * a_slot_bytes) + (uint32_t)h * (uint32_t)parts * A_PART_BYTES;
                        const uint32_t a_lo = a_hi + A_PART_BYTES;
                        if (kc == kc_begin) {
                            // first write into this accumulator: wait until the epilogue has drained it
                            pm_x = SY_NOW(); mbar_wait(smem_u32(&ctl->t_empty[h]), te_phase ^ 1u); pm_t += SY_NOW() - pm_x;
                            te_phase ^= 1u;
                            tc_fence_after();
                        }
                        // ---- B_hi: (A_lo x B_hi) then (A_hi x B_hi)
                        pm_x = SY_NOW(); mbar_wait(smem_u32(&ctl->b_full[b.idx]), b.phase); pm_b += SY_NOW() - pm_x;
                        tc_fence_after();
                        if (elect_one()) {
                            const uint64_t bd = smem_desc_sw128(smem_u32(b_ring + b.idx * SY_B_ENTRY));
                            uint32_t acc = kc > kc_begin;
                            if (parts > 1) {
                                const uint64_t ad = smem_desc_sw128(a_lo);
#pragma unroll
                                for (int k = 0; k < KC / 16; ++k) { umma_bf16<CG>(d, ad + 2 * k, bd + 2 * k, idesc, acc); acc = 1; }
                            }
                            const uint64_t ad = smem_desc_sw128(a_hi);
#pragma unroll
                            for (int k = 0; k < KC / 16; ++k) { umma_bf16<CG>(d, ad + 2 * k, bd + 2 * k, idesc, acc); acc = 1; }
                            commit_cg<CG>(smem_u32(&ctl->b_empty[b.idx]), pair_mask);
                        }
                        __syncwarp();
                        b.advance(SY_B_ENTRIES);
                        // ---- B_lo: (A_hi x B_lo)
                        if (parts > 1) {
                            pm_x = SY_NOW(); mbar_wait(smem_u32(&ctl->b_full[b.idx]), b.phase); pm_b += SY_NOW() - pm_x;
                            tc_fence_after();
                            if (elect_one()) {
                                const uint64_t bd = smem_desc_sw128(smem_u32(b_ring + b.idx * SY_B_ENTRY));
                                const uint64_t ad = smem_desc_sw128(a_hi);
#pragma unroll
                                for (int k = 0; k < KC / 16; ++k) umma_bf16<CG>(d, ad + 2 * k, bd + 2 * k, idesc, 1);
                                commit_cg<CG>(smem_u32(&ctl->b_empty[b.idx]), pair_mask);
                            }
                            __syncwarp();
                            b.advance(SY_B_ENTRIES);
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
            if (SY_PROF && prm.prof && lane == 0) {
                unsigned long long* pp = prm.prof + blockIdx.x * 16 + h * 4;
                pp[0] = SY_NOW() - pm_tot; pp[1] = pm_a; pp[2] = pm_b; pp[3] = pm_t;
            }
        }
    } else if (warp >= EPI_WARP0 && warp < EPI_WARP0 + 4) {
        EpiCtx ec;
        ec.t_full0 = smem_u32(&ctl->t_full[0]); ec.t_full1 = smem_u32(&ctl->t_full[1]);
        ec.t_empty0 = smem_u32(&ctl->t_empty[0]); ec.t_empty1 = smem_u32(&ctl->t_empty[1]);
        ec.stage = smem_u32(stage); ec.tmem_base = tmem_base; ec.rank = rank; ec.cl = cl; ec.n_cl = n_cl;
        sym_epilogue<false>(prm, &tmap_out, &tmap_out2, ec, warp - EPI_WARP0, lane);
    } else if (warp >= PROD_WARP0 && warp < PROD_WARP0 + N_PROD_WARPS) {
        // ============================ FIR producers =========================================
        // A chunk is 64 complex columns = two sub-steps of 32 (one complex sample per lane, 16 frames per
        // warp, as in tina_umma.cu).  Software pipeline over the flattened (work item, chunk, sub-step)
        // sequence: the loads of the next sub-step are issued right after the arithmetic of this one.
        const int pw = warp - PROD_WARP0;
        const uint32_t a_ring_s = smem_u32(a_ring);
        // byte offset of this lane's 2-byte cell in row 0 of the warp's slab, per swizzle phase (row & 7), for
        // sub-step 0: complex column lane -> 16-byte chunk lane >> 3, stored at chunk ^ (row & 7); sub-step 1 is
        // chunk + 4, i.e. the same offset with bit 6 flipped
        uint32_t cell0[8];
#pragma unroll
        for (int j = 0; j < 8; ++j)
            cell0[j] = a_ring_s + (uint32_t)(pw * FPW) * 128u + ((((uint32_t)lane >> 3) ^ (uint32_t)j) << 4) + ((uint32_t)lane & 7u) * 2u;
        constexpr int WA = MT > 0 ? MT : 1;
        const float* const window = prm.window;
        const int M = prm.M;
        const long long K = 2LL * P, nblk = prm.NBLK;
        FirRegs<MT> rg;
        int w = cl, st = 0;                                   // st = 2 * kc + sub
        const int n_st = 2 * n_kc;
        uint32_t n = 0;                                       // chunk counter over this CTA's whole sequence
        const float* xs = nullptr;
        long long f0 = 0;
        bool interior = false;
        auto set_tile = [&](int ww) {
            const int tile = ww / npg;
            const int s = tile / prm.tiles_per_stream;
            f0 = (long long)(tile % prm.tiles_per_stream) * (BM * CG) + rank * BM + pw * FPW;
            xs = prm.x + (long long)s * prm.stream_stride + 2 * lane;
            interior = (f0 + M - WA >= 0) && (f0 + FPW + M - 1 <= nblk);
        };
        auto load = [&](int sst) {
            const int c0 = sst * KC + 2 * lane;                // first float column of this lane in the sub-step
            if (interior) fir_load<MT, false, false>(rg, window, P, M, K, nblk, xs + sst * KC, c0, f0);
            else          fir_load<MT, false, true>(rg, window, P, M, K, nblk, xs + sst * KC, c0, f0);
        };
        long long pq_w = 0, pq_c = 0, pq_f = 0, pq_x, pq_tot = SY_NOW();
        bool have = w < prm.total_work;
        if (have) { set_tile(w); load(st); }
        while (have) {
            int w2 = w, st2 = st + 1;
            if (st2 == n_st) { st2 = 0; w2 += n_cl; }
            const bool have2 = w2 < prm.total_work;
            const uint32_t slot_i = n % n_a, slot_ph = (n / n_a) & 1u;
            const int sub = st & 1;
            pq_x = SY_NOW();
            if (sub == 0) mbar_wait(smem_u32(&ctl->a_empty[slot_i]), slot_ph ^ 1);
            pq_w += SY_NOW() - pq_x; pq_x = SY_NOW();
            {
                uint32_t cell[8];
                const uint32_t so = slot_i * a_slot_bytes, sx = sub ? 64u : 0u;
#pragma unroll
                for (int j = 0; j < 8; ++j) cell[j] = (cell0[j] ^ sx) + so;     // bit 6 of a 1024-byte-aligned base is clear
                fir_compute_store_sym<MT, (PARTS > 1)>(rg, cell, prm.fp16 != 0);
            }
            if (have2) {
                if (w2 != w) set_tile(w2);
                load(st2);
            }
            pq_c += SY_NOW() - pq_x; pq_x = SY_NOW();
            if (sub == 1) {
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&ctl->a_full[slot_i]));
                ++n;
            }
            pq_f += SY_NOW() - pq_x;
            w = w2; st = st2; have = have2;
        }
        if (SY_PROF && prm.prof && pw == 0 && lane == 0) {
            unsigned long long* pp = prm.prof + blockIdx.x * 16 + 12;
            pp[0] = SY_NOW() - pq_tot; pp[1] = pq_w; pp[2] = pq_c; pp[3] = pq_f;
        }
    }

    tc_fence_before();
    cluster_sync();                                           // the peer's smem / barriers stay live until both are done
    if (warp == ALLOC_WARP) tmem_dealloc<CG>(tmem_base, 512);
}

// Epilogue of the REAL kind (pfb_symt_kernel<.., REAL = true>).  The real frame y[p] is contracted as its even
// samples (the "yr" tiles) and its odd samples (the "yi" tiles) against the cos / sin columns of the bins
// k in [0, P/4):  U = sum_q y[2q] c, Z = sum_q y[2q] s  (D1),  W = sum_q y[2q+1] c', V = sum_q y[2q+1] s'  (D2),
// with c, s at angle 2 pi (2q) k / P and c', s' at 2 pi (2q+1) k / P.  Columns k and P/2 - k of the Fourier
// matrix agree on the even samples and differ in sign on the odd ones, so
//     X[k] = (U + W) - i (Z + V),        X[P/2 - k] = (U - W) + i (Z - V).
// Bin 0 has s = s' = 0: its sine columns carry (-1)^q instead and deliver the unpaired bin P/4
// (X[P/4] = D1[1] - i D2[1]); the mirror of bin 0 is the Nyquist bin.  Output rows are P + 2 floats, i.e. only
// 8-byte aligned, so the tiles leave through a swizzled shared-memory transpose and 8-byte stores (two rows x
// 128 contiguous bytes per instruction); later accumulation chains add with red.global.add.v2.f32.
__device__ __forceinline__ void sym_epilogue_real(const SymParams& prm, const EpiCtx& e, const int q, const int lane)
{
    constexpr int CG = UMMA_CG;
    const int P = prm.P, quarter = P >> 2, npg = prm.n_passes;
    const uint32_t sb = e.stage + (uint32_t)q * SY_STAGE;
    const uint32_t taddr = e.tmem_base + ((uint32_t)(q * 32) << 16);
    const uint32_t rowoff = (uint32_t)lane * 128u, sw = (uint32_t)lane & 7u;
    // transposed read-out: lane -> (row lane >> 4 (+ 2 i), bin lane & 15)
    const uint32_t rd_c = (uint32_t)lane & 15u, rd_r0 = (uint32_t)lane >> 4;
    uint32_t tf_phase = 0;
    // several accumulation chains (K > 1024): the first chain's plain stores are marked evict-last so that the tile is
    // still in L2 when the next chain's red.global.add arrives (measured at c5: DRAM traffic 1.86 GB without the hint)
    const bool keep_l2 = prm.k_splits > 1;
    const uint64_t pol_keep = l2_policy_evict_last();
    long long pe_w = 0, pe_d = 0, pe_x, pe_tot = SY_NOW();
    for (int w = e.cl; w < prm.total_work; w += e.n_cl) {
        const int tile = w / npg;
        const int k0 = (w % npg) * SY_BINS;
        const int ncol = 2 * min(SY_BINS, quarter - k0);
        const int s = tile / prm.tiles_per_stream;
        const long long row0 = (long long)(tile % prm.tiles_per_stream) * (BM * CG) + e.rank * BM + q * 32;
        const int rows_valid = (int)min(32LL, prm.F - row0);
        float* const otile = prm.out + ((long long)s * prm.F + row0) * (long long)(P + 2);
        for (int ks = 0; ks < prm.k_splits; ++ks) {
            pe_x = SY_NOW();
            mbar_wait<256>(e.t_full0, tf_phase);
            mbar_wait<256>(e.t_full1, tf_phase);
            pe_w += SY_NOW() - pe_x; pe_x = SY_NOW();
            tf_phase ^= 1u;
            tc_fence_after();
            uint32_t r1[32], r2[32];
            tmem_ld32(taddr, r1);
            tmem_ld32(taddr + 256u, r2);
            // store a staged 32 x 16-bin tile whose first bin is `bin0`: lanes 0-15 / 16-31 take rows 2 i / 2 i + 1
            auto flush = [&](uint32_t tile_s, int bin0) {
#pragma unroll 4
                for (int i = 0; i < 16; ++i) {
                    const uint32_t r = rd_r0 + 2u * (uint32_t)i;
                    const float2 v = lds_f2(tile_s + r * 128u + ((((rd_c >> 1) ^ (r & 7u))) << 4) + (rd_c & 1u) * 8u);
                    if ((int)r < rows_valid) {
                        float2* g = reinterpret_cast<float2*>(otile + (long long)r * (P + 2) + 2 * (bin0 + (int)rd_c));
                        if (ks > 0) atomicAdd(g, v);
                        else if (keep_l2) st_f2_evict_last(g, v, pol_keep);    // a later chain adds into this tile: keep it in L2
                        else *g = v;
                    }
                }
            };
            for (int cb = 0; cb < ncol; cb += 32) {
                const int kb = k0 + (cb >> 1);
                const bool last = cb + 32 >= ncol;
                tmem_ld_wait();
                if (last) {
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) {
                        arrive_leader<CG>(e.t_empty0, e.rank, 0);
                        arrive_leader<CG>(e.t_empty1, e.rank, 0);
                    }
                    pe_d += SY_NOW() - pe_x;
                }
#define SY_F(v) __uint_as_float(v)
                if (kb == 0) {
                    // the sine slots of bin 0 carry (-1)^q: X[P/4] = D1[1] - i D2[1] (unpaired)
                    if (lane < rows_valid) {
                        float2* g = reinterpret_cast<float2*>(otile + (long long)lane * (P + 2) + 2 * quarter);
                        const float2 v = make_float2(SY_F(r1[1]), -SY_F(r2[1]));
                        if (ks > 0) atomicAdd(g, v); else *g = v;
                    }
                    r1[1] = 0u; r2[1] = 0u;                      // Z = V = 0 for bin 0
                }
                __syncwarp();                                     // the previous step's read-out of both tiles is done
#pragma unroll
                for (int g = 0; g < 8; ++g) {
                    const float U0 = SY_F(r1[4 * g]), Z0 = SY_F(r1[4 * g + 1]), U1 = SY_F(r1[4 * g + 2]), Z1 = SY_F(r1[4 * g + 3]);
                    const float W0 = SY_F(r2[4 * g]), V0 = SY_F(r2[4 * g + 1]), W1 = SY_F(r2[4 * g + 2]), V1 = SY_F(r2[4 * g + 3]);
                    // forward: bins kb + 2g, kb + 2g + 1 -> 16-byte chunk g; the imaginary part of bin 0 is +0
                    const float i0 = (kb == 0 && g == 0) ? 0.f : -(Z0 + V0);
                    sts128(sb + rowoff + (((uint32_t)g ^ sw) << 4), __float_as_uint(U0 + W0), __float_as_uint(i0),
                           __float_as_uint(U1 + W1), __float_as_uint(-(Z1 + V1)));
                    // mirrored: bin P/2 - kb - j at position 15 - j: j = 2g + 1 -> position 14 - 2g, j = 2g -> 15 - 2g: chunk 7 - g
                    sts128(sb + 4096u + rowoff + (((uint32_t)(7 - g) ^ sw) << 4), __float_as_uint(U1 - W1), __float_as_uint(Z1 - V1),
                           __float_as_uint(U0 - W0), __float_as_uint(Z0 - V0));
                }
#undef SY_F
                if (!last) { tmem_ld32(taddr + cb + 32, r1); tmem_ld32(taddr + 256u + cb + 32, r2); }
                __syncwarp();
                flush(sb, kb);
                flush(sb + 4096u, (P >> 1) - kb - 15);
            }
        }
    }
    if (SY_PROF && prm.prof && q == 0 && lane == 0) {
        unsigned long long* pp = prm.prof + blockIdx.x * 16 + 8;
        pp[0] = SY_NOW() - pe_tot; pp[1] = pe_w; pp[2] = pe_d;
    }
}

__device__ __forceinline__ void sts64f(uint32_t addr, float a, float b)
{
    asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(addr), "f"(a), "f"(b) : "memory");
}

// Real-kind epilogue through the TMA engine (even F, or one stream: see sym_pfb).  Output rows are P + 2 floats, so
// only PAIRS of rows have a 16-byte-multiple pitch: the tensor maps view the output as [S][F/2][2 (P + 2)] and a
// warp's 32 rows leave as 16-row boxes, even rows and odd rows separately.  TMA boxes must start 16-byte aligned:
//   forward tile  (bins kb .. kb+15, floats 2 kb ..):        even rows aligned -> 32-float box; odd rows start 8
//                 bytes off -> 28-float box over the floats 2 .. 29 of the tile, the edge pairs (floats 0-1, 30-31)
//                 are stored from registers;
//   mirrored tile (bins P/2-kb-15 .. P/2-kb, floats P-2kb-30 ..): the other way round (odd rows aligned).
// So every lane fills one swizzled 128-byte row (its "full" tile) and one dense 112-byte row (its "part" tile) per
// step and stores two 8-byte edges; later accumulation chains use the add-reduce forms (fp32 add at L2).
__device__ __forceinline__ void sym_epilogue_real_tma(const SymParams& prm, const CUtensorMap* tmap32, const CUtensorMap* tmap28,
                                                      const EpiCtx& e, const int q, const int lane)
{
    constexpr int CG = UMMA_CG;
    const int P = prm.P, quarter = P >> 2, npg = prm.n_passes;
    const uint32_t sb = e.stage + (uint32_t)q * SY_STAGE;
    // staging (8 KB per warp): full tiles of the even rows (forward) and of the odd rows (mirrored), 16 x 128 B
    // swizzled; part tiles of the odd rows (forward) and of the even rows (mirrored), 16 x 112 B dense
    const uint32_t b_fe = sb, b_mo = sb + 2048u, b_f28 = sb + 4096u, b_m28 = sb + 4096u + 1792u;
    const uint32_t taddr = e.tmem_base + ((uint32_t)(q * 32) << 16);
    const bool odd = (lane & 1) != 0;
    const uint32_t rr = (uint32_t)lane >> 1, sw = rr & 7u;
    const uint32_t full_row = (odd ? b_mo : b_fe) + rr * 128u;
    const uint32_t part_row = (odd ? b_f28 : b_m28) + rr * 112u;
    uint32_t tf_phase = 0;
    const bool issuer = elect_one();                          // see sym_epilogue: one elected thread issues and waits
    const bool keep_l2 = prm.k_splits > 1;
    const uint64_t pol_keep = l2_policy_evict_last();
    long long pe_w = 0, pe_d = 0, pe_d0 = 0, pe_x, pe_tot = SY_NOW();
    for (int w = e.cl; w < prm.total_work; w += e.n_cl) {
        const int tile = w / npg;
        const int k0 = (w % npg) * SY_BINS;
        const int ncol = 2 * min(SY_BINS, quarter - k0);
        const int s = tile / prm.tiles_per_stream;
        const long long row0 = (long long)(tile % prm.tiles_per_stream) * (BM * CG) + e.rank * BM + q * 32;
        const bool row_ok = lane < (int)min(32LL, prm.F - row0);
        float* const orow = prm.out + ((long long)s * prm.F + row0 + lane) * (long long)(P + 2);
        const int pr0 = (int)(row0 >> 1);
        // odd F (one stream only): the last row has no partner, the row-pair maps end before it; its lane (an even
        // one) stores everything from registers
        const bool lone = (prm.F & 1) && row0 + lane == prm.F - 1;
        for (int ks = 0; ks < prm.k_splits; ++ks) {
            if (ks > 0 && issuer) bulk_wait<0>();          // the previous chain's stores to this tile are complete
            pe_x = SY_NOW();
            mbar_wait<256>(e.t_full0, tf_phase);
            mbar_wait<256>(e.t_full1, tf_phase);
            pe_w += SY_NOW() - pe_x; pe_x = SY_NOW();
            tf_phase ^= 1u;
            tc_fence_after();
            auto put = [&](float* g, float re, float im) {        // one complex value from registers (8-byte aligned)
                if (row_ok && !SY_DBG(16)) {
                    float2* g2 = reinterpret_cast<float2*>(g);
                    if (ks > 0) atomicAdd(g2, make_float2(re, im)); else *g2 = make_float2(re, im);
                }
            };
            for (int cb = 0; cb < ncol; cb += 32) {
                const int kb = k0 + (cb >> 1);
                const bool last = cb + 32 >= ncol;
                const int f_col = 2 * kb, m_col = P - 2 * kb - 30;      // first float of the forward / mirrored tile in a row
                if (issuer) bulk_wait_read<0>();                // the staged tiles of the previous step have been read
                __syncwarp();
                float e0x = 0.f, e0y = 0.f, e7x = 0.f, e7y = 0.f;   // the part tile's edge pairs (floats 0-1 and 30-31)
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    // 16 accumulator columns = 8 bins at a time (32 live accumulator registers instead of 64: the
                    // 32-column form spilled, and spill reloads queue behind the saturated shared-memory pipe)
                    uint32_t r1[16], r2[16];
                    tmem_ld16(taddr + cb + 16 * h, r1);
                    tmem_ld16(taddr + 256u + cb + 16 * h, r2);
                    tmem_ld_wait();
                    if (last && h == 1) {
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) {
                            arrive_leader<CG>(e.t_empty0, e.rank, 0);
                            arrive_leader<CG>(e.t_empty1, e.rank, 0);
                        }
                        pe_d += SY_NOW() - pe_x;
                        if (ks == 0) pe_d0 += SY_NOW() - pe_x;
                    }
#define SY_F(v) __uint_as_float(v)
                    if (kb == 0 && h == 0) {
                        // the sine slots of bin 0 carry (-1)^q: X[P/4] = D1[1] - i D2[1] (unpaired)
                        put(orow + 2 * quarter, SY_F(r1[1]), -SY_F(r2[1]));
                        r1[1] = 0u; r2[1] = 0u;                  // Z = V = 0 for bin 0
                    }
#pragma unroll
                    for (int gg = 0; gg < 4; ++gg) {
                        const int g = 4 * h + gg;
                        const float U0 = SY_F(r1[4 * gg]), Z0 = SY_F(r1[4 * gg + 1]), U1 = SY_F(r1[4 * gg + 2]), Z1 = SY_F(r1[4 * gg + 3]);
                        const float W0 = SY_F(r2[4 * gg]), V0 = SY_F(r2[4 * gg + 1]), W1 = SY_F(r2[4 * gg + 2]), V1 = SY_F(r2[4 * gg + 3]);
                        // forward chunk g: bins kb + 2g, kb + 2g + 1 (the imaginary part of bin 0 is +0);
                        // mirrored chunk 7 - g: bins P/2 - kb - (2g + 1), P/2 - kb - 2g
                        const float fa = U0 + W0, fb = (kb == 0 && g == 0) ? 0.f : -(Z0 + V0), fc = U1 + W1, fd = -(Z1 + V1);
                        const float ma = U1 - W1, mb = Z1 - V1, mc = U0 - W0, md = Z0 - V0;
                        // full tile: even rows forward chunk g, odd rows mirrored chunk 7 - g
                        const uint32_t cf = odd ? (uint32_t)(7 - g) : (uint32_t)g;
                        sts128(full_row + ((cf ^ sw) << 4), __float_as_uint(odd ? ma : fa), __float_as_uint(odd ? mb : fb),
                               __float_as_uint(odd ? mc : fc), __float_as_uint(odd ? md : fd));
                        // part tile (floats 2 .. 29 of the other tile): odd rows forward chunk g, even rows mirrored chunk
                        // 7 - g; chunk c sits at bytes 16 c - 8 .. 16 c + 7 of the dense row, chunks 0 / 7 lose a half to the edges
                        const float pa = odd ? fa : ma, pb = odd ? fb : mb, pc = odd ? fc : mc, pd = odd ? fd : md;
                        const uint32_t c_dense = odd ? (uint32_t)g : (uint32_t)(7 - g);
                        if (g == 0) {
                            if (odd) { e0x = pa; e0y = pb; sts64f(part_row, pc, pd); }
                            else     { e7x = pc; e7y = pd; sts64f(part_row + 104u, pa, pb); }
                        } else if (g == 7) {
                            if (odd) { e7x = pc; e7y = pd; sts64f(part_row + 104u, pa, pb); }
                            else     { e0x = pa; e0y = pb; sts64f(part_row, pc, pd); }
                        } else {
                            sts64f(part_row + 16u * c_dense - 8u, pa, pb);
                            sts64f(part_row + 16u * c_dense, pc, pd);
                        }
                        if (lone) {                                // (an even lane) every value of the row from registers
                            put(orow + f_col + 4 * g, fa, fb); put(orow + f_col + 4 * g + 2, fc, fd);
                            if (g != 7) put(orow + m_col + 4 * (7 - g), ma, mb);
                            if (g != 0) put(orow + m_col + 4 * (7 - g) + 2, mc, md);
                        }
                    }
#undef SY_F
                }
                {
                    float* const pbase = orow + (odd ? f_col : m_col);
                    put(pbase, e0x, e0y);
                    put(pbase + 30, e7x, e7y);
                }
                fence_proxy_async();
                __syncwarp();
                if (issuer) {
                    // paired-row coordinates: an odd row starts at float P + 2 of its pair
                    if (SY_DBG(16)) { }
                    else if (ks == 0 && keep_l2) {                // a later chain adds into this tile: keep it in L2
                        tma_store_3d_hint(tmap32, b_fe, f_col, pr0, s, pol_keep);
                        tma_store_3d_hint(tmap32, b_mo, P + 2 + m_col, pr0, s, pol_keep);
                        tma_store_3d_hint(tmap28, b_f28, P + 2 + f_col + 2, pr0, s, pol_keep);
                        tma_store_3d_hint(tmap28, b_m28, m_col + 2, pr0, s, pol_keep);
                    } else if (ks == 0) {
                        tma_store_3d(tmap32, b_fe, f_col, pr0, s);
                        tma_store_3d(tmap32, b_mo, P + 2 + m_col, pr0, s);
                        tma_store_3d(tmap28, b_f28, P + 2 + f_col + 2, pr0, s);
                        tma_store_3d(tmap28, b_m28, m_col + 2, pr0, s);
                    } else {
                        tma_reduce_add_3d(tmap32, b_fe, f_col, pr0, s);
                        tma_reduce_add_3d(tmap32, b_mo, P + 2 + m_col, pr0, s);
                        tma_reduce_add_3d(tmap28, b_f28, P + 2 + f_col + 2, pr0, s);
                        tma_reduce_add_3d(tmap28, b_m28, m_col + 2, pr0, s);
                    }
                    bulk_commit();
                }
            }
        }
    }
    if (issuer) bulk_wait<0>();                               // staging tiles must outlive their TMA reads
    if (SY_PROF && prm.prof && q == 0 && lane == 0) {
        unsigned long long* pp = prm.prof + blockIdx.x * 16 + 8;
        pp[0] = SY_NOW() - pe_tot; pp[1] = pe_w; pp[2] = pe_d; pp[3] = pe_d0;
    }
}

// =====================================================================================
// pfb_symt_kernel: the same contraction with the INPUT WINDOW AND THE TAPS STAGED BY TMA (the north_star
// sketch): per chunk of 32 complex columns the (128 + MT - 1) x 32 block of input
// rows and the MT x 32 block of prototype-filter taps are bulk-copied into a two-slot shared-memory ring; the
// FIR producers read their sliding window from shared memory (no long-latency global loads in the FIR warps,
// every input row fetched from L2 once per CTA and chunk instead of once per 16-frame warp slab, taps once per
// CTA instead of once per warp).  REAL = true: the real kind, contracted as even / odd samples against the
// cos / sin columns of the bins [0, P/4) -- see sym_epilogue_real; the producers are the same (an adjacent pair of
// real samples takes the place of (re, im)), each MMA warp has its own twiddle entries (even-sample and
// odd-sample matrices), and K = P/2.  To make room the operand tiles are 32 contraction elements wide: A slot =
// 4 x 8 KB, B entry = 8 KB per CTA (64-byte rows, SWIZZLE_64B), two K = 16 MMAs per tile and product.
// The A tiles are MN-MAJOR (frames contiguous, SWIZZLE_128B: [2 blocks of 64 frames][4 groups of 8 columns][8 columns]
// [128 B = 8 units of 8 frames]): a producer lane owns one column, so 8 consecutive frames of one part are ONE 16-byte
// store (conflict-free per quarter warp) instead of eight 2-byte stores -- the K-major layout cost 64 st.shared.b16
// per warp and chunk at two wavefronts each (two lanes share a 32-bit word), 1024 of the ~3000 shared-memory
// wavefronts per chunk that bound the kernel (ncu: 37.9 M store bank conflicts per c4 launch).
//   shared memory: A ring 64 KB (2 slots; 4 for the single pass) | B ring 48 KB (6 entries = 3 chunks) |
//                  input ring 2 x 40 KB | epilogue staging 32 KB
//   warps: 0-7 FIR producers, 8-11 epilogue, 12 TMA (twiddles), 13 / 15 MMA issuers, 14 TMEM allocation + TMA (input)
// =====================================================================================
constexpr int ST_KC = 32;                                  // contraction elements (complex columns) per chunk
constexpr int ST_TILE = BM * ST_KC * 2;                    // 8 KB: 128 frames x 32 columns of bf16
constexpr uint32_t ST_A_LBO = 4096;                        // MN-major A tile: bytes between the two blocks of 64 frames
constexpr uint32_t ST_A_SBO = 1024;                        //                  bytes between groups of 8 columns
constexpr uint32_t ST_A_KSTEP = (2 * ST_A_SBO) >> 4;       // descriptor advance per K = 16 MMA (two column groups)
constexpr int ST_A_RING = 64 * 1024;
constexpr int ST_B_ENTRY = (NSUB / UMMA_CG) * ST_KC * 2;   // 8 KB per CTA
constexpr int ST_B_ENTRIES = 6;
constexpr int ST_IN_ROWS_MAX = BM + 15;                    // 143 input rows of 256 B
constexpr int ST_IN_TAPS = ST_IN_ROWS_MAX * 256;           // byte offset of the taps block in an input slot
constexpr int ST_IN_SLOT = 40 * 1024;                      // 36 608 B of rows + up to 4 KB of taps (real kind: 64 per row)
constexpr int ST_IN_SLOTS = 2;

struct SmemCtlT {
    uint64_t a_full[4], a_empty[4];
    uint64_t b_full[8], b_empty[8];
    uint64_t in_full[2], in_empty[2];
    uint64_t t_full[2], t_empty[2];
    uint32_t tmem_base;
};
constexpr size_t ST_SMEM_BYTES = ST_A_RING + ST_B_ENTRIES * ST_B_ENTRY + ST_IN_SLOTS * ST_IN_SLOT + 4 * SY_STAGE + sizeof(SmemCtlT);
static_assert(ST_SMEM_BYTES <= 232448, "exceeds the 227 KB shared memory opt-in limit");

// GROUPED = true (MT = 16 only): 16 < M <= 64 taps.  The taps are processed in groups of 16: per chunk and group g the
// TMA warp stages the 143 rows starting 16 g rows EARLIER and the tap rows 16 g .. 16 g + 15 (rows >= M read as
// zeros), the producers accumulate y += sum_{m' < 16} w[16 g + m'] x[f + M-1 - 16 g - m'] over the groups in
// registers (two sets of 8 frames so that the sums stay live) and only then split and store the operand tile: the
// subfiltered signal never leaves the SM for any M the library accepts.
template <int MT, int PARTS, bool REAL, bool GROUPED = false>
__global__ void __launch_bounds__(UMMA_THREADS, 1)
pfb_symt_kernel(const __grid_constant__ CUtensorMap tmap_b, const __grid_constant__ CUtensorMap tmap_out,
                const __grid_constant__ CUtensorMap tmap_out2, const __grid_constant__ CUtensorMap tmap_x,
                const __grid_constant__ CUtensorMap tmap_w, const SymParams prm)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    if ((smem_u32(smem) & 1023u) != 0) __trap();
    uint8_t* a_ring = smem;
    uint8_t* b_ring = smem + ST_A_RING;
    uint8_t* in_ring = b_ring + ST_B_ENTRIES * ST_B_ENTRY;
    uint8_t* stage = in_ring + ST_IN_SLOTS * ST_IN_SLOT;
    SmemCtlT* ctl = reinterpret_cast<SmemCtlT*>(stage + 4 * SY_STAGE);

    constexpr int CG = UMMA_CG;
    constexpr int WA = MT > 0 ? MT : 1;
    constexpr int IN_ROWS = BM + WA - 1;                               // input rows one CTA needs per chunk
    constexpr int parts = PARTS;
    constexpr uint32_t a_slot_bytes = 2u * parts * ST_TILE;            // [yr hi | yr lo | yi hi | yi lo] or [yr | yi]
    constexpr uint32_t n_a = (uint32_t)ST_A_RING / a_slot_bytes;       // 2 (bf16x3) or 4 (single pass)
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int P = prm.P, M = prm.M;
    const int kdim = REAL ? (P >> 1) : P;                              // contraction length (sample pairs / complex samples)
    const int n_kc = kdim / ST_KC;
    const int half = REAL ? (P >> 2) : (P >> 1);                       // bins contracted: [0, P/4) real, [0, P/2) complex
    constexpr int EO = REAL ? 2 : 1;                                   // twiddle matrices: even / odd samples, or one
    constexpr uint32_t EPC = (uint32_t)parts * EO;                     // B ring entries per chunk
    const uint32_t rank = cluster_ctarank();
    constexpr uint32_t leader = 0;
    constexpr uint16_t pair_mask = 3;
    const int cl = blockIdx.x / CG, n_cl = gridDim.x / CG;
    const int npg = prm.n_passes;
    const int b_rows = 2 * half;                                       // matrix rows per part (and per even / odd half)
    const uint32_t b_box_bytes = (uint32_t)(b_rows < NSUB ? b_rows : NSUB) / CG * ST_KC * 2;
    static_assert(!GROUPED || MT == 16, "tap groups are groups of 16");
    const int n_groups = GROUPED ? (M + 15) / 16 : 1;                  // tap groups per chunk (GROUPED: 16 < M <= 64)

    if (warp == TMA_WARP && lane == 0) {
        prefetch_tmap(&tmap_b); prefetch_tmap(&tmap_out); prefetch_tmap(&tmap_out2); prefetch_tmap(&tmap_x);
        if (MT > 0) prefetch_tmap(&tmap_w);
        for (int i = 0; i < 4; ++i) { mbar_init(smem_u32(&ctl->a_full[i]), N_PROD_WARPS + (rank == 0 ? CG - 1 : 0)); mbar_init(smem_u32(&ctl->a_empty[i]), 2); }
        for (int i = 0; i < ST_B_ENTRIES; ++i) { mbar_init(smem_u32(&ctl->b_full[i]), 1); mbar_init(smem_u32(&ctl->b_empty[i]), REAL ? 1 : 2); }
        for (int i = 0; i < ST_IN_SLOTS; ++i) { mbar_init(smem_u32(&ctl->in_full[i]), 1); mbar_init(smem_u32(&ctl->in_empty[i]), N_PROD_WARPS); }
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
                // first input row of this CTA's window: frame f0 uses rows f0 + M - WA .. f0 + M - 1 (taps m >= M are zero)
                const int r0 = (tile % prm.tiles_per_stream) * (BM * CG) + (int)rank * BM + M - WA;
                for (int kc = 0; kc < n_kc; ++kc)
                    for (int g = 0; g < n_groups; ++g) {
                        mbar_wait<64>(smem_u32(&ctl->in_empty[in.idx]), in.phase ^ 1);
                        const uint32_t bar = smem_u32(&ctl->in_full[in.idx]);
                        const uint32_t dst = smem_u32(in_ring + in.idx * ST_IN_SLOT);
                        mbar_expect_tx(bar, (uint32_t)IN_ROWS * 256u + (MT > 0 ? (uint32_t)MT * (REAL ? 256u : 128u) : 0u));
                        tma_load_3d(dst, &tmap_x, bar, kc * 2 * ST_KC, r0 - 16 * g, s);   // rows outside [0, NB) arrive as zeros
                        if (MT > 0) tma_load_2d(dst + ST_IN_TAPS, &tmap_w, bar, kc * ST_KC * (REAL ? 2 : 1), 16 * g);   // rows >= M arrive as zeros
                        in.advance(ST_IN_SLOTS);
                    }
            }
        }
    } else if (warp == TMA_WARP) {
        // ============================ TMA producer: [C|S] tiles, hi then lo per chunk ===============
        if (lane == 0) {
            RingPos b;
            for (int w = cl; w < prm.total_work; w += n_cl) {
                const int k0 = (w % npg) * SY_BINS;
                const int nw = 2 * min(SY_BINS, half - k0);
                for (int kc = 0; kc < n_kc; ++kc)
                    for (int pe = 0; pe < (int)EPC; ++pe) {             // (part, even / odd) in ring order
                        mbar_wait<64>(smem_u32(&ctl->b_empty[b.idx]), b.phase ^ 1);
                        const uint32_t bar = smem_u32(&ctl->b_full[b.idx]);
                        const uint32_t dst = smem_u32(b_ring + b.idx * ST_B_ENTRY);
                        const int row = pe * b_rows + 2 * k0 + (int)rank * (nw / CG);
                        if (rank == 0) mbar_expect_tx(bar, 2 * b_box_bytes);
                        tma_load_2d_cg2(dst, &tmap_b, mapa_u32(bar, leader), kc * ST_KC, row);
                        b.advance(ST_B_ENTRIES);
                    }
            }
        }
    } else if (warp == MMA_WARP || warp == MMA_WARP2) {
        // ============================ MMA issuers (as pfb_sym_kernel, two K = 16 steps per tile) ==========
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
            RingPos a;
            uint32_t be = 0;                                       // B ring entries issued before this chunk
            uint32_t te_phase = 0;
            const uint32_t d = tmem_base + (uint32_t)h * 256u;
            long long pm_a = 0, pm_b = 0, pm_t = 0, pm_x, pm_tot = SY_NOW();
            for (int w = cl; w < prm.total_work; w += n_cl) {
                const int k0 = (w % npg) * SY_BINS;
                const int nw = 2 * min(SY_BINS, half - k0);
                const uint32_t idesc = idesc_bf16(BM * CG, nw, prm.fp16 != 0) | IDESC_A_MN_MAJOR;
                for (int ks = 0; ks < prm.k_splits; ++ks) {
                    const int kc_begin = ks * prm.kc_per_split, kc_end = min(n_kc, kc_begin + prm.kc_per_split);
                    for (int kc = kc_begin; kc < kc_end; ++kc) {
                        pm_x = SY_NOW(); mbar_wait(smem_u32(&ctl->a_full[a.idx]), a.phase); pm_a += SY_NOW() - pm_x;
                        tc_fence_after();
                        const uint32_t a_hi = smem_u32(a_ring + a.idx * a_slot_bytes) + (uint32_t)h * (uint32_t)parts * ST_TILE;
                        const uint32_t a_lo = a_hi + ST_TILE;
                        if (kc == kc_begin) {
                            pm_x = SY_NOW(); mbar_wait(smem_u32(&ctl->t_empty[h]), te_phase ^ 1u); pm_t += SY_NOW() - pm_x;
                            te_phase ^= 1u;
                            tc_fence_after();
                        }
                        // ring order per chunk: (hi, even) [(hi, odd)] (lo, even) [(lo, odd)]; the real kind gives each
                        // MMA warp its own matrix (h = 0: even samples, h = 1: odd samples), the complex kind shares one
                        uint32_t e_i = be + (REAL ? (uint32_t)h : 0u);
                        uint32_t bi = e_i % ST_B_ENTRIES, bp = (e_i / ST_B_ENTRIES) & 1u;
                        pm_x = SY_NOW(); mbar_wait(smem_u32(&ctl->b_full[bi]), bp); pm_b += SY_NOW() - pm_x;
                        tc_fence_after();
                        if (elect_one()) {
                            const uint64_t bd = smem_desc_sw64(smem_u32(b_ring + bi * ST_B_ENTRY));
                            uint32_t acc = kc > kc_begin;
                            if (parts > 1) {
                                const uint64_t ad = smem_desc_mn_sw128(a_lo, ST_A_LBO, ST_A_SBO);
#pragma unroll
                                for (int k = 0; k < ST_KC / 16; ++k) { umma_bf16<CG>(d, ad + ST_A_KSTEP * k, bd + 2 * k, idesc, acc); acc = 1; }
                            }
                            const uint64_t ad = smem_desc_mn_sw128(a_hi, ST_A_LBO, ST_A_SBO);
#pragma unroll
                            for (int k = 0; k < ST_KC / 16; ++k) { umma_bf16<CG>(d, ad + ST_A_KSTEP * k, bd + 2 * k, idesc, acc); acc = 1; }
                            commit_cg<CG>(smem_u32(&ctl->b_empty[bi]), pair_mask);
                        }
                        __syncwarp();
                        if (parts > 1) {
                            e_i += EO; bi = e_i % ST_B_ENTRIES; bp = (e_i / ST_B_ENTRIES) & 1u;
                            pm_x = SY_NOW(); mbar_wait(smem_u32(&ctl->b_full[bi]), bp); pm_b += SY_NOW() - pm_x;
                            tc_fence_after();
                            if (elect_one()) {
                                const uint64_t bd = smem_desc_sw64(smem_u32(b_ring + bi * ST_B_ENTRY));
                                const uint64_t ad = smem_desc_mn_sw128(a_hi, ST_A_LBO, ST_A_SBO);
#pragma unroll
                                for (int k = 0; k < ST_KC / 16; ++k) umma_bf16<CG>(d, ad + ST_A_KSTEP * k, bd + 2 * k, idesc, 1);
                                commit_cg<CG>(smem_u32(&ctl->b_empty[bi]), pair_mask);
                            }
                            __syncwarp();
                        }
                        be += EPC;
                        if (elect_one()) {
                            commit_cg<CG>(smem_u32(&ctl->a_empty[a.idx]), pair_mask);
                            if (kc == kc_end - 1) commit_cg<CG>(smem_u32(&ctl->t_full[h]), pair_mask);
                        }
                        __syncwarp();
                        a.advance(n_a);
                    }
                }
            }
            if (SY_PROF && prm.prof && lane == 0) {
                unsigned long long* pp = prm.prof + blockIdx.x * 16 + h * 4;
                pp[0] = SY_NOW() - pm_tot; pp[1] = pm_a; pp[2] = pm_b; pp[3] = pm_t;
            }
        }
    } else if (warp >= EPI_WARP0 && warp < EPI_WARP0 + 4) {
        EpiCtx ec;
        ec.t_full0 = smem_u32(&ctl->t_full[0]); ec.t_full1 = smem_u32(&ctl->t_full[1]);
        ec.t_empty0 = smem_u32(&ctl->t_empty[0]); ec.t_empty1 = smem_u32(&ctl->t_empty[1]);
        ec.stage = smem_u32(stage); ec.tmem_base = tmem_base; ec.rank = rank; ec.cl = cl; ec.n_cl = n_cl;
        if (REAL && prm.real_tma) sym_epilogue_real_tma(prm, &tmap_out, &tmap_out2, ec, warp - EPI_WARP0, lane);
        else if (REAL) sym_epilogue_real(prm, ec, warp - EPI_WARP0, lane);
        else      sym_epilogue<false>(prm, &tmap_out, &tmap_out2, ec, warp - EPI_WARP0, lane);
    } else if (warp >= PROD_WARP0 && warp < PROD_WARP0 + N_PROD_WARPS) {
        // ============================ FIR producers =========================================
        // Warp pw owns frames 16 pw .. 16 pw + 15 of the CTA's tile, lane = complex column of the chunk.  Per
        // chunk: wait for the staged rows, read the 16 + MT - 1 rows of the sliding window and the MT taps from
        // shared memory, polyphase MAC in registers (Eq. (20)), split into bf16 hi / lo, de-interleave into the
        // MN-major yr / yi tiles: column c = lane sits in column group c >> 3, row c & 7 of the atom; the warp's frames
        // 16 pw .. 16 pw + 15 are the 16-byte units 2 (pw & 3), + 1 of the 64-frame block pw >> 2, stored at unit ^ (c & 7).
        const int pw = warp - PROD_WARP0;
        const uint32_t a_ring_s = smem_u32(a_ring), in_ring_s = smem_u32(in_ring);
        uint32_t cell0[FPW / 8];
#pragma unroll
        for (int j = 0; j < FPW / 8; ++j)
            cell0[j] = a_ring_s + (uint32_t)(pw >> 2) * ST_A_LBO + ((uint32_t)lane >> 3) * ST_A_SBO + ((uint32_t)lane & 7u) * 128u +
                       (((2u * ((uint32_t)pw & 3u) + (uint32_t)j) ^ ((uint32_t)lane & 7u)) << 4);
        constexpr uint32_t im_off = (uint32_t)parts * ST_TILE;
        const uint32_t in_lane = in_ring_s + (uint32_t)(pw * FPW) * 256u + (uint32_t)lane * 8u;
        const uint32_t tap_lane = in_ring_s + ST_IN_TAPS + (uint32_t)lane * (REAL ? 8u : 4u);
        long long pq_w = 0, pq_c = 0, pq_f = 0, pq_x, pq_tot = SY_NOW();
        RingPos in, a;
        for (int w = cl; w < prm.total_work; w += n_cl)
            for (int kc = 0; kc < n_kc; ++kc) {
                const uint32_t so = a.idx * a_slot_bytes;
                auto pack2 = [&](float a0, float a1) -> uint32_t {        // (a0 -> low half, a1 -> high half)
                    if (parts == 1 && prm.fp16) { const __half2 hh = __floats2half2_rn(a0, a1); return *reinterpret_cast<const uint32_t*>(&hh); }
                    const __nv_bfloat162 hb = __floats2bfloat162_rn(a0, a1);
                    return *reinterpret_cast<const uint32_t*>(&hb);
                };
                // the (hi, lo) x (re, im) parts of eight frames as four 16-byte stores
                auto store8 = [&](int j, const float2 (&yv)[8]) {
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
                        sts128(addr + ST_TILE, lr[0], lr[1], lr[2], lr[3]);
                        sts128(addr + im_off + ST_TILE, li[0], li[1], li[2], li[3]);
                    }
                };
                if constexpr (GROUPED) {
                    // 16 < M <= 64: accumulate over the tap groups; eight frames at a time so that the 16 partial sums,
                    // the 16 taps and the 23 rows of a half fit in registers
                    float2 ya[8], yb[8];
#pragma unroll
                    for (int g8 = 0; g8 < 8; ++g8) { ya[g8] = make_float2(0.f, 0.f); yb[g8] = make_float2(0.f, 0.f); }
                    for (int g = 0; g < n_groups; ++g) {
                        pq_x = SY_NOW();
                        mbar_wait(smem_u32(&ctl->in_full[in.idx]), in.phase);
                        pq_w += SY_NOW() - pq_x; pq_x = SY_NOW();
                        const uint32_t src = in_lane + in.idx * ST_IN_SLOT, tsrc = tap_lane + in.idx * ST_IN_SLOT;
                        float2 tap[16];
#pragma unroll
                        for (int m = 0; m < 16; ++m) {
                            if (REAL) tap[m] = lds_f2(tsrc + (uint32_t)m * 256u);
                            else { const float hh = lds_f1(tsrc + (uint32_t)m * 128u); tap[m] = make_float2(hh, hh); }
                        }
#pragma unroll
                        for (int j = 0; j < 2; ++j) {
                            float2 row[23];
#pragma unroll
                            for (int r = 0; r < 23; ++r) row[r] = lds_f2(src + (uint32_t)(8 * j + r) * 256u);
#pragma unroll
                            for (int m = 0; m < 16; ++m)
#pragma unroll
                                for (int g8 = 0; g8 < 8; ++g8) {
                                    if (j == 0) ya[g8] = ffma2(tap[m], row[g8 + 15 - m], ya[g8]);
                                    else        yb[g8] = ffma2(tap[m], row[g8 + 15 - m], yb[g8]);
                                }
                        }
                        __syncwarp();
                        if (lane == 0) mbar_arrive(smem_u32(&ctl->in_empty[in.idx]));
                        in.advance(ST_IN_SLOTS);
                        pq_c += SY_NOW() - pq_x;
                    }
                    pq_x = SY_NOW();
                    mbar_wait(smem_u32(&ctl->a_empty[a.idx]), a.phase ^ 1);
                    pq_w += SY_NOW() - pq_x; pq_x = SY_NOW();
                    store8(0, ya);
                    store8(1, yb);
                } else {
                pq_x = SY_NOW();
                mbar_wait(smem_u32(&ctl->in_full[in.idx]), in.phase);
                pq_w += SY_NOW() - pq_x; pq_x = SY_NOW();
                FirRegs<MT> rg;
                {
                    const uint32_t src = in_lane + in.idx * ST_IN_SLOT, tsrc = tap_lane + in.idx * ST_IN_SLOT;
                    if (MT > 0) {
#pragma unroll
                        for (int m = 0; m < WA; ++m) {
                            if (REAL) rg.tap[m] = lds_f2(tsrc + (uint32_t)m * 256u);        // one tap per real sample of the pair
                            else { const float hh = lds_f1(tsrc + (uint32_t)m * 128u); rg.tap[m] = make_float2(hh, hh); }
                        }
                    }
#pragma unroll
                    for (int j = 0; j < WA - 1 + FPW; ++j) rg.row[j] = lds_f2(src + (uint32_t)j * 256u);
                }
                // the window is in registers once its last load has returned: hand the input slot back to the TMA warp now,
                // a whole subfilter computation earlier than after the stores (the copy of the next chunk but one needs the lead)
                if (lane == 0) mbar_arrive_after(smem_u32(&ctl->in_empty[in.idx]), __float_as_uint(rg.row[WA - 2 + FPW].y));
                in.advance(ST_IN_SLOTS);
                pq_c += SY_NOW() - pq_x; pq_x = SY_NOW();
                mbar_wait(smem_u32(&ctl->a_empty[a.idx]), a.phase ^ 1);
                pq_w += SY_NOW() - pq_x; pq_x = SY_NOW();
                // polyphase MAC, eight frames at a time: eight independent FMA chains, then split + de-interleaved store
#pragma unroll
                for (int j = 0; j < FPW / 8; ++j) {
                    float2 yv[8];
                    if (MT > 1) {
#pragma unroll
                        for (int g = 0; g < 8; ++g) yv[g] = fmul2(rg.tap[0], rg.row[8 * j + g + WA - 1]);
#pragma unroll
                        for (int m = 1; m < WA; ++m)
#pragma unroll
                            for (int g = 0; g < 8; ++g) yv[g] = ffma2(rg.tap[m], rg.row[8 * j + g + WA - 1 - m], yv[g]);
                    } else {
#pragma unroll
                        for (int g = 0; g < 8; ++g) yv[g] = MT == 1 ? fmul2(rg.tap[0], rg.row[8 * j + g]) : rg.row[8 * j + g];
                    }
                    store8(j, yv);
                }
                }
                pq_c += SY_NOW() - pq_x; pq_x = SY_NOW();
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&ctl->a_full[a.idx]));
                a.advance(n_a);
                pq_f += SY_NOW() - pq_x;
            }
        if (SY_PROF && prm.prof && pw == 0 && lane == 0) {
            unsigned long long* pp = prm.prof + blockIdx.x * 16 + 12;
            pp[0] = SY_NOW() - pq_tot; pp[1] = pq_w; pp[2] = pq_c; pp[3] = pq_f;
        }
    }

    tc_fence_before();
    cluster_sync();
    if (warp == ALLOC_WARP) tmem_dealloc<CG>(tmem_base, 512);
}

// =====================================================================================
// Host side
// =====================================================================================
bool sym_supported(int P) { return P >= 64 && P <= kMaxP && P % 64 == 0; }

template <int MT, int PARTS, bool REAL, bool GROUPED = false>
static tina_status launch_symt(DevCtx* ctx, const Plan* plan, const CUtensorMap& tmap_out, const CUtensorMap& tmap_out2,
                               const CUtensorMap& tmap_x, const CUtensorMap& tmap_w, const SymParams& prm, int grid, cudaStream_t st)
{
    auto kern = pfb_symt_kernel<MT, PARTS, REAL, GROUPED>;
    tina_status as = ensure_smem(ctx, reinterpret_cast<const void*>(kern), (int)ST_SMEM_BYTES, "cudaFuncSetAttribute(pfb_symt_kernel)");
    if (as != TINA_OK) return as;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(UMMA_THREADS);
    cfg.dynamicSmemBytes = ST_SMEM_BYTES;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = UMMA_CG;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    SymParams prm2 = prm;
#ifdef TINA_DEV
    const bool prof = options().prof;
    if (prof) {
        cudaError_t pe = cudaMalloc(&prm2.prof, (size_t)grid * 16 * 8);
        if (pe == cudaSuccess) pe = cudaMemsetAsync(prm2.prof, 0, (size_t)grid * 16 * 8, st);
        if (pe != cudaSuccess) { if (prm2.prof) cudaFree(prm2.prof); return check_cuda(pe, "TINA_PROF counter buffer"); }
    }
#endif
    cudaError_t e = cudaLaunchKernelEx(&cfg, kern, plan->tmap32, tmap_out, tmap_out2, tmap_x, tmap_w, prm2);
#ifdef TINA_DEV
    if (prof) {
        std::vector<unsigned long long> h((size_t)grid * 16);
        cudaError_t pe = cudaStreamSynchronize(st);
        if (pe == cudaSuccess) pe = cudaMemcpy(h.data(), prm2.prof, h.size() * 8, cudaMemcpyDeviceToHost);
        cudaFree(prm2.prof);
        if (pe != cudaSuccess) return check_cuda(pe, "TINA_PROF counter read-back");
        double acc[16] = {0};
        for (int b = 0; b < grid; b += UMMA_CG) for (int i = 0; i < 16; ++i) acc[i] += (double)h[(size_t)b * 16 + i] / (grid / UMMA_CG);
        fprintf(stderr, "[tina prof symt] leader mean cycles: mma0 tot %.0f a_full %.0f b_full %.0f t_empty %.0f | mma1 tot %.0f a %.0f b %.0f t %.0f | epi tot %.0f t_full %.0f drain %.0f (first chain %.0f) | prod tot %.0f waits %.0f lds+mac+sts %.0f fence %.0f\n",
                acc[0], acc[1], acc[2], acc[3], acc[4], acc[5], acc[6], acc[7], acc[8], acc[9], acc[10], acc[11], acc[12], acc[13], acc[14], acc[15]);
    }
#endif
    count_launch();
    g_last_path = kPathUmma;
    note_kernel(GROUPED ? (REAL ? "pfb_symt_kernel<real, tap groups>" : "pfb_symt_kernel<tap groups>")
                        : (REAL ? "pfb_symt_kernel<real>" : "pfb_symt_kernel"), 0.5);
    if (e != cudaSuccess) return check_cuda(e, "pfb_symt_kernel launch");
    return check_cuda(cudaGetLastError(), "pfb_symt_kernel launch");
}

template <int MT, int PARTS>
static tina_status launch_sym(DevCtx* ctx, const CUtensorMap& tmap, const CUtensorMap& tmap_out, const CUtensorMap& tmap_out2,
                              const SymParams& prm, int grid, cudaStream_t st)
{
    auto kern = pfb_sym_kernel<MT, PARTS>;
    tina_status as = ensure_smem(ctx, reinterpret_cast<const void*>(kern), (int)SY_SMEM_BYTES, "cudaFuncSetAttribute(pfb_sym_kernel)");
    if (as != TINA_OK) return as;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(UMMA_THREADS);
    cfg.dynamicSmemBytes = SY_SMEM_BYTES;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = UMMA_CG;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    SymParams prm2 = prm;
#ifdef TINA_DEV
    const bool prof = options().prof;
    if (prof) {
        cudaError_t pe = cudaMalloc(&prm2.prof, (size_t)grid * 16 * 8);
        if (pe == cudaSuccess) pe = cudaMemsetAsync(prm2.prof, 0, (size_t)grid * 16 * 8, st);
        if (pe != cudaSuccess) { if (prm2.prof) cudaFree(prm2.prof); return check_cuda(pe, "TINA_PROF counter buffer"); }
    }
#endif
    cudaError_t e = cudaLaunchKernelEx(&cfg, kern, tmap, tmap_out, tmap_out2, prm2);
#ifdef TINA_DEV
    if (prof) {
        std::vector<unsigned long long> h((size_t)grid * 16);
        cudaError_t pe = cudaStreamSynchronize(st);
        if (pe == cudaSuccess) pe = cudaMemcpy(h.data(), prm2.prof, h.size() * 8, cudaMemcpyDeviceToHost);
        cudaFree(prm2.prof);
        if (pe != cudaSuccess) return check_cuda(pe, "TINA_PROF counter read-back");
        double acc[16] = {0};
        for (int b = 0; b < grid; b += UMMA_CG) for (int i = 0; i < 16; ++i) acc[i] += (double)h[(size_t)b * 16 + i] / (grid / UMMA_CG);
        fprintf(stderr, "[tina prof sym] leader mean cycles: mma0 tot %.0f a_full %.0f b_full %.0f t_empty %.0f | mma1 tot %.0f a %.0f b %.0f t %.0f | epi tot %.0f t_full %.0f drain %.0f | prod tot %.0f a_empty %.0f work+loads %.0f fence %.0f\n",
                acc[0], acc[1], acc[2], acc[3], acc[4], acc[5], acc[6], acc[7], acc[8], acc[9], acc[10], acc[12], acc[13], acc[14], acc[15]);
    }
#endif
    count_launch();
    g_last_path = kPathUmma;
    note_kernel("pfb_sym_kernel", 0.5);
    if (e != cudaSuccess) return check_cuda(e, "pfb_sym_kernel launch");
    return check_cuda(cudaGetLastError(), "pfb_sym_kernel launch");
}

bool sym_real_supported(int P) { return P >= 128 && P <= kMaxP && P % 64 == 0 && !options().sym_v1; }

// complex kind with P % 64 == 0, or real kind with P % 64 == 0 and P >= 128 (TMA-staged kernel only);
// window == nullptr (DFT batch, complex) or M <= 64 (M > 16: TMA-staged kernel only, taps in groups of 16)
tina_status sym_pfb(const void* x, int S, long long n_samples, int P, int M, const float* window, bool real, bool inverse,
                    tina_precision prec, void* out, cudaStream_t st)
{
    // complex kind with the row pairs folded as well (half the tensor work again): opt-in, it measured no faster
    if (!real && options().fold && symf_supported(P, M, window != nullptr))
        return symf_pfb(x, S, n_samples, P, M, window, inverse, prec, out, st);
    const long long NBLK = n_samples / P;
    const long long F = NBLK - M + 1;
    const int parts = prec == TINA_PREC_FP32 ? 2 : 1;
    const bool fp16 = prec == TINA_PREC_FP16;
    const Plan* plan = nullptr;
    tina_status ps = get_plan(P, real, inverse, parts, fp16, st, &plan, true);
    if (ps != TINA_OK) return ps;
    DevCtx* ctx = nullptr;
    if ((ps = dev_ctx(&ctx)) != TINA_OK) return ps;
    const bool staged = real || !options().sym_v1;                // TMA-staged input window (default) or register-window producers
    const int kdim = real ? P / 2 : P;                            // contraction length
    const int bins = real ? P / 4 : P / 2;                        // bins contracted (the rest are their mirrors)

    SymParams prm;
    memset(&prm, 0, sizeof(prm));
    prm.x = static_cast<const float*>(x);
    prm.window = window;
    prm.out = static_cast<float*>(out);
    prm.stream_stride = real ? n_samples : 2 * n_samples;
    prm.F = F;
    prm.NBLK = NBLK;
    prm.P = P;
    prm.M = M;
    prm.real = real ? 1 : 0;
    prm.tiles_per_stream = (int)((F + BM * UMMA_CG - 1) / (BM * UMMA_CG));
    prm.n_passes = (bins + SY_BINS - 1) / SY_BINS;
    const long long total = (long long)S * prm.tiles_per_stream * prm.n_passes;
    if (total > 0x7fffffffLL) return fail(TINA_ERR_UNSUPPORTED, "tina_pfb: too many tiles");
    prm.total_work = (int)total;
    prm.parts = parts;
    prm.fp16 = fp16 ? 1 : 0;
    const int kc_len = staged ? ST_KC : KC;                       // contraction elements per pipeline chunk
    prm.k_splits = (kdim + KSPLIT_MAX - 1) / KSPLIT_MAX;          // accumulation chains of <= 1024
    prm.kc_per_split = ((kdim / kc_len) + prm.k_splits - 1) / prm.k_splits;
    prm.debug = options().debug_skip;                             // 0 unless -DTINA_DEV
    const int n_cl = ctx->n_sm / UMMA_CG;
    const int grid = UMMA_CG * (prm.total_work < n_cl ? prm.total_work : n_cl);

    EncodeTiledFn enc = encode_fn();
    if (!enc) return fail(TINA_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found");
    const cuuint32_t estr[3] = {1, 1, 1};
    // Output maps (complex kind) over [S][F][2P] floats: 32 x 32 swizzled boxes, and 28-float-wide dense boxes for
    // the mirrored tile of a pass's last step (see the epilogue).  The real kind stores from registers.
    CUtensorMap tmap_out, tmap_out2;
    memset(&tmap_out, 0, sizeof(tmap_out));
    memset(&tmap_out2, 0, sizeof(tmap_out2));
    // the four maps of a call are a pure function of (pointers, shape): repeated calls skip the encodes
    static_assert(sizeof(CUtensorMap) == 128, "TmapSet layout");
    TmapKey tkey;
    memset(&tkey, 0, sizeof(tkey));
    tkey.p[0] = x; tkey.p[1] = window; tkey.p[2] = out;
    tkey.n[0] = n_samples;
    tkey.i[0] = S; tkey.i[1] = P; tkey.i[2] = M; tkey.i[3] = real ? 1 : 0; tkey.i[4] = staged ? 1 : 0; tkey.i[5] = 1;   // tag 1: sym_pfb
    // real kind: the TMA epilogue views the output as row PAIRS, which needs an even number of frames per stream
    // (an odd F is fine for ONE stream: its last row is stored from registers)
    prm.real_tma = (real && F >= 2 && (F % 2 == 0 || S == 1) && !options().no_out_tma) ? 1 : 0;
    tkey.i[4] += 2 * prm.real_tma;
    TmapSet tset;
    const bool cached = tmap_cache_get(ctx, tkey, &tset);
    if (cached) { memcpy(&tmap_out, tset.m[0], 128); memcpy(&tmap_out2, tset.m[1], 128); }
    if (!real && !cached) {
        const cuuint64_t dims[3] = {(cuuint64_t)2 * P, (cuuint64_t)F, (cuuint64_t)S};
        const cuuint64_t strides[2] = {(cuuint64_t)2 * P * sizeof(float), (cuuint64_t)F * 2 * P * sizeof(float)};
        const cuuint32_t box[3] = {32, 32, 1};
        CUresult r = enc(&tmap_out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, out, dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                         CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        const cuuint32_t box2[3] = {28, 32, 1};
        if (r == CUDA_SUCCESS)
            r = enc(&tmap_out2, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, out, dims, strides, box2, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                    CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return fail(TINA_ERR_CUDA, "cuTensorMapEncodeTiled(out) failed (%d)", (int)r);
    }
    if (real && prm.real_tma && !cached) {
        // output as [S][F/2][2 (P + 2)] floats: 16-row boxes of 32 floats (swizzled) and of 28 floats (dense)
        const cuuint64_t dims[3] = {(cuuint64_t)2 * (P + 2), (cuuint64_t)(F / 2), (cuuint64_t)S};
        const cuuint64_t strides[2] = {(cuuint64_t)2 * (P + 2) * sizeof(float), (cuuint64_t)(F + (F & 1)) * (P + 2) * sizeof(float)};
        const cuuint32_t box[3] = {32, 16, 1};
        CUresult r = enc(&tmap_out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, out, dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                         CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        const cuuint32_t box2[3] = {28, 16, 1};
        if (r == CUDA_SUCCESS)
            r = enc(&tmap_out2, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, out, dims, strides, box2, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                    CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return fail(TINA_ERR_CUDA, "cuTensorMapEncodeTiled(out, row pairs) failed (%d)", (int)r);
    }
    if (staged) {
        // input as [S][NB][row] floats (row = 2P complex, P real), boxes of 64 floats (32 complex columns / 32 pairs of
        // real samples) x (128 + MT - 1) rows; the window as [M][P] floats, boxes of (32 | 64) x MT (rows >= M read as zeros)
        const int MT = !window ? 0 : (M <= 4 ? 4 : (M <= 8 ? 8 : 16));
        if (M > kMaxTapsPfb) return fail(TINA_ERR_UNSUPPORTED, "tina_pfb: at most %d taps", kMaxTapsPfb);
        const long long row_f = real ? P : 2LL * P;
        CUtensorMap tmap_x, tmap_w;
        memset(&tmap_x, 0, sizeof(tmap_x));
        memset(&tmap_w, 0, sizeof(tmap_w));
        if (cached) { memcpy(&tmap_x, tset.m[2], 128); memcpy(&tmap_w, tset.m[3], 128); }
        else {
        const cuuint64_t xdims[3] = {(cuuint64_t)row_f, (cuuint64_t)NBLK, (cuuint64_t)S};
        const cuuint64_t xstrides[2] = {(cuuint64_t)row_f * sizeof(float),
                                        S > 1 ? (cuuint64_t)prm.stream_stride * sizeof(float) : (cuuint64_t)NBLK * row_f * sizeof(float)};
        const cuuint32_t xbox[3] = {64, (cuuint32_t)(BM + (MT > 0 ? MT : 1) - 1), 1};
        CUresult r = enc(&tmap_x, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<void*>(x), xdims, xstrides, xbox, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                         CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r == CUDA_SUCCESS && MT > 0) {
            const cuuint64_t wdims[2] = {(cuuint64_t)P, (cuuint64_t)M};
            const cuuint64_t wstrides[1] = {(cuuint64_t)P * sizeof(float)};
            const cuuint32_t wbox[2] = {real ? 64u : 32u, (cuuint32_t)MT};
            r = enc(&tmap_w, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float*>(window), wdims, wstrides, wbox, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                    CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        }
        if (r != CUDA_SUCCESS) return fail(TINA_ERR_CUDA, "cuTensorMapEncodeTiled(input) failed (%d)", (int)r);
        memcpy(tset.m[0], &tmap_out, 128); memcpy(tset.m[1], &tmap_out2, 128);
        memcpy(tset.m[2], &tmap_x, 128); memcpy(tset.m[3], &tmap_w, 128);
        tmap_cache_put(ctx, tkey, tset);
        }
#define TINA_SYMT2(MT_, R_) (parts == 2 ? launch_symt<MT_, 2, R_>(ctx, plan, tmap_out, tmap_out2, tmap_x, tmap_w, prm, grid, st) \
                                        : launch_symt<MT_, 1, R_>(ctx, plan, tmap_out, tmap_out2, tmap_x, tmap_w, prm, grid, st))
#define TINA_SYMT(MT_) (real ? TINA_SYMT2(MT_, true) : TINA_SYMT2(MT_, false))
        if (MT == 0) return real ? fail(TINA_ERR_UNSUPPORTED, "real kind needs a window") : TINA_SYMT2(0, false);
        if (MT == 4) return TINA_SYMT(4);
        if (MT == 8) return TINA_SYMT(8);
        if (M > 16) {                                              // taps in groups of 16, accumulated in registers
            if (real) return parts == 2 ? launch_symt<16, 2, true, true>(ctx, plan, tmap_out, tmap_out2, tmap_x, tmap_w, prm, grid, st)
                                        : launch_symt<16, 1, true, true>(ctx, plan, tmap_out, tmap_out2, tmap_x, tmap_w, prm, grid, st);
            return parts == 2 ? launch_symt<16, 2, false, true>(ctx, plan, tmap_out, tmap_out2, tmap_x, tmap_w, prm, grid, st)
                              : launch_symt<16, 1, false, true>(ctx, plan, tmap_out, tmap_out2, tmap_x, tmap_w, prm, grid, st);
        }
        return TINA_SYMT(16);
#undef TINA_SYMT
#undef TINA_SYMT2
    }
#define TINA_SYM(MT_) (parts == 2 ? launch_sym<MT_, 2>(ctx, plan->tmap, tmap_out, tmap_out2, prm, grid, st) \
                                  : launch_sym<MT_, 1>(ctx, plan->tmap, tmap_out, tmap_out2, prm, grid, st))
    if (!window) return TINA_SYM(0);
    if (M <= 4) return TINA_SYM(4);
    if (M <= 8) return TINA_SYM(8);
    return TINA_SYM(16);
#undef TINA_SYM
}

}  // namespace tina
