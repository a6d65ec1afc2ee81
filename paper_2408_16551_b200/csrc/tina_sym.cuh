// tina_sym.cuh -- pieces shared by the column-paired dense kernels (tina_sym.cu) and the row-and-column-paired one
// (tina_symf.cu): parameter block, the development-build macros, small PTX helpers and the complex-kind epilogue.
#pragma once
#include "tina_umma.cuh"

namespace tina {

using namespace ptx;

constexpr int SY_BINS = 128;                              // bins per pass: D1 + D2 = 4 x 128 = 512 TMEM columns
constexpr int SY_A_RING = 128 * 1024;                     // 2 slots of 64 KB (bf16x3) or 4 of 32 KB (single pass)
constexpr int SY_B_ENTRY = B_ENTRY_BYTES / UMMA_CG;       // 16 KB per CTA
constexpr int SY_B_ENTRIES = 4;
constexpr int SY_STAGE = 8192;                            // per epilogue warp: forward + mirrored 32 x 32 fp32 tiles
constexpr size_t SY_SMEM_BYTES = SY_A_RING + SY_B_ENTRIES * SY_B_ENTRY + 4 * SY_STAGE + sizeof(SmemCtl);
static_assert(SY_SMEM_BYTES <= 232448, "exceeds the 227 KB shared memory opt-in limit");

struct SymParams {
    const float* x;            // [S][stream_stride] floats (interleaved complex64)
    const float* window;       // [M][P] or nullptr (plain DFT batch)
    float* out;                // [S][F][2P] floats
    long long stream_stride;   // floats between streams of x
    long long F, NBLK;
    int P, M;
    int tiles_per_stream, n_passes, total_work;
    int parts;                 // 2: bf16x3, 1: single pass
    int fp16;
    int k_splits, kc_per_split;
    int real;                  // 1: real kind (pfb_symt_kernel<.., REAL = true>): x is float32, out rows are P + 2 floats
    int real_tma;              // real kind: tiles leave through row-pair tensor maps (even F); 0: register / shared-memory stores
    int debug;                 // -DTINA_DEV only (TINA_DEBUG_SKIP): 16 no mirrored-tile stores, 32 no forward-tile stores
    unsigned long long* prof;  // -DTINA_DEV only (TINA_PROF): [grid][16] cycle counters
};

#ifdef TINA_DEV
#define SY_DBG(bit) (prm.debug & (bit))
#define SY_NOW() (prm.prof ? clock64() : 0LL)
#define SY_PROF 1
#else
#define SY_DBG(bit) 0
#define SY_NOW() 0LL
#define SY_PROF 0
#endif

__device__ __forceinline__ float2 lds_f2(uint32_t addr)
{
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ float lds_f1(uint32_t addr)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}

__device__ __forceinline__ uint64_t l2_policy_evict_last()
{
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void st_f2_evict_last(float2* g, float2 v, uint64_t pol)
{
    asm volatile("st.global.L2::cache_hint.v2.f32 [%0], {%1, %2}, %3;" ::"l"(g), "f"(v.x), "f"(v.y), "l"(pol) : "memory");
}
__device__ __forceinline__ void sts16(uint32_t addr, uint32_t v)
{
    asm volatile("st.shared.b16 [%0], %1;" ::"r"(addr), "h"((unsigned short)v) : "memory");
}


struct EpiCtx {
    uint32_t t_full0, t_full1, t_empty0, t_empty1;   // shared-memory addresses of the accumulator barriers
    uint32_t stage, tmem_base, rank;
    int cl, n_cl;
};

// Epilogue of one lane quarter q (a warp): see the comment inside.  Shared by both kernels of this file.
// FOLD = false: D1 = TMEM columns 0-255 holds (U, Z) interleaved per bin, D2 = 256-511 holds (W, V) (tina_sym.cu).
// FOLD = true: four accumulators of 128 columns, U | Z | W | V, one column per bin (tina_symf.cu).
template <bool FOLD>
__device__ __forceinline__ void sym_epilogue(const SymParams& prm, const CUtensorMap* tmap_out, const CUtensorMap* tmap_out2,
                                             const EpiCtx& e, const int q, const int lane)
{
    constexpr int CG = UMMA_CG;
    const int P = prm.P, half = P >> 1, npg = prm.n_passes;
    // ============================ epilogue ==============================================
    // Lane = frame (TMEM lane); a step takes 32 accumulator columns = 16 bins kb .. kb+15 from D1 (U, Z) and
    // D2 (W, V).  Forward tile: bins kb .. kb+15, stored by TMA at column 2 kb.  The mirrored bins P-kb-j are
    // one bin off any 16-byte-aligned tile (TMA needs 16-byte-aligned box starts), so the mirrored tile is
    // the ALIGNED group P-kb-16 .. P-kb-1 = the mirrors of j = 1 .. 16, j = 16 being the first bin of the next
    // step (two extra TMEM columns are read for it).  What does not fit that scheme is stored from registers,
    // 8 bytes per row: the mirror of a pass's first bin (j = 0; none for bin 0, whose "mirror" is bin 0 itself),
    // the mirror of j = 15 in the pass's last step (whose tile goes out 28 floats wide through a second map,
    // because j = 16 belongs to the next pass), and the Nyquist bin.
            const uint32_t sb_f = e.stage + (uint32_t)q * SY_STAGE, sb_m = sb_f + 4096u;
    const uint32_t taddr = e.tmem_base + ((uint32_t)(q * 32) << 16);
    const uint32_t rowoff = (uint32_t)lane * 128u, sw = (uint32_t)lane & 7u;
    uint32_t tf_phase = 0;
    // ONE elected thread per warp issues every TMA store and waits on their bulk groups (the groups belong to the thread
    // that committed them).  Elected rather than `lane == 0`: ptxas then knows a single thread is active and emits the
    // uniform-datapath instructions straight instead of inside an any-thread loop.
    const bool issuer = elect_one();
    // several accumulation chains (P > 1024): the first chain's tiles are stored with an L2 evict-last policy so that
    // the later chains' add-reduce finds them resident
    const bool keep_l2 = prm.k_splits > 1;
    const uint64_t pol_keep = l2_policy_evict_last();
    long long pe_w = 0, pe_d = 0, pe_x, pe_tot = SY_NOW();
    for (int w = e.cl; w < prm.total_work; w += e.n_cl) {
        const int tile = w / npg;
        const int k0 = (w % npg) * SY_BINS;
        const int ncol = 2 * min(SY_BINS, half - k0);
        const int s = tile / prm.tiles_per_stream;
        const long long row0 = (long long)(tile % prm.tiles_per_stream) * (BM * CG) + e.rank * BM + q * 32;
        const bool row_ok = lane < (int)min(32LL, prm.F - row0);
        float* const orow = prm.out + ((long long)s * prm.F + row0 + lane) * (2LL * P);
        for (int ks = 0; ks < prm.k_splits; ++ks) {
            if (ks > 0 && issuer) bulk_wait<0>();          // the previous chain's stores to this tile are complete
            pe_x = SY_NOW();
            mbar_wait<256>(e.t_full0, tf_phase);
            mbar_wait<256>(e.t_full1, tf_phase);
            pe_w += SY_NOW() - pe_x; pe_x = SY_NOW();
            tf_phase ^= 1u;
            tc_fence_after();
            // one bin (complex value) straight from registers: plain store for the first chain, fp32 add at L2 after
            auto put = [&](int bin, float re, float im) {
                if (row_ok && !SY_DBG(16)) {
                    float2* g = reinterpret_cast<float2*>(orow + 2 * bin);
                    if (ks > 0) atomicAdd(g, make_float2(re, im)); else *g = make_float2(re, im);
                }
            };
            uint32_t r1[32], r2[32], e1[2] = {0u, 0u}, e2[2] = {0u, 0u};
            // load the 16 bins starting at accumulator column pair `c` (in interleaved (U, Z) / (W, V) order either way)
            auto load16 = [&](int c) {
                if (!FOLD) { tmem_ld32(taddr + c, r1); tmem_ld32(taddr + 256u + c, r2); return; }
                uint32_t u[16], z[16], ww[16], v[16];
                tmem_ld16(taddr + (c >> 1), u); tmem_ld16(taddr + 128u + (c >> 1), z);
                tmem_ld16(taddr + 256u + (c >> 1), ww); tmem_ld16(taddr + 384u + (c >> 1), v);
                tmem_ld_wait();
#pragma unroll
                for (int j = 0; j < 16; ++j) { r1[2 * j] = u[j]; r1[2 * j + 1] = z[j]; r2[2 * j] = ww[j]; r2[2 * j + 1] = v[j]; }
            };
            auto load_extra = [&](int c) {                      // the first bin of the next step (j = 16)
                if (!FOLD) { tmem_ld2(taddr + c, e1); tmem_ld2(taddr + 256u + c, e2); return; }
                uint32_t t0[2], t1[2], t2[2], t3[2];
                tmem_ld2(taddr + (c >> 1), t0); tmem_ld2(taddr + 128u + (c >> 1), t1);
                tmem_ld2(taddr + 256u + (c >> 1), t2); tmem_ld2(taddr + 384u + (c >> 1), t3);
                tmem_ld_wait();
                e1[0] = t0[0]; e1[1] = t1[0]; e2[0] = t2[0]; e2[1] = t3[0];
            };
            load16(0);
            if (32 < ncol) load_extra(32);
            for (int cb = 0; cb < ncol; cb += 32) {
                const int kb = k0 + (cb >> 1);
                const bool last = cb + 32 >= ncol;
                tmem_ld_wait();
                if (last) {
                    // both accumulators have been read out completely: hand them back to the MMA warps
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) {
                        arrive_leader<CG>(e.t_empty0, e.rank, 0);
                        arrive_leader<CG>(e.t_empty1, e.rank, 0);
                    }
                    pe_d += SY_NOW() - pe_x;                  // accumulator wait -> release: the exposed drain
                }
#define SY_F(v) __uint_as_float(v)
                if (kb == 0) {
                    // bin 0: its sine column carries (-1)^p, i.e. r1[1] + i r2[1] = X[P/2] (unpaired)
                    put(half, SY_F(r1[1]), SY_F(r2[1]));
                    r1[1] = 0u; r2[1] = 0u;                  // V = Z = 0 for bin 0: X[0] = U + i W
                } else if (cb == 0) {
                    put(P - kb, SY_F(r1[0]) - SY_F(r2[1]), SY_F(r2[0]) + SY_F(r1[1]));          // mirror of j = 0
                }
                if (last) put(P - kb - 15, SY_F(r1[30]) - SY_F(r2[31]), SY_F(r2[30]) + SY_F(r1[31]));   // mirror of j = 15
                if (issuer) bulk_wait_read<1>();           // the forward tile of the previous step has been read
                __syncwarp();
#pragma unroll
                for (int g = 0; g < 8; ++g) {
                    const float U0 = SY_F(r1[4 * g]), Z0 = SY_F(r1[4 * g + 1]), U1 = SY_F(r1[4 * g + 2]), Z1 = SY_F(r1[4 * g + 3]);
                    const float W0 = SY_F(r2[4 * g]), V0 = SY_F(r2[4 * g + 1]), W1 = SY_F(r2[4 * g + 2]), V1 = SY_F(r2[4 * g + 3]);
                    sts128(sb_f + rowoff + (((uint32_t)g ^ sw) << 4), __float_as_uint(U0 + V0), __float_as_uint(W0 - Z0),
                           __float_as_uint(U1 + V1), __float_as_uint(W1 - Z1));
                }
                fence_proxy_async();
                __syncwarp();
                if (issuer) {
                    if (SY_DBG(32)) { }
                    else if (ks == 0 && keep_l2) tma_store_3d_hint(tmap_out, sb_f, 2 * kb, (int)row0, s, pol_keep);
                    else if (ks == 0) tma_store_3d(tmap_out, sb_f, 2 * kb, (int)row0, s);
                    else              tma_reduce_add_3d(tmap_out, sb_f, 2 * kb, (int)row0, s);
                    bulk_commit();
                    bulk_wait_read<1>();                      // the mirrored tile of the previous step has been read
                }
                __syncwarp();
                // mirrored tile: position t <-> bin P-kb-16+t <-> j = 16 - t; 16-byte chunk c holds j = 16-2c, 15-2c
                // = accumulator columns 32-4c .. 33-4c and 30-4c .. 31-4c (columns 32, 33 = e1 / e2)
#pragma unroll
                for (int c = 0; c < 8; ++c) {
                    const float Ua = SY_F(c ? r1[32 - 4 * c] : e1[0]), Za = SY_F(c ? r1[33 - 4 * c] : e1[1]);
                    const float Wa = SY_F(c ? r2[32 - 4 * c] : e2[0]), Va = SY_F(c ? r2[33 - 4 * c] : e2[1]);
                    const float Ub = SY_F(r1[30 - 4 * c]), Zb = SY_F(r1[31 - 4 * c]);
                    const float Wb = SY_F(r2[30 - 4 * c]), Vb = SY_F(r2[31 - 4 * c]);
                    if (!last)
                        sts128(sb_m + rowoff + (((uint32_t)c ^ sw) << 4), __float_as_uint(Ua - Va), __float_as_uint(Wa + Za),
                               __float_as_uint(Ub - Vb), __float_as_uint(Wb + Zb));
                    else if (c > 0)                              // last step of the pass: dense rows of 28 floats, positions 2 .. 15
                        sts128(sb_m + (uint32_t)lane * 112u + (uint32_t)(c - 1) * 16u, __float_as_uint(Ua - Va), __float_as_uint(Wa + Za),
                               __float_as_uint(Ub - Vb), __float_as_uint(Wb + Zb));
                }
#undef SY_F
                if (!last) {
                    load16(cb + 32);
                    if (cb + 64 < ncol) load_extra(cb + 64);
                }
                fence_proxy_async();
                __syncwarp();
                if (issuer) {
                    if (SY_DBG(16)) { }
                    else if (!last) {
                        const int cm = 2 * (P - kb - 16);
                        if (ks == 0 && keep_l2) tma_store_3d_hint(tmap_out, sb_m, cm, (int)row0, s, pol_keep);
                        else if (ks == 0) tma_store_3d(tmap_out, sb_m, cm, (int)row0, s);
                        else         tma_reduce_add_3d(tmap_out, sb_m, cm, (int)row0, s);
                    } else {
                        const int cm = 2 * (P - kb - 14);
                        if (ks == 0 && keep_l2) tma_store_3d_hint(tmap_out2, sb_m, cm, (int)row0, s, pol_keep);
                        else if (ks == 0) tma_store_3d(tmap_out2, sb_m, cm, (int)row0, s);
                        else         tma_reduce_add_3d(tmap_out2, sb_m, cm, (int)row0, s);
                    }
                    bulk_commit();
                }
            }
        }
    }
    if (issuer) bulk_wait<0>();                               // staging tiles must outlive their TMA reads
    if (SY_PROF && prm.prof && q == 0 && lane == 0) {
        unsigned long long* pp = prm.prof + blockIdx.x * 16 + 8;
        pp[0] = SY_NOW() - pe_tot; pp[1] = pe_w; pp[2] = pe_d;
    }
}


}  // namespace tina
