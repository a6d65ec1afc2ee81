// tina_umma.cu -- the fused PFB / DFT kernel of libtina on the sm_100a tensor cores.
//
// One persistent, warp-specialised kernel computes, per tile of frames,
//     y[f][c]   = sum_m w[m][c] * x[f + M-1-m][c]          (Eq. (20); CUDA cores)
//     out[f][n] = sum_c y[f][c] * T[c][n]                   (Eq. (12)-(13); tcgen05)
// where x is viewed as a real [NB][K] matrix (K = 2P interleaved re/im for the complex kind,
// K = P for the real kind), and T is the real block form of the Fourier matrix (N = K columns).
// y is split on the fly into bf16 hi + lo parts and written straight into the swizzled shared
// memory tiles the MMA consumes: the subfiltered signal never touches HBM.  fp32 accuracy
// comes from the error-compensated product  y*T ~= y_lo*T_hi + y_hi*T_hi + y_hi*T_lo  (bf16x3,
// fp32 accumulation in TMEM); TINA_PREC_BF16 issues the single y_hi*T_hi pass.
//
// Launched as clusters of two CTAs (one per SM of a TPC pair) running tcgen05.mma.cta_group::2: the
// pair owns a 256-frame x 512-column tile, each CTA supplies its own 128 frames of A and half of every
// twiddle tile.  Accumulation chains are kept to 1024 contraction elements (the tensor-core fp32
// accumulator truncates: DESIGN.md section 7); later chains are added into the output in fp32.
//
// Warp roles (512 threads, 1 CTA per SM):
//   warps 0-7   FIR producers: polyphase MAC in fp32 registers (fma.rn.f32x2) -> bf16 hi/lo -> A ring
//   warps 8-11  epilogue: tcgen05.ld (TMEM -> registers) -> swizzled staging tile -> TMA store / add-reduce
//   warp 12     TMA producer: twiddle half-tiles T_hi / T_lo -> B ring (SWIZZLE_128B), barrier on the leader
//   warps 13,15 MMA issuers of the leader CTA, one per 256-column accumulator half (kind::f16, M=256, K=16);
//               the peer's warp 13 forwards "A tile ready" to the leader
//   warp 14     TMEM allocator
// The same kernel serves the standalone DFT (no window) and the Toeplitz FIR (overlapping A rows, N != K).
#include "tina_umma.cuh"

#include <atomic>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <tuple>
#include <vector>

namespace tina {

using namespace ptx;


struct UmmaParams {
    const float* x;            // [S][stream_stride] floats
    const float* window;       // [M][P] or nullptr (M == 1, unit taps)
    float* out;                // [S][F][out_row] floats
    long long stream_stride;   // floats between streams of x
    long long F, NBLK;         // frames per stream, input blocks per stream
    long long out_row;         // floats per output row (complex: 2P, real: P+2)
    long long out_stream_stride; // floats between streams of out (F * out_row; FIR: L - M + 1)
    int K;                     // GEMM K: floats of one A row (multiple of 64)
    int N;                     // GEMM N: output columns (= K for the PFB / DFT; block length for the Toeplitz FIR)
    long long x_row_stride;    // floats between consecutive A rows (= K for the PFB / DFT; block length for the FIR)
    long long x_len;           // 0, or number of valid floats per stream: elements beyond it read as zero (FIR)
    long long out_len;         // (scalar store mode) valid output floats per stream
    int a_ring_bytes, b_ring_bytes, stage_bytes;   // shared-memory carve-up (defaults A_RING_BYTES / B_RING_BYTES / EPI_STAGE_BYTES)
    int out_scalar;            // 1: epilogue stores rows of N contiguous floats, 4-byte aligned, clipped at out_len (FIR)
    int P, M;
    int tiles_per_stream, n_passes, total_work;
    int nt_pass;               // accumulator columns per pass
    int parts;                 // 2: bf16x3 (hi+lo), 1: single pass
    int fp16;                  // 1: the single pass uses fp16 operands (TINA_PREC_FP16)
    unsigned long long* prof;  // optional [grid][16] cycle counters (TINA_PROF=1, diagnostics only)
    int out_tma;               // 1: epilogue leaves through TMA tensor stores (always for the complex kind)
    int debug;                 // TINA_DEBUG_SKIP bits (1: no FIR work, 2: no epilogue global traffic, 4: no MMAs, 8: no TMA)
    int k_splits, kc_per_split; // accumulation chains per tile
};

// =====================================================================================
// Plan: twiddle matrix Tt[part][n][c] (bf16, "K-major" = row n holds the K contraction index)
// built on the device from float64 sincospi, + its TMA tensor map.
// =====================================================================================
// sym = 1 (complex kind, column-paired contraction of tina_sym.cu): a P x P matrix, row n = 2k + j for the bin
// k in [0, P/2): j = 0 cos(2 pi p k / P), j = 1 sin(2 pi p k / P) (inverse: -sin) against the contraction index
// c = p; row 1 (sin of bin 0, identically zero) carries the Nyquist column (-1)^p instead.
__global__ void twiddle_kernel(__nv_bfloat16* __restrict__ tt, int P, int real, int inverse, int parts, int fp16, int sym)
{
    const int N = (real || sym) ? P : 2 * P;
    const int Kd = (real && sym) ? P / 2 : N;          // contraction length (row length); real + sym: sample PAIRS
    const long long total = (long long)N * Kd;
    const double scale = inverse ? 1.0 / (double)P : 1.0;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total;
         e += (long long)gridDim.x * blockDim.x) {
        const int n = (int)(e / Kd), c = (int)(e % Kd);
        double v;
        if (sym && real) {
            // real kind, column-paired (tina_sym.cu): rows [eo][2k + j], eo = 0 the even samples p = 2q, eo = 1 the odd
            // samples p = 2q + 1, k in [0, P/4): j = 0 cos(2 pi p k / P), j = 1 sin(2 pi p k / P); the sine rows of
            // bin 0 (identically zero) carry (-1)^q, which gives the unpaired bin P/4
            const int eo = n / (P / 2), nn = n % (P / 2);
            if (nn == 1) v = (c & 1) ? -1.0 : 1.0;
            else {
                const int k = nn >> 1;
                const long long r = ((long long)(2 * c + eo) * k) % P;
                double sn, cs;
                sincospi(2.0 * (double)r / (double)P, &sn, &cs);
                v = (nn & 1) ? sn : cs;
            }
        } else if (sym) {
            if (n == 1) v = (c & 1) ? -1.0 : 1.0;
            else {
                const int k = n >> 1;
                const long long r = ((long long)c * k) % P;
                double sn, cs;
                sincospi(2.0 * (double)r / (double)P, &sn, &cs);
                v = (n & 1) ? (inverse ? -sn : sn) : cs;
            }
        } else if (real) {
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
        if (fp16) { reinterpret_cast<__half*>(tt)[e] = __double2half(v); continue; }   // single part only
        const __nv_bfloat16 hi = __double2bfloat16(v);
        tt[e] = hi;
        if (parts > 1) tt[total + e] = __double2bfloat16(v - (double)__bfloat162float(hi));
    }
}

using PlanKey = std::tuple<int, int, int, int, int, int, int>;   // device, P, real, inverse, parts, fp16, sym
static std::mutex g_plan_mu;
static std::map<PlanKey, Plan> g_plans;


EncodeTiledFn encode_fn()
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

tina_status get_plan(int P, bool real, bool inverse, int parts, bool fp16, cudaStream_t st, const Plan** out, bool sym)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return check_cuda(e, "cudaGetDevice");
    std::lock_guard<std::mutex> lk(g_plan_mu);
    const PlanKey key{dev, P, real ? 1 : 0, inverse ? 1 : 0, parts, fp16 ? 1 : 0, sym ? 1 : 0};
    auto it = g_plans.find(key);
    if (it != g_plans.end()) { *out = &it->second; return TINA_OK; }

    const int N = (real || sym) ? P : 2 * P;
    const int Kd = (real && sym) ? P / 2 : N;           // row length (contraction elements)
    Plan pl;
    const size_t bytes = (size_t)parts * N * Kd * sizeof(__nv_bfloat16);
    e = cudaMalloc(&pl.tt, bytes);
    if (e != cudaSuccess) return check_cuda(e, "cudaMalloc(twiddles)");
    twiddle_kernel<<<592, 256, 0, st>>>(pl.tt, P, real ? 1 : 0, inverse ? 1 : 0, parts, fp16 ? 1 : 0, sym ? 1 : 0);
    count_launch();
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { cudaFree(pl.tt); return check_cuda(e, "twiddle_kernel"); }

    EncodeTiledFn enc = encode_fn();
    if (!enc) { cudaFree(pl.tt); return fail(TINA_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found"); }
    const cuuint64_t dims[2] = {(cuuint64_t)Kd, (cuuint64_t)parts * N};      // innermost (K) first
    const cuuint64_t strides[1] = {(cuuint64_t)Kd * sizeof(__nv_bfloat16)};
    const int nb_rows = (real && sym) ? N / 2 : N;       // rows of one matrix (real + sym: even- and odd-sample halves)
    const cuuint32_t box[2] = {(cuuint32_t)KC, (cuuint32_t)((nb_rows < NSUB ? nb_rows : NSUB) / UMMA_CG)};
    const cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(&pl.tmap, fp16 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT16 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, pl.tt, dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                     CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    memset(&pl.tmap32, 0, sizeof(pl.tmap32));
    if (r == CUDA_SUCCESS && sym) {
        const cuuint32_t box32[2] = {32, box[1]};
        r = enc(&pl.tmap32, fp16 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT16 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, pl.tt, dims, strides, box32, estr,
                CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_64B,
                CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    }
    if (r != CUDA_SUCCESS) { cudaFree(pl.tt); return fail(TINA_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r); }
    auto ins = g_plans.emplace(key, pl);
    *out = &ins.first->second;
    return TINA_OK;
}

const __nv_bfloat16* umma_twiddle_plan(int P, bool real, bool inverse, cudaStream_t st, tina_status* status)
{
    const Plan* pl = nullptr;
    *status = get_plan(P, real, inverse, 2, false, st, &pl);
    return *status == TINA_OK ? pl->tt : nullptr;
}

void umma_clear_plans()
{
    std::lock_guard<std::mutex> lk(g_plan_mu);
    for (auto& kv : g_plans) cudaFree(kv.second.tt);
    g_plans.clear();
}


// Development-only instrumentation (-DTINA_DEV): TINA_DEBUG_SKIP role-skipping bits and the TINA_PROF
// in-kernel cycle counters.  The default build compiles both out: no knob can skip work.
#ifdef TINA_DEV
#define TINA_DBG(bit) (prm.debug & (bit))
#define PF_NOW() (prm.prof ? clock64() : 0LL)
#define PF_ON() (prm.prof != nullptr)
#else
#define TINA_DBG(bit) 0
#define PF_NOW() 0LL
#define PF_ON() false
#endif

// =====================================================================================
// The fused kernel.  MT = compile-time tap count the sliding window is unrolled for
// (taps m >= M are zero; MT == 0: no window, y = x, i.e. a plain DFT batch).
// =====================================================================================
template <int MT, bool REAL, int CG, bool SHARE>
__global__ void __launch_bounds__(UMMA_THREADS, 1)
pfb_umma_kernel(const __grid_constant__ CUtensorMap tmap_b, const __grid_constant__ CUtensorMap tmap_out,
                const __grid_constant__ CUtensorMap tmap_out2, const UmmaParams prm)
{
    extern __shared__ __align__(1024) uint8_t smem[];           // dynamic shared memory starts 1024-byte aligned (checked below)
    if ((smem_u32(smem) & 1023u) != 0) __trap();                // the swizzled tiles need 1024-byte alignment
    uint8_t* a_ring = smem;
    uint8_t* b_ring = smem + prm.a_ring_bytes;
    uint8_t* stage = b_ring + prm.b_ring_bytes;                         // 4 epilogue warps x EPI_STAGE_BYTES (1024-aligned)
    SmemCtl* ctl = reinterpret_cast<SmemCtl*>(stage + 4 * prm.stage_bytes);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int parts = prm.parts;
    const uint32_t a_slot_bytes = A_PART_BYTES * parts;
    const uint32_t n_a = (uint32_t)prm.a_ring_bytes / a_slot_bytes;            // 4 (bf16x3) or 8 (single pass)
    const int N = prm.N;
    const int n_kc = prm.K / KC;
    const int NTP = prm.nt_pass;                                  // accumulator columns per pass (256 or 512)
    const int nt_max = N < NTP ? N : NTP;
    const uint32_t n_acc = nt_max <= 256 ? 2 : 1;                 // TMEM accumulator stages
    // cta_group::2: the CTA pair shares every twiddle tile (each CTA stages half of its N rows) and
    // the leader (rank 0) issues M=256 MMAs over both CTAs' A tiles; barriers the leader waits on
    // live in the leader's shared memory and are signalled remotely by the peer.
    // SHARE: clusters of four = two CTA pairs working on the SAME 256 frames and two different
    // 512-column passes.  CTA r of pair X and CTA r of pair Y need identical A tiles, so each computes
    // the FIR for every other K chunk and writes it into both CTAs' rings (remote st.shared::cluster):
    // the subfilter stage is then recomputed n_passes / 2 times per frame instead of n_passes times.
    const uint32_t crank = CG == 2 ? cluster_ctarank() : 0;     // rank in the cluster
    const uint32_t pr = SHARE ? (crank >> 1) : 0;                // pair index within the cluster
    const uint32_t rank = crank & 1u;                            // rank within the pair
    const uint32_t leader = pr * 2;                              // cluster rank of this pair's leader
    const uint32_t sib = crank ^ 2u;                             // (SHARE) the CTA with the same frames in the other pair
    const uint16_t pair_mask = (uint16_t)(3u << (2 * pr));
    constexpr int CL = SHARE ? 4 : CG;                           // CTAs per cluster
    const int cl = blockIdx.x / CL, n_cl = gridDim.x / CL;       // cluster id / number of clusters
    const int npg = SHARE ? prm.n_passes / 2 : prm.n_passes;     // column passes per work item group
#define TINA_PASS(w) (SHARE ? 2 * ((w) % npg) + (int)pr : (w) % npg)
    constexpr uint32_t B_ENTRY = B_ENTRY_BYTES / CG;             // bytes per B ring entry in this CTA
    const uint32_t N_B = (uint32_t)prm.b_ring_bytes / B_ENTRY;    // ring entries (<= 8)
    const uint32_t b_box_bytes = (uint32_t)(N < NSUB ? N : NSUB) / CG * KC * 2;   // bytes one TMA box delivers

    if (warp == TMA_WARP && lane == 0) {
        prefetch_tmap(&tmap_b);
        if (prm.out_tma) { prefetch_tmap(&tmap_out); if (REAL) prefetch_tmap(&tmap_out2); }
        // a_full: this CTA's 8 producer warps (+ in the leader one forwarded arrival from the peer's warp 1)
        for (int i = 0; i < 8; ++i) { mbar_init(smem_u32(&ctl->a_full[i]), N_PROD_WARPS + (rank == 0 ? CG - 1 : 0)); mbar_init(smem_u32(&ctl->a_empty[i]), SHARE ? 4 : 2); }
        for (int i = 0; i < (int)N_B; ++i) { mbar_init(smem_u32(&ctl->b_full[i]), 1); mbar_init(smem_u32(&ctl->b_empty[i]), 1); }
        for (int i = 0; i < 2; ++i) { mbar_init(smem_u32(&ctl->t_full[i]), 1); mbar_init(smem_u32(&ctl->t_empty[i]), 4 * CG); }
        fence_mbar_init();
    }
    if (warp == ALLOC_WARP) {
        tmem_alloc<CG>(smem_u32(&ctl->tmem_base), 512);
        tmem_relinquish<CG>();
    }
    tc_fence_before();
    if (CG == 2) cluster_sync(); else __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = ctl->tmem_base;

    if (warp == TMA_WARP) {
        // ============================ TMA producer: twiddle tiles ============================
        if (lane == 0) {
            RingPos b;
            for (int w = cl; w < prm.total_work; w += n_cl) {
                const int n0 = TINA_PASS(w) * NTP;
                const int nt = min(NTP, N - n0);
                const int n_sub = (nt + NSUB - 1) / NSUB;
                for (int kc = 0; kc < n_kc; ++kc)
                    for (int nh = 0; nh < n_sub; ++nh) {
                        const int nw = min(NSUB, nt - nh * NSUB);
                        for (int part = 0; part < parts; ++part) {
                            mbar_wait<64>(smem_u32(&ctl->b_empty[b.idx]), b.phase ^ 1);
                            const uint32_t bar = smem_u32(&ctl->b_full[b.idx]);
                            const uint32_t dst = smem_u32(b_ring + b.idx * B_ENTRY);
                            const int row = part * N + n0 + nh * NSUB + (int)rank * (nw / CG);
                            if (TINA_DBG(8)) { if (rank == 0) mbar_arrive(bar); }
                            else if (CG == 1) {
                                mbar_expect_tx(bar, b_box_bytes);
                                tma_load_2d(dst, &tmap_b, bar, kc * KC, row);
                            } else {
                                if (rank == 0) mbar_expect_tx(bar, 2 * b_box_bytes);
                                tma_load_2d_cg2(dst, &tmap_b, mapa_u32(bar, leader), kc * KC, row);
                            }
                            b.advance(N_B);
                        }
                    }
            }
        }
    } else if (warp == MMA_WARP || warp == MMA_WARP2) {
        // ============================ MMA issuers ===========================================
        // Two issuing warps, one per 256-column half of the accumulator tile (warp MMA_WARP: columns
        // 0-255, MMA_WARP2: 256-511).  tcgen05.mma issue blocks on a short queue and every barrier
        // wait / commit costs the issuing thread ~70-100 cycles in which it queues nothing; with two
        // threads the tensor pipe always has the other half's MMAs to run.  Both wait on the same A
        // slot, each consumes its own twiddle entries, and a_empty / t_full take one commit from each.
        // (cta_group::2: only the leader CTA issues; the peer's MMA_WARP forwards "my A tile is ready"
        //  to the leader's barrier, one remote arrive per chunk instead of one per producer warp.)
        const int h = warp == MMA_WARP ? 0 : 1;
        if (CG == 2 && rank != 0 && h == 0) {
            RingPos a;
            for (int w = cl; w < prm.total_work; w += n_cl)
                for (int kc = 0; kc < n_kc; ++kc) {
                    mbar_wait(smem_u32(&ctl->a_full[a.idx]), a.phase);
                    if (lane == 0) mbar_arrive_cluster(smem_u32(&ctl->a_full[a.idx]), leader);
                    __syncwarp();
                    a.advance(n_a);
                }
        }
        if (CG == 1 || rank == 0) {
        RingPos a, t;
        uint32_t g = 0;                                        // twiddle entries produced before this chunk
        long long pf_a = 0, pf_b = 0, pf_t = 0, pf_tot = PF_NOW(), pf_c;
#define PF_BEGIN() (pf_c = PF_NOW())
#define PF_END(acc) (acc += PF_NOW() - pf_c)
        uint32_t te_bits = 0;                                  // phase bit per 256-column TMEM block
        for (int w = cl; w < prm.total_work; w += n_cl) {
            const int n0 = TINA_PASS(w) * NTP;
            const int nt = min(NTP, N - n0);
            const int n_sub = (nt + NSUB - 1) / NSUB;
            const bool active = h < n_sub;                     // this warp's column half exists in this pass
            const int nw = active ? min(NSUB, nt - h * NSUB) : 0;
            const uint32_t idesc = idesc_bf16(BM * CG, nw, prm.fp16 != 0);
            for (int ks = 0; ks < prm.k_splits; ++ks) {
            const uint32_t blk = (n_acc == 2 ? t.idx : 0) + h;   // this warp's 256-column TMEM block
            const uint32_t d = tmem_base + blk * 256;
            const int kc_begin = ks * prm.kc_per_split, kc_end = min(n_kc, kc_begin + prm.kc_per_split);
            for (int kc = kc_begin; kc < kc_end; ++kc) {
                PF_BEGIN(); mbar_wait(smem_u32(&ctl->a_full[a.idx]), a.phase); PF_END(pf_a);
                tc_fence_after();
                const uint32_t a_hi = smem_u32(a_ring + a.idx * a_slot_bytes);
                const uint32_t a_lo = a_hi + A_PART_BYTES;
                if (active) {
                    if (kc == kc_begin) {
                        // first write into this TMEM block: wait until the epilogue has drained it
                        PF_BEGIN(); mbar_wait(smem_u32(&ctl->t_empty[blk]), ((te_bits >> blk) & 1u) ^ 1u); PF_END(pf_t);
                        te_bits ^= 1u << blk;
                        tc_fence_after();
                    }
                    // ---- B_hi: (A_lo x B_hi) then (A_hi x B_hi)
                    uint32_t e = g + (uint32_t)h * (uint32_t)parts;
                    uint32_t bi = e % N_B, bp = (e / N_B) & 1u;
                    PF_BEGIN(); mbar_wait(smem_u32(&ctl->b_full[bi]), bp); PF_END(pf_b);
                    tc_fence_after();
                    if (elect_one()) {
                        const uint64_t bd = smem_desc_sw128(smem_u32(b_ring + bi * B_ENTRY));
                        uint32_t acc = kc > kc_begin;
                        if (TINA_DBG(4)) { } else
                        if (parts > 1) {
                            const uint64_t ad = smem_desc_sw128(a_lo);
#pragma unroll
                            for (int k = 0; k < KC / 16; ++k) { umma_bf16<CG>(d, ad + 2 * k, bd + 2 * k, idesc, acc); acc = 1; }
                        }
                        const uint64_t ad = smem_desc_sw128(a_hi);
                        if (!TINA_DBG(4))
#pragma unroll
                        for (int k = 0; k < KC / 16; ++k) { umma_bf16<CG>(d, ad + 2 * k, bd + 2 * k, idesc, acc); acc = 1; }
                        commit_cg<CG>(smem_u32(&ctl->b_empty[bi]), pair_mask);
                    }
                    __syncwarp();
                    // ---- B_lo: (A_hi x B_lo)
                    if (parts > 1) {
                        ++e; bi = e % N_B; bp = (e / N_B) & 1u;
                        PF_BEGIN(); mbar_wait(smem_u32(&ctl->b_full[bi]), bp); PF_END(pf_b);
                        tc_fence_after();
                        if (elect_one()) {
                            const uint64_t bd = smem_desc_sw128(smem_u32(b_ring + bi * B_ENTRY));
                            const uint64_t ad = smem_desc_sw128(a_hi);
                            if (!TINA_DBG(4))
#pragma unroll
                            for (int k = 0; k < KC / 16; ++k) umma_bf16<CG>(d, ad + 2 * k, bd + 2 * k, idesc, 1);
                            commit_cg<CG>(smem_u32(&ctl->b_empty[bi]), pair_mask);
                        }
                        __syncwarp();
                    }
                }
                g += (uint32_t)(n_sub * parts);
                if (elect_one()) {
                    commit_cg<CG>(smem_u32(&ctl->a_empty[a.idx]), SHARE ? (uint16_t)0xF : pair_mask);
                    // one "accumulator ready" barrier per 256-column TMEM block: the two halves finish (and are
                    // drained) independently, so one half's drain overlaps the other half's MMAs
                    if (kc == kc_end - 1 && active) commit_cg<CG>(smem_u32(&ctl->t_full[blk]), pair_mask);
                }
                __syncwarp();
                a.advance(n_a);
            }
            t.advance(n_acc);
            }
        }
        if (PF_ON() && lane == 0 && h == 0) {
            unsigned long long* pp = prm.prof + blockIdx.x * 16;
            pp[0] = PF_NOW() - pf_tot; pp[1] = pf_a; pp[2] = pf_b; pp[3] = pf_t;
        }
        }
    } else if (warp >= EPI_WARP0 && warp < EPI_WARP0 + 4) {
        // ============================ epilogue: TMEM -> smem transpose -> global =============
        // tcgen05.ld hands each lane one accumulator ROW; a row-per-lane global store touches 32
        // cache lines per instruction.  Each warp therefore bounces its 32x32 block through a
        // padded shared-memory tile and stores it with 128-byte-contiguous row segments
        // (4 rows x 128 B per float4 instruction; 2 rows x 128 B per float2 for the real kind,
        // whose rows are only 8-byte aligned).  Later accumulation chains add into the output.
        const int q = warp - EPI_WARP0;
        float* stg = reinterpret_cast<float*>(stage + q * prm.stage_bytes);   // register / shared-memory store path
        const uint32_t sbuf = smem_u32(stage) + q * 4096u;                    // TMA path: 1024-byte aligned swizzled tile
        RingPos t;
        long long pe_w = 0, pe_tot = PF_NOW(), pe_x, pe_ld = 0, pe_sts = 0, pe_st = 0, pe_fo = 0, pe_sy = 0;
        uint32_t tf_bits = 0;                                  // phase bit per TMEM block's t_full barrier
        for (int w = cl; w < prm.total_work; w += n_cl) {
            const int tile = w / npg;
            const int n0 = TINA_PASS(w) * NTP;
            const int nt = min(NTP, N - n0);
            const int s = tile / prm.tiles_per_stream;
            const long long row0 = (long long)(tile % prm.tiles_per_stream) * (BM * CG) + rank * BM + q * 32;
            float* obase = prm.out + (long long)s * prm.out_stream_stride + row0 * prm.out_row + n0;
            const int rows_valid = TINA_DBG(2) ? 0 : (int)min(32LL, prm.F - row0);   // <= 0: nothing to store
            for (int ks = 0; ks < prm.k_splits; ++ks) {
                const uint32_t blk0 = n_acc == 2 ? t.idx : 0;
                // wait for the 256-column TMEM block that column cb starts (called before its first tcgen05.ld)
                auto wait_block = [&](int cb) {
                    const uint32_t bk = blk0 + ((uint32_t)cb >> 8);
                    pe_x = PF_NOW(); mbar_wait<256>(smem_u32(&ctl->t_full[bk]), (tf_bits >> bk) & 1u); pe_w += PF_NOW() - pe_x;
                    tf_bits ^= 1u << bk;
                    tc_fence_after();
                };
                const uint32_t taddr = tmem_base + blk0 * 256 + ((uint32_t)(q * 32) << 16);
                if (prm.out_tma) {
                    // The tile leaves through the TMA engine.  Each 32x32 block is written (bank-conflict
                    // free, 128-byte swizzle) into one of two 4 KB staging tiles and stored -- or, for later
                    // accumulation chains, add-reduced in fp32 at L2 -- by bulk tensor instructions; rows
                    // >= F are clipped by the tensor map.  Complex kind: one 32-row box.  Real kind: rows
                    // are only 8-byte aligned, but PAIRS of rows have a 16-byte-multiple pitch, so even
                    // and odd rows go out as two 16-row boxes through two maps over row pairs.
                    if (ks > 0 && lane == 0) bulk_wait<0>();     // the previous chain's stores to this tile are complete
                    uint32_t r[32];
                    wait_block(0);
                    tmem_ld32(taddr, r);
                    const uint32_t rr = REAL ? ((uint32_t)lane >> 1) : (uint32_t)lane;       // row within the staged box
                    const bool odd = REAL && (lane & 1);
                    float* const orow = obase + (long long)lane * prm.out_row;               // this lane's output row
                    for (int cb = 0; cb < nt; cb += 32) {
                        tmem_ld_wait();
                        if (REAL && lane < rows_valid && !TINA_DBG(2)) {
                            if (n0 + cb == 0) {
                                // columns 0 / 1 carry Re X[0] and Re X[P/2]; Im X[0] = Im X[P/2] = 0
                                float2* ny = reinterpret_cast<float2*>(orow + prm.P);
                                const float nyq = __uint_as_float(r[1]);
                                if (ks > 0) atomicAdd(&ny->x, nyq);           // fire-and-forget fp32 add at L2
                                else *ny = make_float2(nyq, 0.f);
                                r[1] = 0u;
                            }
                            if (odd) {
                                // odd rows start 8 bytes off a 16-byte boundary: their TMA box covers columns
                                // cb+2 .. cb+29; the two edge pairs are stored from registers
                                float2* e0 = reinterpret_cast<float2*>(orow + cb);           // (obase already points at column n0)
                                float2* e1 = reinterpret_cast<float2*>(orow + cb + 30);
                                float2 a = make_float2(__uint_as_float(r[0]), __uint_as_float(r[1]));
                                float2 b = make_float2(__uint_as_float(r[30]), __uint_as_float(r[31]));
                                if (ks > 0) { atomicAdd(e0, a); atomicAdd(e1, b); }   // red.global.add.v2.f32, no round trip
                                else { *e0 = a; *e1 = b; }
                            }
                        } else if (REAL && n0 + cb == 0) {
                            r[1] = 0u;
                        }
                        if (lane == 0) bulk_wait_read<0>();      // the previous block's tile has been read by the TMA engine
                        __syncwarp();
                        const uint32_t tile_s = sbuf;
                        if (!odd) {
                            const uint32_t dst = tile_s + rr * 128u;
#pragma unroll
                            for (int j = 0; j < 8; ++j)
                                sts128(dst + (((uint32_t)j ^ (rr & 7u)) << 4), r[4 * j], r[4 * j + 1], r[4 * j + 2], r[4 * j + 3]);
                        } else {
                            const uint32_t dst = tile_s + 2048u + rr * 112u;                 // dense 16 x 28 floats
#pragma unroll
                            for (int j = 0; j < 7; ++j)
                                sts128(dst + 16u * j, r[4 * j + 2], r[4 * j + 3], r[4 * j + 4], r[4 * j + 5]);
                        }
                        const bool last_of_block = (cb & 255) == 224;            // next 32 columns start another TMEM block
                        if (cb + 32 < nt && !last_of_block) tmem_ld32(taddr + cb + 32, r);
                        fence_proxy_async();
                        __syncwarp();
                        if (lane == 0 && !TINA_DBG(2)) {
                            if (!REAL) {
                                if (ks == 0) tma_store_3d(&tmap_out, tile_s, n0 + cb, (int)row0, s);
                                else         tma_reduce_add_3d(&tmap_out, tile_s, n0 + cb, (int)row0, s);
                            } else {
                                const int pr = (int)(row0 >> 1), c_odd = prm.P + 2 + n0 + cb + 2;
                                if (ks == 0) { tma_store_3d(&tmap_out, tile_s, n0 + cb, pr, s); tma_store_3d(&tmap_out2, tile_s + 2048u, c_odd, pr, s); }
                                else { tma_reduce_add_3d(&tmap_out, tile_s, n0 + cb, pr, s); tma_reduce_add_3d(&tmap_out2, tile_s + 2048u, c_odd, pr, s); }
                            }
                            bulk_commit();
                        }
                        if (last_of_block || cb + 32 >= nt) {
                            // this TMEM block has been read out completely: hand it back, then (if there is
                            // another block) wait for it and start reading it
                            tc_fence_before();
                            __syncwarp();
                            if (lane == 0) arrive_leader<CG>(smem_u32(&ctl->t_empty[blk0 + (cb >> 8)]), rank, leader);
                            if (cb + 32 < nt) { wait_block(cb + 32); tmem_ld32(taddr + cb + 32, r); }
                        }
                    }
                    t.advance(n_acc);
                    continue;
                }
                if (prm.out_scalar) {
                    // Toeplitz FIR: the warp's 32 rows x N columns are ONE contiguous run of 32 N floats of a
                    // [C][L-M+1] array that is only 4-byte aligned.  Misaligned 128-byte row segments leave
                    // partially written sectors behind (measured 4.5x slower), so the whole sub-tile is staged
                    // (row pitch FIR_PITCH), TMEM is handed back at once, and the run is written as 16-byte
                    // aligned float4 with scalar head / tail.
                    uint32_t r[32];
                    wait_block(0);
                    tmem_ld32(taddr, r);
                    for (int cb = 0; cb < nt; cb += 32) {
                        tmem_ld_wait();
#pragma unroll
                        for (int j = 0; j < 8; ++j)
                            *reinterpret_cast<float4*>(stg + lane * FIR_PITCH + cb + 4 * j) =
                                make_float4(__uint_as_float(r[4 * j]), __uint_as_float(r[4 * j + 1]),
                                            __uint_as_float(r[4 * j + 2]), __uint_as_float(r[4 * j + 3]));
                        if (cb + 32 < nt) { if (((cb + 32) & 255) == 0) wait_block(cb + 32); tmem_ld32(taddr + cb + 32, r); }
                    }
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) arrive_leader<CG>(smem_u32(&ctl->t_empty[blk0]), rank, leader);
                    // linear element l of the run <-> staged [l / nt][l % nt]; stream index e0 + l
                    const long long e0 = row0 * prm.out_row + n0;
                    long long n_run = prm.out_len - e0;                        // valid elements of the run
                    if (n_run > 32LL * 128) n_run = 32LL * 128;
                    if (n_run > 0 && !TINA_DBG(2)) {
                        float* g = obase;                                        // address of l = 0
                        const int run = (int)n_run;
                        const int head = min(run, (int)(((16u - ((uint32_t)(uintptr_t)g & 15u)) & 15u) >> 2));
                        const int nv4 = (run - head) >> 2;                       // aligned float4 stores
                        auto at = [&](int l) { return stg[(l >> 7) * FIR_PITCH + (l & 127)]; };   // nt == 128 in this mode
                        if (lane < head) g[lane] = at(lane);
                        for (int v = lane; v < nv4; v += 32) {
                            const int l = head + 4 * v;
                            *reinterpret_cast<float4*>(g + l) = make_float4(at(l), at(l + 1), at(l + 2), at(l + 3));
                        }
                        const int tail0 = head + 4 * nv4;
                        if (tail0 + lane < run) g[tail0 + lane] = at(tail0 + lane);
                    }
                    __syncwarp();
                    t.advance(n_acc);
                    continue;
                }
                // lane -> (row, column) of the transposed (coalesced) global access pattern
                constexpr int NV = REAL ? 16 : 8;                     // accesses per lane per 32-column block
                constexpr int RSTEP = REAL ? 2 : 4;
                const int c = REAL ? 2 * (lane & 15) : 4 * (lane & 7);
                const int rbase = REAL ? (lane >> 4) : (lane >> 3);
                float* const gp0 = obase + (long long)rbase * prm.out_row + c;
                const long long gstep = (long long)RSTEP * prm.out_row;
                float4 o4[REAL ? 1 : 8];
                float2 o2[REAL ? 16 : 1];
                float nyq_old[REAL ? 16 : 1];
                // later chains: the running sums of a block are fetched one block ahead
                auto fetch_old = [&](int cb) {
                    const bool special = REAL && (n0 + cb == 0) && c == 0;
#pragma unroll
                    for (int i = 0; i < NV; ++i) {
                        if (rbase + RSTEP * i < rows_valid) {
                            const float* g = gp0 + cb + i * gstep;
                            if (REAL) {
                                o2[i] = *reinterpret_cast<const float2*>(g);
                                if (special) nyq_old[i] = *(g + prm.P);
                            } else {
                                o4[i] = *reinterpret_cast<const float4*>(g);
                            }
                        }
                    }
                };
                uint32_t r[32];
                if (ks > 0) fetch_old(0);
                wait_block(0);
                tmem_ld32(taddr, r);
                for (int cb = 0; cb < nt; cb += 32) {
                    const bool special = REAL && (n0 + cb == 0) && c == 0;   // columns 0 / 1 = Re X[0], Re X[P/2]
                    pe_x = PF_NOW(); tmem_ld_wait(); pe_ld += PF_NOW() - pe_x; pe_x = PF_NOW();
#pragma unroll
                    for (int j = 0; j < 8; ++j)
                        *reinterpret_cast<float4*>(stg + lane * EPI_LD + 4 * j) =
                            make_float4(__uint_as_float(r[4 * j]), __uint_as_float(r[4 * j + 1]),
                                        __uint_as_float(r[4 * j + 2]), __uint_as_float(r[4 * j + 3]));
                    // the next block's TMEM read overlaps this block's transpose and stores
                    const bool last_of_block = (cb & 255) == 224;
                    if (cb + 32 < nt && !last_of_block) tmem_ld32(taddr + cb + 32, r);
                    __syncwarp();
                    pe_sts += PF_NOW() - pe_x; pe_x = PF_NOW();
#pragma unroll
                    for (int i = 0; i < NV; ++i) {
                        const int rr = rbase + RSTEP * i;
                        if (rr < rows_valid) {
                            float* g = gp0 + cb + i * gstep;
                            if (REAL) {
                                float2 v = *reinterpret_cast<const float2*>(stg + rr * EPI_LD + c);
                                if (special) {
                                    if (ks > 0) { v.x += o2[i].x; v.y += nyq_old[i]; }
                                    *reinterpret_cast<float2*>(g + prm.P) = make_float2(v.y, 0.f);   // out[P], out[P+1]
                                    v.y = 0.f;
                                } else if (ks > 0) {
                                    v.x += o2[i].x; v.y += o2[i].y;
                                }
                                *reinterpret_cast<float2*>(g) = v;
                            } else {
                                float4 v = *reinterpret_cast<const float4*>(stg + rr * EPI_LD + c);
                                if (ks > 0) { v.x += o4[i].x; v.y += o4[i].y; v.z += o4[i].z; v.w += o4[i].w; }
                                *reinterpret_cast<float4*>(g) = v;
                            }
                        }
                    }
                    pe_st += PF_NOW() - pe_x; pe_x = PF_NOW();
                    if (ks > 0 && cb + 32 < nt) fetch_old(cb + 32);
                    pe_fo += PF_NOW() - pe_x; pe_x = PF_NOW();
                    __syncwarp();
                    pe_sy += PF_NOW() - pe_x;
                    if (last_of_block || cb + 32 >= nt) {
                        // a 256-column TMEM block has been read out: hand it back to the MMA warp, then wait
                        // for the next block (if any) and start reading it
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) arrive_leader<CG>(smem_u32(&ctl->t_empty[blk0 + (cb >> 8)]), rank, leader);
                        if (cb + 32 < nt) { wait_block(cb + 32); tmem_ld32(taddr + cb + 32, r); }
                    }
                }
                t.advance(n_acc);
            }
        }
        if (prm.out_tma && lane == 0) bulk_wait<0>();            // staging tiles must outlive their TMA reads
        if (PF_ON() && q == 0 && lane == 0) {
            unsigned long long* pp = prm.prof + blockIdx.x * 16;
            pp[8] = PF_NOW() - pe_tot; pp[9] = pe_w; pp[10] = pe_ld; pp[11] = pe_sts; pp[12] = pe_st; pp[13] = pe_fo; pp[14] = pe_sy;
        }
    } else if (warp >= PROD_WARP0 && warp < PROD_WARP0 + N_PROD_WARPS) {
        // ============================ FIR producers =========================================
        // Software pipeline over the flattened (work item, K chunk) sequence: the loads of chunk
        // c+1 are issued right after the arithmetic of chunk c and before its fence / arrive, so
        // their latency (and the fence's) overlaps the hand-off and the wait for the next slot.
        const int pw = warp - PROD_WARP0;
        const uint32_t a_ring_s = smem_u32(a_ring);
        // byte offset of this lane's 4-byte cell in row 0 of an A tile, for each swizzle phase (row & 7):
        // row r, 16-byte chunk (lane >> 2) is stored at chunk position (lane >> 2) ^ (r & 7)
        uint32_t swz[8];
#pragma unroll
        for (int j = 0; j < 8; ++j)
            swz[j] = (uint32_t)(pw * FPW) * 128u + ((((uint32_t)lane >> 2) ^ (uint32_t)j) << 4) + ((uint32_t)lane & 3u) * 4u;
        constexpr int WA = MT > 0 ? MT : 1;
        const float* const window = prm.window;
        const int P = prm.P, M = prm.M;
        const long long K = prm.x_row_stride, nblk = prm.NBLK, x_len = prm.x_len;
        const bool split = parts > 1;
        FirRegs<MT> rg;
        const uint32_t r_ring_s = SHARE ? mapa_u32(a_ring_s, sib) : 0;   // the sibling's A ring (cluster address)
        int w = cl, kc = 0;
        uint32_t n = 0;                                      // chunk counter over the cluster's whole sequence
        const float* xs = nullptr;
        long long f0 = 0;
        bool interior = false;
        auto set_tile = [&](int ww) {
            const int tile = ww / npg;
            const int s = tile / prm.tiles_per_stream;
            f0 = (long long)(tile % prm.tiles_per_stream) * (BM * CG) + rank * BM + pw * FPW;
            xs = prm.x + (long long)s * prm.stream_stride + 2 * lane;
            // rows f0 + M - WA .. f0 + FPW + M - 2 are touched; interior tiles need no bounds checks
            interior = (f0 + M - WA >= 0) && (f0 + FPW + M - 1 <= nblk) &&
                       (x_len == 0 || (f0 + FPW + M - 2) * K + prm.K <= x_len);
        };
        auto load = [&](int kk) {
            if (TINA_DBG(1)) return;
            if (interior) fir_load<MT, REAL, false>(rg, window, P, M, K, nblk, xs + kk * KC, kk * KC + 2 * lane, f0);
            else          fir_load<MT, REAL, true>(rg, window, P, M, K, nblk, xs + kk * KC, kk * KC + 2 * lane, f0, x_len);
        };
        // next chunk of the sequence that this CTA produces (SHARE: chunks alternate between the siblings)
        auto advance = [&](int& ww, int& kk, uint32_t& nn) {
            do {
                ++nn;
                if (++kk == n_kc) { kk = 0; ww += n_cl; }
            } while (SHARE && ww < prm.total_work && (nn & 1u) != pr);
        };
        long long pq_w = 0, pq_c = 0, pq_f = 0, pq_tot = PF_NOW(), pq_x;
        if (SHARE && pr != 0) advance(w, kc, n);             // pair 1 starts with chunk 1
        bool have = w < prm.total_work;
        if (have) { set_tile(w); load(kc); }
        while (have) {
            int w2 = w, kc2 = kc;
            uint32_t n2 = n;
            advance(w2, kc2, n2);
            const bool have2 = w2 < prm.total_work;
            const uint32_t slot_i = n % n_a, slot_ph = (n / n_a) & 1u;
            pq_x = PF_NOW(); mbar_wait(smem_u32(&ctl->a_empty[slot_i]), slot_ph ^ 1); pq_w += PF_NOW() - pq_x;
            pq_x = PF_NOW();
            if (!TINA_DBG(1))
                fir_compute_store<MT>(rg, a_ring_s + slot_i * a_slot_bytes, swz, split, 0, prm.fp16 != 0);
            if (have2) {
                if (w2 != w) set_tile(w2);
                load(kc2);
            }
            pq_c += PF_NOW() - pq_x; pq_x = PF_NOW();
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) {
                const uint32_t bar = smem_u32(&ctl->a_full[slot_i]);
                mbar_arrive(bar);
                if (SHARE) {
                    // publish this warp's 16-row slab of the tile (2 KB per part, contiguous) to the same slot
                    // of the sibling CTA: async bulk copy, one arrival + the bytes on the sibling's barrier
                    const uint32_t slab = slot_i * a_slot_bytes + (uint32_t)(pw * FPW) * 128u;
                    const uint32_t rbar = mapa_u32(bar, sib);
                    mbar_expect_tx_cluster(bar, sib, (uint32_t)parts * (FPW * 128u));
                    for (int part = 0; part < parts; ++part)
                        bulk_copy_to_cluster(r_ring_s + slab + part * A_PART_BYTES, a_ring_s + slab + part * A_PART_BYTES,
                                             FPW * 128u, rbar);
                }
            }
            pq_f += PF_NOW() - pq_x;
            w = w2; kc = kc2; n = n2; have = have2;
        }
        if (PF_ON() && pw == 0 && lane == 0) {
            unsigned long long* pp = prm.prof + blockIdx.x * 16;
            pp[4] = PF_NOW() - pq_tot; pp[5] = pq_w; pp[6] = pq_c; pp[7] = pq_f;
        }
    }

    tc_fence_before();
    if (CG == 2) cluster_sync(); else __syncthreads();   // the peer's smem / barriers stay live until both are done
    if (warp == ALLOC_WARP) tmem_dealloc<CG>(tmem_base, 512);
}

// =====================================================================================
// Host side
// =====================================================================================
bool umma_supported(int P, bool real)
{
    if (P < 32 || P > kMaxP) return false;
    return real ? (P % 64 == 0) : (P % 32 == 0);
}

template <int MT, bool REAL, bool SHARE>
static tina_status launch_umma(DevCtx* ctx, const CUtensorMap& tmap, const CUtensorMap& tmap_out, const CUtensorMap& tmap_out2,
                               const UmmaParams& prm, int grid, cudaStream_t st)
{
    auto kern = pfb_umma_kernel<MT, REAL, UMMA_CG, SHARE>;
    tina_status as = ensure_smem(ctx, reinterpret_cast<const void*>(kern), (int)UMMA_SMEM_BYTES, "cudaFuncSetAttribute(pfb_umma_kernel)");
    if (as != TINA_OK) return as;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(UMMA_THREADS);
    cfg.dynamicSmemBytes = UMMA_SMEM_BYTES;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = SHARE ? 4 : UMMA_CG;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    UmmaParams prm2 = prm;
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
        for (int b = 0; b < grid; b += UMMA_CG) for (int i = 0; i < 16; ++i) acc[i] += (double)h[(size_t)b * 16 + i] / (grid / UMMA_CG);   // leaders: even ranks
        fprintf(stderr, "[tina prof] leader CTA mean cycles: mma tot %.0f a_full %.0f b_full %.0f t_empty %.0f | prod tot %.0f a_empty %.0f work %.0f fence %.0f | epi tot %.0f t_full %.0f ldwait %.0f sts %.0f lds+stg %.0f fetch %.0f sync %.0f\n",
                acc[0], acc[1], acc[2], acc[3], acc[4], acc[5], acc[6], acc[7], acc[8], acc[9], acc[10], acc[11], acc[12], acc[13], acc[14]);
    }
#endif
    count_launch();
    g_last_path = kPathUmma; note_kernel("pfb_umma_kernel");
    if (e != cudaSuccess) return check_cuda(e, "pfb_umma_kernel launch");
    return check_cuda(cudaGetLastError(), "pfb_umma_kernel launch");
}

tina_status umma_pfb(const void* x, int S, long long n_samples, int P, int M, const float* window,
                     bool real, bool inverse, tina_precision prec, void* out, cudaStream_t st)
{
    const int K = real ? P : 2 * P;
    const long long NBLK = n_samples / P;
    const long long F = NBLK - M + 1;
    const int parts = prec == TINA_PREC_FP32 ? 2 : 1;
    const bool fp16 = prec == TINA_PREC_FP16;

    // the column-paired, TMA-staged kernel takes every M <= 64 fused (taps in groups of 16)
    const bool symt_ok = !options().no_sym && !options().sym_v1 && (real ? (window && sym_real_supported(P)) : sym_supported(P));
    if (window && M > 16 && !symt_ok) {
        // Rare shape (P not a multiple of 64, or the round-1 kernels selected): more taps than the register window is
        // unrolled for.  Run the subfilter stage on its own into a stream-ordered temporary, then the contraction as a DFT batch.
        float* y = nullptr;
        const size_t bytes = (size_t)S * F * K * sizeof(float);
        cudaError_t e = cudaMallocAsync(reinterpret_cast<void**>(&y), bytes, st);
        if (e != cudaSuccess) return check_cuda(e, "cudaMallocAsync(subfiltered)");
        tina_status s1 = simt_pfb_fir(x, S, n_samples, P, M, window, real, y, st);
        if (s1 == TINA_OK) s1 = umma_pfb(y, 1, (long long)S * F * P, P, 1, nullptr, real, inverse, prec, out, st);
        cudaFreeAsync(y, st);
        return s1;
    }

    // complex kind: the column-paired contraction (half the tensor work) wherever its tiling applies
    if (!options().no_sym && (real ? (window && sym_real_supported(P)) : sym_supported(P)))
        return sym_pfb(x, S, n_samples, P, M, window, real, inverse, prec, out, st);

    const Plan* plan = nullptr;
    tina_status ps = get_plan(P, real, inverse, parts, fp16, st, &plan);
    if (ps != TINA_OK) return ps;
    DevCtx* ctx = nullptr;
    if ((ps = dev_ctx(&ctx)) != TINA_OK) return ps;
    const Options& opt = options();
    const int n_sm = ctx->n_sm;

    UmmaParams prm;
    prm.x = static_cast<const float*>(x);
    prm.window = window;
    prm.out = static_cast<float*>(out);
    prm.stream_stride = real ? n_samples : 2 * n_samples;
    prm.F = F;
    prm.NBLK = NBLK;
    prm.out_row = real ? P + 2 : 2 * P;
    prm.out_stream_stride = F * prm.out_row;
    prm.K = K;
    prm.N = K;
    prm.x_row_stride = K;
    prm.x_len = 0;
    prm.out_len = 0;
    prm.out_scalar = 0;
    prm.a_ring_bytes = A_RING_BYTES; prm.b_ring_bytes = B_RING_BYTES; prm.stage_bytes = EPI_STAGE_BYTES;
#ifdef TINA_DEV
    {   // experiment knobs: ring depths (A slots of 32 KB, B half-tile entries of 16 KB)
        if (opt.a_slots) prm.a_ring_bytes = opt.a_slots * 2 * A_PART_BYTES;
        if (opt.b_entries) prm.b_ring_bytes = opt.b_entries * (B_ENTRY_BYTES / UMMA_CG);
        if ((size_t)prm.a_ring_bytes + prm.b_ring_bytes + 4 * prm.stage_bytes + sizeof(SmemCtl) > UMMA_SMEM_BYTES)
            return fail(TINA_ERR_UNSUPPORTED, "ring sizes exceed shared memory");
    }
#endif
    prm.P = P;
    prm.M = M;
    prm.tiles_per_stream = (int)((F + BM * UMMA_CG - 1) / (BM * UMMA_CG));
    // Column pass width: all 512 TMEM columns (one accumulator stage, both MMA-issuing warps busy).  256-column
    // passes (two TMEM stages, epilogue overlapped) measured slower at config 2 because only one warp issues.
    prm.nt_pass = opt.nt256 ? 256 : NT_MAX;
    prm.n_passes = (K + prm.nt_pass - 1) / prm.nt_pass;
    // SHARE (clusters of four, FIR computed once per two column passes) needs an even number of passes
    // Measured on B200 (c4 / c5): equal or slightly slower than independent pairs (only 33 clusters of four are
    // co-resident on 148 SMs and the twiddle ring becomes the limiter), so it is opt-in: TINA_SHARE=1.
    const bool share = prm.n_passes % 2 == 0 && n_sm >= 4 && opt.share;
    const long long total = (long long)S * prm.tiles_per_stream * (share ? prm.n_passes / 2 : prm.n_passes);
    if (total > 0x7fffffffLL) return fail(TINA_ERR_UNSUPPORTED, "tina_pfb: too many tiles");
    prm.total_work = (int)total;
    prm.parts = parts;
    prm.fp16 = fp16 ? 1 : 0;
    prm.prof = nullptr;
    prm.debug = opt.debug_skip;                                   // 0 unless -DTINA_DEV
    { const int kmax = opt.ksplit > 0 ? opt.ksplit : KSPLIT_MAX; prm.k_splits = (K + kmax - 1) / kmax; }
    prm.kc_per_split = ((K / KC) + prm.k_splits - 1) / prm.k_splits;

    const int cl_size = share ? 4 : UMMA_CG;
    int n_cl = n_sm / cl_size;
    if (share) {
        // clusters of four do not tile every GPC (16 / 18 / 20 SMs): launch only as many as are co-resident
        const int max_cl4 = opt.cl4 > 0 ? opt.cl4 : 33;
        if (n_cl > max_cl4) n_cl = max_cl4;
    }
    const int grid = cl_size * (prm.total_work < n_cl ? prm.total_work : n_cl);

    // Output tensor maps for the TMA-store epilogue.  Complex kind: [S][F][2P] floats, 32x32 boxes.
    // Real kind: a row is P+2 floats (8-byte aligned only), so the maps run over row PAIRS, whose
    // pitch (2P+4 floats) is a multiple of 16 bytes: one map sees the even rows (extent P+2 in x,
    // ceil(F/2) pairs), the other the whole pair (extent 2P+4, floor(F/2) pairs) and is addressed at
    // x >= P+2 for the odd rows.  Needs a 16-byte-multiple stream pitch (S == 1 or F even) and F >= 2;
    // other real shapes use the register/shared-memory store path.
    CUtensorMap tmap_out, tmap_out2;
    memset(&tmap_out, 0, sizeof(tmap_out));
    memset(&tmap_out2, 0, sizeof(tmap_out2));
    prm.out_tma = real ? ((S == 1 || F % 2 == 0) && F >= 2) : 1;
    if (opt.no_out_tma && real) prm.out_tma = 0;
    if (prm.out_tma) {
        EncodeTiledFn enc = encode_fn();
        if (!enc) return fail(TINA_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found");
        const cuuint32_t estr[3] = {1, 1, 1};
        CUresult r;
        if (!real) {
            const cuuint64_t dims[3] = {(cuuint64_t)K, (cuuint64_t)F, (cuuint64_t)S};
            const cuuint64_t strides[2] = {(cuuint64_t)K * sizeof(float), (cuuint64_t)F * K * sizeof(float)};
            const cuuint32_t box[3] = {32, 32, 1};
            r = enc(&tmap_out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, out, dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                    CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        } else {
            const cuuint64_t row = (cuuint64_t)P + 2;
            const cuuint64_t pitch2 = 2 * row * sizeof(float);
            const cuuint64_t spitch = S > 1 ? (cuuint64_t)F * row * sizeof(float) : pitch2 * (cuuint64_t)((F + 1) / 2);
            const cuuint64_t strides[2] = {pitch2, spitch};
            const cuuint32_t box[3] = {32, 16, 1};
            const cuuint64_t dims_e[3] = {row, (cuuint64_t)((F + 1) / 2), (cuuint64_t)S};
            const cuuint64_t dims_o[3] = {2 * row, (cuuint64_t)(F / 2), (cuuint64_t)S};
            r = enc(&tmap_out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, out, dims_e, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                    CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            const cuuint32_t box_o[3] = {28, 16, 1};      // odd rows: columns +2 .. +29 of each block (16-byte aligned start)
            if (r == CUDA_SUCCESS)
                r = enc(&tmap_out2, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, out, dims_o, strides, box_o, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                        CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        }
        if (r != CUDA_SUCCESS) return fail(TINA_ERR_CUDA, "cuTensorMapEncodeTiled(out) failed (%d)", (int)r);
    }

#define TINA_LAUNCH(MT_)                                                                           \
    (real ? (share ? launch_umma<MT_, true, true>(ctx, plan->tmap, tmap_out, tmap_out2, prm, grid, st)                  \
                   : launch_umma<MT_, true, false>(ctx, plan->tmap, tmap_out, tmap_out2, prm, grid, st))                \
          : (share ? launch_umma<MT_, false, true>(ctx, plan->tmap, tmap_out, tmap_out2, prm, grid, st)                 \
                   : launch_umma<MT_, false, false>(ctx, plan->tmap, tmap_out, tmap_out2, prm, grid, st)))
    if (!window) return TINA_LAUNCH(0);
    if (M <= 4) return TINA_LAUNCH(4);
    if (M <= 8) return TINA_LAUNCH(8);
    return TINA_LAUNCH(16);
#undef TINA_LAUNCH
}

}  // namespace tina

// =====================================================================================
// Subfilter stage only (Eq. (20); Fig. 3 left column): the FIR producer's register
// sliding window with a direct global store.  One CTA = 128 frames x 64 scalar columns (8 warps x
// 16 frames); HBM-bound: every input sample is read once from HBM (the (M-1)-row halo between
// neighbouring warps / CTAs comes from L1 / L2), every output written once.
// =====================================================================================
namespace tina {

template <int MT, bool REAL>
__global__ void __launch_bounds__(256)
pfb_fir_win_kernel(const float* __restrict__ x, long long stream_stride, const float* __restrict__ window,
                   float* __restrict__ y, long long F, long long NBLK, int K, int P, int M, int tiles_per_stream)
{
    constexpr int WA = MT;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int kc = blockIdx.x;                                   // 64-column chunk
    const int tile = blockIdx.y;
    const int s = tile / tiles_per_stream;
    const long long f0 = (long long)(tile % tiles_per_stream) * BM + warp * FPW;
    if (f0 >= F) return;
    const int c0 = kc * KC + 2 * lane;
    const float* xs = x + (long long)s * stream_stride + c0;
    const bool interior = (f0 + M - WA >= 0) && (f0 + FPW + M - 1 <= NBLK);
    FirRegs<MT> rg;
    if (interior) fir_load<MT, REAL, false>(rg, window, P, M, K, NBLK, xs, c0, f0);
    else          fir_load<MT, REAL, true>(rg, window, P, M, K, NBLK, xs, c0, f0);
    float* yo = y + ((long long)s * F + f0) * K + c0;
#pragma unroll
    for (int i0 = 0; i0 < FPW; i0 += 8) {
        float2 acc[8];
#pragma unroll
        for (int g = 0; g < 8; ++g) acc[g] = fmul2(rg.tap[0], rg.row[i0 + g + WA - 1]);
#pragma unroll
        for (int m = 1; m < WA; ++m)
#pragma unroll
            for (int g = 0; g < 8; ++g) acc[g] = ffma2(rg.tap[m], rg.row[i0 + g + WA - 1 - m], acc[g]);
#pragma unroll
        for (int g = 0; g < 8; ++g)
            if (f0 + i0 + g < F) *reinterpret_cast<float2*>(yo + (long long)(i0 + g) * K) = acc[g];
    }
}

// true if the windowed-register kernel handled the call
bool umma_pfb_fir(const void* x, int S, long long n_samples, int P, int M, const float* window, bool real,
                  void* y, cudaStream_t st, tina_status* status)
{
    const int K = real ? P : 2 * P;
    if (K % KC != 0 || M > 16) return false;
    const long long NBLK = n_samples / P, F = NBLK - M + 1;
    const int tiles_per_stream = (int)((F + BM - 1) / BM);
    const long long tiles = (long long)S * tiles_per_stream;
    if (tiles > 65535) return false;
    const dim3 grid((unsigned)(K / KC), (unsigned)tiles);
    const long long stride = real ? n_samples : 2 * n_samples;
    const float* xf = static_cast<const float*>(x);
    float* yf = static_cast<float*>(y);
#define TINA_FIRWIN(MT_)                                                                                        \
    do {                                                                                                        \
        if (real) pfb_fir_win_kernel<MT_, true><<<grid, 256, 0, st>>>(xf, stride, window, yf, F, NBLK, K, P, M, tiles_per_stream); \
        else      pfb_fir_win_kernel<MT_, false><<<grid, 256, 0, st>>>(xf, stride, window, yf, F, NBLK, K, P, M, tiles_per_stream); \
    } while (0)
    if (M <= 4) TINA_FIRWIN(4);
    else if (M <= 8) TINA_FIRWIN(8);
    else TINA_FIRWIN(16);
#undef TINA_FIRWIN
    count_launch();
    g_last_path = kPathSimt; note_kernel("pfb_fir_win_kernel");
    *status = check_cuda(cudaGetLastError(), "pfb_fir_win_kernel launch");
    return true;
}

}  // namespace tina

// =====================================================================================
// Standalone FIR on the tensor cores (the paper's unfolding view, Eq. (17)-(19), PAPER.md:183-202:
// a FIR is a product of the unfolded signal with a banded Toeplitz matrix of the taps).
// The signal of one channel is cut into blocks of T = 128 outputs; block b needs the T + M - 1
// inputs x[bT .. bT + T + M - 2], i.e. OVERLAPPING rows of an "A" matrix with row pitch T:
//     y[bT + n] = sum_c x[bT + c] * Tz[c][n],   Tz[c][n] = a[n + M-1 - c]  (0 outside the band)
// This is the fused kernel with MT = 0 (A = x, split into bf16 hi / lo on the fly), the Toeplitz
// matrix in place of the twiddles (built per call from the caller's taps, hi / lo split, K padded
// to a multiple of 64 with zero rows) and N = T output columns.  With 64 taps 2/3 of the MMA work
// is useful and the kernel is bound by HBM, not by the fp32 pipes (the CUDA-core kernel is
// register-file-bandwidth bound at ~16 TFMA/s, 31 % of the HBM roofline at config 3).
// =====================================================================================
namespace tina {

constexpr int FIR_T = 128;

__global__ void toeplitz_kernel(__nv_bfloat16* __restrict__ tz, const float* __restrict__ taps, int M, int Kp)
{
    const int total = FIR_T * Kp;
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < total; e += gridDim.x * blockDim.x) {
        const int n = e / Kp, c = e % Kp;
        const int k = n + M - 1 - c;
        const float v = (k >= 0 && k < M) ? taps[k] : 0.f;
        const __nv_bfloat16 hi = __float2bfloat16(v);
        tz[e] = hi;
        tz[total + e] = __float2bfloat16(v - __bfloat162float(hi));
    }
}

bool umma_fir(const float* x, const float* taps, float* y, int C, long long L, int M, cudaStream_t st,
              tina_status* status)
{
    if (M > 193 || (L & 1) || options().fir_simt) return false;
    const long long Lo = L - M + 1;
    const int Kp = (FIR_T + M - 1 + KC - 1) / KC * KC;
    const long long R = (Lo + FIR_T - 1) / FIR_T;                    // output blocks (A rows) per channel
    const long long tps = (R + BM * UMMA_CG - 1) / (BM * UMMA_CG);
    if (tps * C > 0x7fffffffLL) return false;

    // Toeplitz scratch: a small ring of device buffers (the matrix is rebuilt from the caller's taps on every
    // call, in stream order; eight calls may be in flight on different streams before a buffer is reused)
    constexpr int kRing = 8;
    constexpr size_t kTzBytes = (size_t)2 * FIR_T * 320 * sizeof(__nv_bfloat16);
    DevCtx* ctx = nullptr;
    if ((*status = dev_ctx(&ctx)) != TINA_OK) return true;
    const int n_sm = ctx->n_sm;
    {
        std::lock_guard<std::mutex> lk(ctx->mu);
        if (!ctx->tz_ring) {
            cudaError_t e = cudaMalloc(&ctx->tz_ring, kRing * kTzBytes);
            if (e != cudaSuccess) { ctx->tz_ring = nullptr; *status = check_cuda(e, "cudaMalloc(toeplitz)"); return true; }
        }
    }
    __nv_bfloat16* tz = reinterpret_cast<__nv_bfloat16*>(static_cast<char*>(ctx->tz_ring) + (ctx->tz_next.fetch_add(1) % kRing) * kTzBytes);
    toeplitz_kernel<<<(FIR_T * Kp + 255) / 256, 256, 0, st>>>(tz, taps, M, Kp);
    count_launch();
    CUtensorMap tmap, zero1, zero2;
    memset(&zero1, 0, sizeof(zero1));
    memset(&zero2, 0, sizeof(zero2));
    EncodeTiledFn enc = encode_fn();
    tina_status rs = TINA_OK;
    if (!enc) rs = fail(TINA_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found");
    if (rs == TINA_OK) {
        const cuuint64_t dims[2] = {(cuuint64_t)Kp, (cuuint64_t)2 * FIR_T};
        const cuuint64_t strides[1] = {(cuuint64_t)Kp * sizeof(__nv_bfloat16)};
        const cuuint32_t box[2] = {(cuuint32_t)KC, (cuuint32_t)(FIR_T / UMMA_CG)};
        const cuuint32_t estr[2] = {1, 1};
        CUresult r = enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, tz, dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                         CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) rs = fail(TINA_ERR_CUDA, "cuTensorMapEncodeTiled(toeplitz) failed (%d)", (int)r);
    }
    if (rs == TINA_OK) {
        UmmaParams prm;
        memset(&prm, 0, sizeof(prm));
        prm.x = x; prm.window = nullptr; prm.out = y;
        prm.stream_stride = L;
        prm.F = R; prm.NBLK = R;
        prm.out_row = FIR_T; prm.out_stream_stride = Lo;
        prm.K = Kp; prm.N = FIR_T;
        prm.x_row_stride = FIR_T; prm.x_len = L; prm.out_len = Lo; prm.out_scalar = 1;
        prm.P = FIR_T; prm.M = 1;
        prm.tiles_per_stream = (int)tps;
        prm.nt_pass = NT_MAX; prm.n_passes = 1;
        prm.total_work = (int)(tps * C);
        prm.parts = 2;
        prm.out_tma = 0;
        prm.a_ring_bytes = 2 * 2 * A_PART_BYTES;                  // 2 slots of hi+lo
        prm.b_ring_bytes = 4 * (B_ENTRY_BYTES / UMMA_CG);         // 4 half-tile entries (only 64 rows of each are used)
        prm.stage_bytes = 32 * FIR_PITCH * 4;                     // 32 rows x 128 columns per epilogue warp
        prm.debug = 0;
        prm.k_splits = 1; prm.kc_per_split = Kp / KC;
        const int n_cl = n_sm / UMMA_CG;
        const int grid = UMMA_CG * (prm.total_work < n_cl ? prm.total_work : n_cl);
        rs = launch_umma<0, false, false>(ctx, tmap, zero1, zero2, prm, grid, st);
    }
    *status = rs;
    return true;
}

}  // namespace tina
