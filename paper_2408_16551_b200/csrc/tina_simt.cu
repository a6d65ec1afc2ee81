// tina_simt.cu -- CUDA-core kernels of libtina (sm_100a):
//   * fir_kernel        standalone FIR, Eq. (15) PAPER.md:171 (register-tiled, smem-staged)
//   * pfb_simt_kernel   generic-size PFB / DFT: Eq. (20) PAPER.md:230 + direct DFT Eq. (12)/(14)
//   * pfb_fir_kernel    subfilter stage only (Fig. 3 left column)
// These serve sizes the tcgen05 path does not cover and the HBM-bound regime (small P).
#include "tina_common.cuh"

namespace tina {

// =====================================================================================
// FIR: y[c][j] = sum_k a[k] x[c][j + M-1-k] = sum_i ta[i] x[c][j+i],  ta[i] = a[M-1-i]
// One CTA computes FIR_TILE consecutive outputs of one channel; each thread owns 16
// consecutive outputs and slides a 16-register window over the staged input, so the hot loop
// is 256 FFMA per 16 LDS.32 (window) + 4 broadcast LDS.128 (taps).  The input tile is staged
// TRANSPOSED -- element e lives at [e % 16][e / 16] with a row pitch = 2 (mod 32) -- so that
// both the coalesced fill (consecutive e per lane) and the per-thread walk (lane t reads
// element 16 t + m: row m % 16, column t + m / 16) are bank-conflict free.  Results leave
// through the same tile for fully coalesced stores.
// =====================================================================================
__device__ __forceinline__ float2 ffma2s(float2 a, float2 b, float2 c)
{
    float2 d;
    asm("{\n\t.reg .b64 ra, rb, rc, rd;\n\tmov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\tmov.b64 rc, {%6, %7};\n\t"
        "fma.rn.f32x2 rd, ra, rb, rc;\n\tmov.b64 {%0, %1}, rd;\n\t}"
        : "=f"(d.x), "=f"(d.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y), "f"(c.x), "f"(c.y));
    return d;
}

constexpr int FIR_THREADS = 256;
constexpr int FIR_PER_THREAD = 16;
constexpr int FIR_TILE = FIR_THREADS * FIR_PER_THREAD;  // 4096 outputs per CTA

// Row pitch of the transposed tile: compile-time (immediate address offsets in the hot loop), = 2 mod 32.
constexpr int FIR_LD_SMALL = 290;    // M <= 512  (needs 256 + Mp/16 + 1 columns)
constexpr int FIR_LD_LARGE = 514;    // M <= 4096

// Shared-memory load the compiler may not merge with another load of the same word: the E and O
// windows both hold every sample, and a register move instead of the second LDS would cost an
// FMA-pipe slot (IMAD.MOV) in a loop that is bound by that pipe.
__device__ __forceinline__ float lds_nomerge(const float* p)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"((unsigned)__cvta_generic_to_shared(p)));
    return v;
}

// two unmerged 32-bit shared loads straight into the halves of one 64-bit register pair
__device__ __forceinline__ unsigned long long lds_pair(const float* plo, const float* phi)
{
    unsigned long long v;
    asm volatile("{\n\t.reg .f32 lo, hi;\n\tld.volatile.shared.f32 lo, [%1];\n\tld.volatile.shared.f32 hi, [%2];\n\tmov.b64 %0, {lo, hi};\n\t}"
                 : "=l"(v) : "r"((unsigned)__cvta_generic_to_shared(plo)), "r"((unsigned)__cvta_generic_to_shared(phi)));
    return v;
}
// d = (a, a) * b + c on packed fp32 pairs held in 64-bit registers
__device__ __forceinline__ unsigned long long ffma2_bcast(float a, unsigned long long b, unsigned long long c)
{
    unsigned long long d;
    asm("{\n\t.reg .b64 ra;\n\tmov.b64 ra, {%1, %1};\n\tfma.rn.f32x2 %0, ra, %2, %3;\n\t}" : "=l"(d) : "f"(a), "l"(b), "l"(c));
    return d;
}

__device__ __forceinline__ void cp_async4(float* dst_smem, const float* src, bool valid)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst_smem);
    const int sz = valid ? 4 : 0;                      // src-size 0: the 4 bytes are zero-filled
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(d), "l"(src), "r"(sz) : "memory");
}

// Persistent: each CTA walks tiles blockIdx.x, + gridDim.x, ...; the next tile is staged with
// cp.async (LDGSTS) into the other buffer while the current one is being filtered.
template <int LD>
__global__ void __launch_bounds__(FIR_THREADS)
fir_kernel(const float* __restrict__ x, const float* __restrict__ taps, float* __restrict__ y,
           long long L, int M, long long Lo, int tiles_per_chan, int total_tiles, int taps_stride)
{
    extern __shared__ __align__(16) float smem[];
    const int Mp = (M + 15) & ~15;                     // taps padded to a multiple of 16 (zeros)
    float* s_taps = smem;                              // [Mp]  reversed: s_taps[i] = a[M-1-i]
    float* s_buf0 = smem + Mp;                         // 2 x [16][LD] input tiles, then [16][LD] output tile
    float* s_out = s_buf0 + 2 * 16 * LD;
    const int n_stage = FIR_TILE + Mp;                 // elements the walk may touch

    auto stage = [&](int tile, float* dst) {
        const int c = tile / tiles_per_chan;
        const long long j0 = (long long)(tile % tiles_per_chan) * FIR_TILE;
        const float* xc = x + (long long)c * L + j0;
        const int n_in = (int)min((long long)FIR_TILE, Lo - j0) + M - 1;
        for (int e = threadIdx.x; e < n_stage; e += FIR_THREADS)
            cp_async4(dst + (e & 15) * LD + (e >> 4), xc + (e < n_in ? e : 0), e < n_in);
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    // taps_stride == 0: one tap vector for every channel (loaded once); otherwise channel c filters with
    // taps + c * taps_stride, reloaded whenever the tile's channel changes (every read of s_taps for the
    // previous tile lies before the __syncthreads() that follows its s_out writes)
    int tile = blockIdx.x, buf = 0, cur_chan = -1;
    if (tile < total_tiles) stage(tile, s_buf0);
    for (; tile < total_tiles; tile += gridDim.x, buf ^= 1) {
    {
        const int c = taps_stride ? tile / tiles_per_chan : 0;
        if (c != cur_chan) {
            const float* tc = taps + (long long)c * taps_stride;
            for (int i = threadIdx.x; i < Mp; i += FIR_THREADS) s_taps[i] = (i < M) ? __ldg(tc + (M - 1 - i)) : 0.f;
            cur_chan = c;
        }
    }
    float* s_x = s_buf0 + buf * 16 * LD;
    const int nxt = tile + gridDim.x;
    if (nxt < total_tiles) { stage(nxt, s_buf0 + (buf ^ 1) * 16 * LD); asm volatile("cp.async.wait_group 1;" ::: "memory"); }
    else asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncthreads();                                   // tile `tile` (and the taps) are visible to every thread

    // Packed arithmetic (fma.rn.f32x2): the 16 outputs are 8 accumulator pairs (y[2q], y[2q+1]); tap i
    // multiplies the input pair (x[2q+i], x[2q+i+1]).  64-bit operands must be aligned register
    // pairs, so two windows are kept: E[m] = (x[2m], x[2m+1]) for even taps, O[m] = (x[2m+1], x[2m+2])
    // for odd taps (8 pairs each, refreshed with two LDS.32 per pair as the walk advances).
    const int t = threadIdx.x;
    unsigned long long acc[8], E[8], O[8];             // packed fp32 pairs
    const float* c0 = s_x + t;                         // element 16 t + m lives at c0[(m & 15) * LD + (m >> 4)]
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        acc[q] = 0ull;
        E[q] = lds_pair(c0 + (2 * q) * LD, c0 + (2 * q + 1) * LD);
        O[q] = lds_pair(c0 + (2 * q + 1) * LD, q < 7 ? c0 + (2 * q + 2) * LD : c0 + 1);
    }
    const float* col = s_x + t + 1;                    // column of element 16 t + 16 + i0 + (row)
    for (int i0 = 0; i0 < Mp; i0 += 16, ++col) {
#pragma unroll
        for (int u4 = 0; u4 < 16; u4 += 4) {
            const float4 tq = *reinterpret_cast<const float4*>(s_taps + i0 + u4);
            const float tp[4] = {tq.x, tq.y, tq.z, tq.w};
#pragma unroll
            for (int v = 0; v < 4; ++v) {
                const int u = u4 + v;                  // tap i = i0 + u
                if ((u & 1) == 0) {
                    // pairs (x[2q+i], x[2q+i+1]) = E[q + i/2]; slot (q + u/2) & 7
#pragma unroll
                    for (int q = 0; q < 8; ++q) acc[q] = ffma2_bcast(tp[v], E[(q + u / 2) & 7], acc[q]);
                    // slot (u/2) & 7 held E[i/2]; it next holds E[i/2 + 8] = (x[i+16], x[i+17])
                    E[(u / 2) & 7] = lds_pair(col + u * LD, col + (u + 1) * LD);
                } else {
                    // pairs = O[q + (i-1)/2]
#pragma unroll
                    for (int q = 0; q < 8; ++q) acc[q] = ffma2_bcast(tp[v], O[(q + u / 2) & 7], acc[q]);
                    // O[(i-1)/2 + 8] = (x[i+16], x[i+17]); row of x[i+17] wraps to the next column at u = 15
                    O[(u / 2) & 7] = lds_pair(col + u * LD, u < 15 ? col + (u + 1) * LD : col + 1);
                }
            }
        }
    }
    // results leave through their own transposed tile (conflict-free writes, coalesced stores)
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        s_out[(2 * q) * LD + t] = __uint_as_float((unsigned)(acc[q] & 0xffffffffull));
        s_out[(2 * q + 1) * LD + t] = __uint_as_float((unsigned)(acc[q] >> 32));
    }
    __syncthreads();                                   // also: everyone is done reading s_x before it is restaged
    {
        const int c = tile / tiles_per_chan;
        const long long j0 = (long long)(tile % tiles_per_chan) * FIR_TILE;
        const int n_out = (int)min((long long)FIR_TILE, Lo - j0);
        float* yc = y + (long long)c * Lo + j0;
        for (int e = threadIdx.x; e < n_out; e += FIR_THREADS) yc[e] = s_out[(e & 15) * LD + (e >> 4)];
    }
    }
}

tina_status simt_fir(const float* x, const float* taps, float* y, int C, long long L, int M,
                     cudaStream_t st, bool per_channel)
{
    const int taps_stride = per_channel ? M : 0;
    const long long Lo = L - M + 1;
    const long long tiles = (Lo + FIR_TILE - 1) / FIR_TILE;
    if (tiles * C > 0x7fffffffLL) return fail(TINA_ERR_UNSUPPORTED, "tina_fir: C*L too large for one grid");
    const int Mp = (M + 15) & ~15;
    const bool small = Mp <= 512;
    const size_t smem = sizeof(float) * ((size_t)Mp + 3 * 16 * (size_t)(small ? FIR_LD_SMALL : FIR_LD_LARGE));
    DevCtx* ctx = nullptr;
    tina_status cs = dev_ctx(&ctx);
    if (cs != TINA_OK) return cs;
    const int n_sm = ctx->n_sm;
    const void* kern = small ? (const void*)fir_kernel<FIR_LD_SMALL> : (const void*)fir_kernel<FIR_LD_LARGE>;
    if ((cs = ensure_smem(ctx, kern, small ? 64 * 1024 : 120 * 1024, "fir_kernel setup")) != TINA_OK) return cs;
    const long long total = tiles * C;
    // resident CTAs per SM (registers / shared memory): a persistent grid must not exceed one wave.  The query
    // depends on the dynamic shared memory size, i.e. on Mp: cached per (device, kernel, Mp).
    int occ = 0;
    {
        std::lock_guard<std::mutex> lk(ctx->mu);
        const void* key = reinterpret_cast<const char*>(kern) + Mp;       // distinct key per padded tap count
        auto it = ctx->occupancy.find(key);
        if (it != ctx->occupancy.end()) occ = it->second;
        else {
            cudaError_t e = small ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fir_kernel<FIR_LD_SMALL>, FIR_THREADS, smem)
                                  : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fir_kernel<FIR_LD_LARGE>, FIR_THREADS, smem);
            if (e != cudaSuccess || occ < 1) return check_cuda(e != cudaSuccess ? e : cudaErrorLaunchOutOfResources, "cudaOccupancyMaxActiveBlocksPerMultiprocessor(fir_kernel)");
            ctx->occupancy[key] = occ;
        }
    }
    const int per_sm = occ;
    const unsigned grid = (unsigned)(total < (long long)n_sm * per_sm ? total : (long long)n_sm * per_sm);
    if (small)
        fir_kernel<FIR_LD_SMALL><<<grid, FIR_THREADS, smem, st>>>(x, taps, y, L, M, Lo, (int)tiles, (int)total, taps_stride);
    else
        fir_kernel<FIR_LD_LARGE><<<grid, FIR_THREADS, smem, st>>>(x, taps, y, L, M, Lo, (int)tiles, (int)total, taps_stride);
    count_launch();
    g_last_path = kPathSimt; note_kernel("fir_kernel");
    return check_cuda(cudaGetLastError(), "fir_kernel launch");
}

// =====================================================================================
// Generic-size PFB / DFT on CUDA cores.
// One CTA handles TF consecutive frames of one stream: (1) subfilter stage into a shared
// y tile, Eq. (20); (2) direct DFT across the P branches with a shared twiddle table
// W[r] = exp(-+2 pi i r / P), r = (p k) mod P advanced in integers.
// =====================================================================================
constexpr int PFB_SIMT_THREADS = 256;

template <bool REAL>
__global__ void __launch_bounds__(PFB_SIMT_THREADS)
pfb_simt_kernel(const void* __restrict__ x_, long long stream_stride, int P, int M,
                const float* __restrict__ window, long long F, int TF, int tiles_per_stream,
                int inverse, float scale, void* __restrict__ out_)
{
    extern __shared__ __align__(16) float smem[];
    float2* s_w = reinterpret_cast<float2*>(smem);                 // [P] twiddles
    float*  s_y = smem + 2 * P;                                    // [TF][P] (float or float2)

    const int s = blockIdx.x / tiles_per_stream;
    const long long f0 = (long long)(blockIdx.x % tiles_per_stream) * TF;
    const int nf = (int)min((long long)TF, F - f0);
    const int NK = REAL ? P / 2 + 1 : P;

    for (int r = threadIdx.x; r < P; r += blockDim.x) {
        double sn, cs;
        sincospi(2.0 * (double)r / (double)P, &sn, &cs);
        s_w[r] = make_float2((float)cs, (float)(inverse ? sn : -sn));
    }
    // ---- subfilter stage -------------------------------------------------------------
    if (REAL) {
        const float* x = reinterpret_cast<const float*>(x_) + (long long)s * stream_stride;
        for (int e = threadIdx.x; e < nf * P; e += blockDim.x) {
            const int f = e / P, p = e - f * P;
            float acc = 0.f;
            if (window) {
                for (int m = 0; m < M; ++m)
                    acc = fmaf(__ldg(window + (long long)m * P + p),
                               __ldg(x + (f0 + f + M - 1 - m) * P + p), acc);
            } else {
                acc = __ldg(x + (f0 + f) * P + p);
            }
            s_y[e] = acc;
        }
    } else {
        const float2* x = reinterpret_cast<const float2*>(x_) + (long long)s * stream_stride;
        float2* sy = reinterpret_cast<float2*>(s_y);
        for (int e = threadIdx.x; e < nf * P; e += blockDim.x) {
            const int f = e / P, p = e - f * P;
            float2 acc = make_float2(0.f, 0.f);
            if (window) {
                for (int m = 0; m < M; ++m) {
                    const float h = __ldg(window + (long long)m * P + p);
                    const float2 v = __ldg(x + (f0 + f + M - 1 - m) * P + p);
                    acc.x = fmaf(h, v.x, acc.x);
                    acc.y = fmaf(h, v.y, acc.y);
                }
            } else {
                acc = __ldg(x + (f0 + f) * P + p);
            }
            sy[e] = acc;
        }
    }
    __syncthreads();
    // ---- Fourier stage ---------------------------------------------------------------
    float2* out = reinterpret_cast<float2*>(out_) + ((long long)s * F + f0) * NK;
    for (int e = threadIdx.x; e < nf * NK; e += blockDim.x) {
        const int f = e / NK, k = e - f * NK;
        float ar = 0.f, ai = 0.f;
        int r = 0;
        if (REAL) {
            const float* yr = s_y + f * P;
            for (int p = 0; p < P; ++p) {
                const float2 w = s_w[r];
                ar = fmaf(yr[p], w.x, ar);
                ai = fmaf(yr[p], w.y, ai);
                r += k; if (r >= P) r -= P;
            }
        } else {
            const float2* yc = reinterpret_cast<const float2*>(s_y) + f * P;
            for (int p = 0; p < P; ++p) {
                const float2 w = s_w[r];
                const float2 v = yc[p];
                ar = fmaf(v.x, w.x, ar); ar = fmaf(-v.y, w.y, ar);
                ai = fmaf(v.x, w.y, ai); ai = fmaf(v.y, w.x, ai);
                r += k; if (r >= P) r -= P;
            }
        }
        out[e] = make_float2(ar * scale, ai * scale);
    }
}

tina_status simt_pfb(const void* x, int S, long long n_samples, int P, int M, const float* window,
                     bool real, bool inverse, void* out, cudaStream_t st)
{
    const long long F = n_samples / P - M + 1;
    const int elem = real ? 1 : 2;                       // floats per y element
    const long long budget = 40 * 1024 / 4;              // floats of smem for the y tile
    int TF = (int)(budget / ((long long)P * elem));
    if (TF < 1) TF = 1;
    if (TF > 64) TF = 64;
    // keep at least ~2 waves of CTAs when the problem is small
    while (TF > 1 && (F + TF - 1) / TF * S < 2 * 148) TF >>= 1;
    const long long tiles = (F + TF - 1) / TF;
    if (tiles * S > 0x7fffffffLL) return fail(TINA_ERR_UNSUPPORTED, "tina_pfb: too many tiles");
    const size_t smem = sizeof(float) * (2 * (size_t)P + (size_t)TF * P * elem);
    DevCtx* ctx = nullptr;
    tina_status cs = dev_ctx(&ctx);
    if (cs != TINA_OK) return cs;
    const void* kern = real ? (const void*)pfb_simt_kernel<true> : (const void*)pfb_simt_kernel<false>;
    if ((cs = ensure_smem(ctx, kern, 200 * 1024, "cudaFuncSetAttribute(pfb_simt_kernel)")) != TINA_OK) return cs;
    const float scale = inverse ? (float)(1.0 / (double)P) : 1.f;
    if (real)
        pfb_simt_kernel<true><<<(unsigned)(tiles * S), PFB_SIMT_THREADS, smem, st>>>(
            x, n_samples, P, M, window, F, TF, (int)tiles, inverse ? 1 : 0, scale, out);
    else
        pfb_simt_kernel<false><<<(unsigned)(tiles * S), PFB_SIMT_THREADS, smem, st>>>(
            x, n_samples, P, M, window, F, TF, (int)tiles, inverse ? 1 : 0, scale, out);
    count_launch();
    g_last_path = kPathSimt; note_kernel("pfb_simt_kernel");
    return check_cuda(cudaGetLastError(), "pfb_simt_kernel launch");
}

// =====================================================================================
// Subfilter stage only: y[s][f][p] = sum_m w[mP+p] x[s][(f+M-1-m)P+p].
// A thread owns one 8-byte column (one complex sample, or two adjacent real branches) and
// RUN consecutive frames, walking the RUN+M-1 input rows once: HBM sees each sample once,
// the (M-1)-row halo between neighbouring runs is served by L2.
// =====================================================================================
constexpr int PF_RUN = 16;

template <bool REAL>
__global__ void __launch_bounds__(256)
pfb_fir_kernel(const float2* __restrict__ x, long long stream_stride2, int P2, int M,
               const float* __restrict__ window, long long F, float2* __restrict__ y,
               long long total_cols, int runs_per_stream)
{
    // column index c in [0,P2): float2 column (P2 = P for complex, P/2 for real)
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= total_cols) return;
    const int c = (int)(gid % P2);
    const long long rs = gid / P2;
    const int run = (int)(rs % runs_per_stream);
    const int s = (int)(rs / runs_per_stream);
    const long long f0 = (long long)run * PF_RUN;
    const int nf = (int)min((long long)PF_RUN, F - f0);
    const float2* xs = x + (long long)s * stream_stride2 + c;
    const int Pw = REAL ? 2 * P2 : P2;                   // window row length P

    float2 acc[PF_RUN];
#pragma unroll
    for (int r = 0; r < PF_RUN; ++r) acc[r] = make_float2(0.f, 0.f);
    for (int i = 0; i < nf + M - 1; ++i) {
        const float2 v = __ldg(xs + (f0 + i) * P2);
#pragma unroll
        for (int r = 0; r < PF_RUN; ++r) {
            const int m = r + M - 1 - i;                 // input row f0+i feeds frame f0+r with tap m
            if (m >= 0 && m < M && r < nf) {
                if (REAL) {
                    const float2 h = __ldg(reinterpret_cast<const float2*>(window + (long long)m * Pw) + c);
                    acc[r].x = fmaf(h.x, v.x, acc[r].x);
                    acc[r].y = fmaf(h.y, v.y, acc[r].y);
                } else {
                    const float h = __ldg(window + (long long)m * Pw + c);
                    acc[r].x = fmaf(h, v.x, acc[r].x);
                    acc[r].y = fmaf(h, v.y, acc[r].y);
                }
            }
        }
    }
    float2* ys = y + ((long long)s * F + f0) * P2 + c;
#pragma unroll
    for (int r = 0; r < PF_RUN; ++r)
        if (r < nf) ys[(long long)r * P2] = acc[r];
}

tina_status simt_pfb_fir(const void* x, int S, long long n_samples, int P, int M,
                         const float* window, bool real, void* y, cudaStream_t st)
{
    const long long F = n_samples / P - M + 1;
    const int P2 = real ? P / 2 : P;
    const long long stride2 = real ? n_samples / 2 : n_samples;
    const long long runs = (F + PF_RUN - 1) / PF_RUN;
    const long long total = runs * S * P2;
    const long long blocks = (total + 255) / 256;
    if (blocks > 0x7fffffffLL) return fail(TINA_ERR_UNSUPPORTED, "tina_pfb_fir: too large");
    if (real)
        pfb_fir_kernel<true><<<(unsigned)blocks, 256, 0, st>>>(
            (const float2*)x, stride2, P2, M, window, F, (float2*)y, total, (int)runs);
    else
        pfb_fir_kernel<false><<<(unsigned)blocks, 256, 0, st>>>(
            (const float2*)x, stride2, P2, M, window, F, (float2*)y, total, (int)runs);
    count_launch();
    g_last_path = kPathSimt; note_kernel("pfb_fir_kernel");
    return check_cuda(cudaGetLastError(), "pfb_fir_kernel launch");
}

// =====================================================================================
// Unfolding, Eq. (17): Y(i, j) = X(i + j).  One thread per output element, flat index
// e = i J + j: consecutive threads write consecutive addresses and read x[i + j] (stride-1 within
// a row, rows overlap by J - 1: L1 / L2 hits).
// =====================================================================================
__global__ void __launch_bounds__(256)
unfold_kernel(const float* __restrict__ x, float* __restrict__ y, long long total, int J)
{
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total;
         e += (long long)gridDim.x * blockDim.x) {
        const long long i = e / J;
        const int j = (int)(e - i * J);
        y[e] = __ldg(x + i + j);
    }
}

tina_status simt_unfold(const float* x, float* y, long long I, int J, cudaStream_t st)
{
    const long long total = (I - J + 1) * (long long)J;
    long long blocks = (total + 255) / 256;
    if (blocks > 148LL * 32) blocks = 148LL * 32;
    unfold_kernel<<<(unsigned)blocks, 256, 0, st>>>(x, y, total, J);
    count_launch();
    g_last_path = kPathSimt; note_kernel("unfold_kernel");
    return check_cuda(cudaGetLastError(), "unfold_kernel launch");
}

}  // namespace tina
