"""GPU parity: libtina (through the C ABI binding) vs the float64 oracle, element by element
on identical seeded inputs.  Tolerances (BASELINE.json north_star):
relative L2 per output frame <= 1e-5 (fp32 configs), <= 2e-2 (bf16 config)."""
import numpy as np
import pytest

import tina_inputs as ti
from conftest import rel_l2_rows

pytestmark = pytest.mark.gpu

TOL_FP32 = 1e-5
TOL_BF16 = 2e-2


@pytest.fixture(scope="module")
def tina():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2408_16551_b200 as t
    t.lib()  # raises if libtina.so is missing -- no fallback
    return t


@pytest.fixture
def tina_env(tina, monkeypatch):
    """Set TINA_* variant switches for one test: the library reads its environment once, so the
    options are reloaded after every change and once more when the test ends."""
    def set_(**kv):
        for k, v in kv.items():
            monkeypatch.setenv(k, str(v))
        tina.reload_options()
    yield set_
    monkeypatch.undo()
    tina.reload_options()


def _cuda(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _run_pfb(tina, case, prec=0):
    import torch
    x = _cuda(case.x)
    w = _cuda(case.window)
    out = tina.pfb(x, case.P, case.M, w, prec=prec)
    torch.cuda.synchronize()
    return out.cpu().numpy()


# ------------------------------------------------------------------ FIR
@pytest.mark.parametrize("C,L,K", [(1, 64, 64), (3, 5000, 64), (2, 2048 + 63, 64), (2, 2049 + 63, 64),
                                   (5, 777, 1), (2, 9000, 7), (1, 4500, 200), (4, 100000, 64)])
def test_fir_parity_small(tina, oracle, C, L, K):
    import torch
    rng = np.random.default_rng(100 + C * 7 + K)
    x = ti.noise_real(rng, C * L).reshape(C, L)
    a = ti.random_taps(rng, K)                       # asymmetric: a flipped kernel would fail
    y = tina.fir(_cuda(x), _cuda(a))
    torch.cuda.synchronize()
    ref = oracle.fir(x, a)
    assert y.shape == ref.shape
    assert rel_l2_rows(y.cpu().numpy(), ref) <= TOL_FP32


def test_fir_impulse_response_is_taps(tina):
    import torch
    K = 64
    a = ti.random_taps(np.random.default_rng(5), K)
    x = np.zeros((1, 2 * K - 1), np.float32); x[0, K - 1] = 1
    y = tina.fir(_cuda(x), _cuda(a))
    torch.cuda.synchronize()
    assert np.array_equal(y.cpu().numpy()[0], a)


@pytest.mark.parametrize("C,L,K", [(2, 128 + 192, 193), (3, 4096, 1), (1, 130, 3), (5, 33000, 129), (2, 70000, 65)])
def test_fir_toeplitz_tensor_path(tina, oracle, C, L, K):
    """Even L and K <= 193 run as a banded-Toeplitz contraction on the tensor cores (the paper's
    unfolding view): ragged last block, K = 1, the largest covered K."""
    import torch
    rng = np.random.default_rng(150 + K)
    x = ti.noise_real(rng, C * L).reshape(C, L)
    a = ti.random_taps(rng, K)
    y = tina.fir(_cuda(x), _cuda(a))
    torch.cuda.synchronize()
    assert tina.last_path() == 2
    ref = oracle.fir(x, a)
    assert y.shape == ref.shape
    assert rel_l2_rows(y.cpu().numpy(), ref) <= TOL_FP32
    # impulse response = taps in order (to the bf16x3 split accuracy of each tap)
    xi = np.zeros((1, 2 * K + 2), np.float32); xi[0, K - 1] = 1
    yi = tina.fir(_cuda(xi), _cuda(a)); torch.cuda.synchronize()
    assert np.allclose(yi.cpu().numpy()[0, :K], a, rtol=2e-5, atol=1e-6 * np.abs(a).max())


@pytest.mark.parametrize("C,L,K", [(1, 128, 64), (3, 4096, 1), (2, 128 * 70, 64), (5, 128 * 300, 193), (2, 128 * 257, 33),
                                   (3, 128 * 1025, 64), (70, 128 * 40, 17)])
@pytest.mark.parametrize("per_channel", [False, True])
def test_fir_resident_toeplitz_kernel(tina, oracle, C, L, K, per_channel):
    """L % 128 == 0 and K <= 193: fir_umma_kernel (Toeplitz matrix resident in shared memory, signal staged by TMA,
    operand in tensor memory, three accumulator stages).  Single block, one tap, the largest K, ragged last tile, more channels than CTA pairs
    (per-channel taps rebuild the matrix at every channel change); asymmetric random taps."""
    import torch
    rng = np.random.default_rng(190 + C + K)
    x = ti.noise_real(rng, C * L).reshape(C, L)
    if per_channel:
        a = rng.standard_normal((C, K)).astype(np.float32)
        y = tina.fir_multi(_cuda(x), _cuda(a)); ref = oracle.fir_multi(x, a)
    else:
        a = ti.random_taps(rng, K)
        y = tina.fir(_cuda(x), _cuda(a)); ref = oracle.fir(x, a)
    torch.cuda.synchronize()
    assert tina.last_kernel().startswith("fir_umma_kernel")
    assert y.shape == ref.shape
    assert rel_l2_rows(y.cpu().numpy(), ref) <= TOL_FP32


def test_fir_round1_toeplitz_route_still_correct(tina, oracle, tina_env):
    import torch
    tina_env(TINA_FIR_V1=1)
    rng = np.random.default_rng(199)
    x = ti.noise_real(rng, 3 * 128 * 40).reshape(3, 128 * 40)
    a = ti.random_taps(rng, 64)
    y = tina.fir(_cuda(x), _cuda(a)); torch.cuda.synchronize()
    assert tina.last_kernel() == "pfb_umma_kernel"
    assert rel_l2_rows(y.cpu().numpy(), oracle.fir(x, a)) <= TOL_FP32


def test_unfold_matches_oracle_and_paper_example(tina, oracle):
    """Eq. (17); bit-exact (a gather).  Includes the paper's worked example."""
    import torch
    y = tina.unfold(_cuda(np.array([1, 2, 3, 4], np.float32)), 2); torch.cuda.synchronize()
    assert np.array_equal(y.cpu().numpy(), np.array([[1, 2], [2, 3], [3, 4]], np.float32))
    rng = np.random.default_rng(77)
    for (I, J) in [(1, 1), (1000, 1), (1000, 1000), (70001, 64), (5000, 333)]:
        x = ti.noise_real(rng, I)
        y = tina.unfold(_cuda(x), J); torch.cuda.synchronize()
        assert np.array_equal(y.cpu().numpy().astype(np.float64), oracle.unfold(x, J))


def test_config3_fir_full(tina, oracle):
    """c3 at full size; per-channel rel L2 and per-4096-sample-block rel L2."""
    import torch
    x, taps, taps_asym = ti.config3()
    xd = _cuda(x)
    for a in (taps, taps_asym):
        y = tina.fir(xd, _cuda(a))
        torch.cuda.synchronize()
        y = y.cpu().numpy()
        ref = oracle.fir(x, a)
        assert y.shape == (64, (1 << 20) - 63)
        assert rel_l2_rows(y, ref) <= TOL_FP32
        nblk = ref.shape[1] // 4096
        yb = y[:, : nblk * 4096].reshape(-1, 4096)
        rb = ref[:, : nblk * 4096].reshape(-1, 4096)
        assert rel_l2_rows(yb, rb) <= TOL_FP32


# ------------------------------------------------------------------ DFT
@pytest.mark.parametrize("B,N", [(1, 2), (7, 3), (33, 12), (300, 16), (129, 100), (5, 250)])
def test_dft_generic_sizes(tina, oracle, B, N):
    import torch
    rng = np.random.default_rng(200 + N)
    x = ti.noise_complex(rng, B * N).reshape(B, N)
    Z = tina.dft(_cuda(x)); Xi = tina.dft(_cuda(x), inverse=True)
    torch.cuda.synchronize()
    assert rel_l2_rows(Z.cpu().numpy(), oracle.dft(x)) <= TOL_FP32
    assert rel_l2_rows(Xi.cpu().numpy(), oracle.dft(x, inverse=True)) <= TOL_FP32


@pytest.mark.parametrize("B,N", [(1, 32), (128, 32), (130, 64), (257, 96), (1000, 128), (300, 256),
                                 (77, 512), (140, 1024), (129, 2048)])
@pytest.mark.parametrize("prec,tol", [(0, TOL_FP32), (1, TOL_BF16)])
def test_dft_tensor_sizes(tina, oracle, B, N, prec, tol):
    """N % 32 == 0: tcgen05 path; spans several M tiles and a ragged tail."""
    import torch
    rng = np.random.default_rng(300 + N + B)
    x = ti.noise_complex(rng, B * N).reshape(B, N)
    Z = tina.dft(_cuda(x), prec=prec); Xi = tina.dft(_cuda(x), inverse=True, prec=prec)
    torch.cuda.synchronize()
    assert rel_l2_rows(Z.cpu().numpy(), oracle.dft(x)) <= tol
    assert rel_l2_rows(Xi.cpu().numpy(), oracle.dft(x, inverse=True)) <= tol


def test_dft_unit_impulse_and_tone(tina):
    import torch
    N = 256
    x = np.zeros((2, N), np.complex64)
    x[0, 0] = 1
    x[1] = np.exp(2j * np.pi * ((17 * np.arange(N)) % N) / N)
    Z = tina.dft(_cuda(x)); torch.cuda.synchronize()
    Z = Z.cpu().numpy()
    assert np.allclose(Z[0], 1, atol=1e-5)
    want = np.zeros(N, np.complex128); want[17] = N
    assert np.linalg.norm(Z[1] - want) / N <= TOL_FP32


def test_config2_dft_roundtrip_full(tina, oracle):
    """c2: B=65536, N=256 forward then inverse; oracle on a seeded row sample."""
    import torch
    x = ti.config2()
    xd = _cuda(x)
    Z = tina.dft(xd)
    xb = tina.dft(Z, inverse=True)
    torch.cuda.synchronize()
    rows = ti.sample_frames(x.shape[0], 480, ti.SEED_BASE + 2)
    assert rel_l2_rows(Z.cpu().numpy()[rows], oracle.dft(x[rows])) <= TOL_FP32
    xb = xb.cpu().numpy()
    assert rel_l2_rows(xb, x.astype(np.complex128)) <= 2 * TOL_FP32          # two transforms
    ref_rt = oracle.dft(oracle.dft(x[rows]), inverse=True)
    assert rel_l2_rows(xb[rows], ref_rt) <= 2 * TOL_FP32


# ------------------------------------------------------------------ PFB
@pytest.mark.parametrize("P,M,F,real", [
    (2, 1, 1, False), (4, 3, 5, False), (16, 4, 100, False), (10, 2, 33, True), (24, 5, 17, False),
    (32, 4, 300, False), (64, 8, 200, False), (64, 8, 129, True), (128, 16, 257, False),
    (256, 3, 140, True), (96, 2, 131, False), (192, 4, 70, True), (1024, 16, 130, False),
    (2048, 2, 129, True), (32, 1, 128, False), (64, 64, 40, False)])
def test_pfb_parity_small(tina, oracle, P, M, F, real):
    rng = np.random.default_rng(400 + P + M)
    case = ti.pfb_case(P, M, F, real=real, seed=401 + P, window=ti.random_taps(rng, P * M))
    got = _run_pfb(tina, case)
    ref = oracle.pfb(case.x[0], P, M, case.window)
    assert got.shape[1:] == ref.shape
    assert rel_l2_rows(got[0], ref) <= TOL_FP32


@pytest.mark.parametrize("P,M,F,real", [(64, 4, 200, False), (128, 8, 150, True), (1024, 16, 130, False)])
def test_pfb_bf16_small(tina, oracle, P, M, F, real):
    case = ti.pfb_case(P, M, F, real=real, seed=500 + P)
    got = _run_pfb(tina, case, prec=1)
    ref = oracle.pfb(case.x[0], P, M, case.window)
    assert rel_l2_rows(got[0], ref) <= TOL_BF16


@pytest.mark.parametrize("P,M,F,real", [(64, 4, 200, False), (256, 8, 150, True), (1024, 16, 130, False)])
def test_pfb_fp16_single_pass(tina, oracle, P, M, F, real):
    """TINA_PREC_FP16: the paper's "16 bit" variant (fp16 operands, fp32 accumulate)."""
    case = ti.pfb_case(P, M, F, real=real, seed=520 + P)
    got = _run_pfb(tina, case, prec=2)
    ref = oracle.pfb(case.x[0], P, M, case.window)
    err = rel_l2_rows(got[0], ref)
    assert err <= 2e-3            # 11-bit significands: ~4x tighter than the bf16 pass
    x = ti.noise_complex(np.random.default_rng(9), 300 * 256).reshape(300, 256)
    import torch
    Z = tina.dft(_cuda(x), prec=2); torch.cuda.synchronize()
    assert rel_l2_rows(Z.cpu().numpy(), oracle.dft(x)) <= 2e-3


def test_pfb_batched_streams_and_tail(tina, oracle):
    """S streams in one launch; n_samples not a multiple of P (tail ignored, reading R8)."""
    P, M, F, S = 64, 4, 140, 3
    case = ti.pfb_case(P, M, F, streams=S, seed=600)
    x = np.concatenate([case.x, np.ones((S, 6), np.complex64)], axis=1)     # ragged tail
    case.x = np.ascontiguousarray(x)
    got = _run_pfb(tina, case)
    assert got.shape == (S, F, P)
    for s in range(S):
        assert rel_l2_rows(got[s], oracle.pfb(case.x[s], P, M, case.window)) <= TOL_FP32


@pytest.mark.parametrize("P,M,F,S", [(128, 4, 130, 2), (128, 4, 129, 2), (2048, 2, 258, 2), (1024, 3, 131, 3),
                                     (2048, 2, 259, 2), (4096, 2, 131, 3), (2048, 3, 1, 2),
                                     (128, 4, 33, 1), (512, 8, 257, 1), (4096, 2, 67, 1), (8192, 2, 2, 1), (256, 4, 1, 1)])
def test_pfb_real_batched_epilogue_paths(tina, oracle, P, M, F, S):
    """Real kind: even F takes the TMA-store epilogue (row-pair tensor maps; 32- and 28-float boxes plus register
    edges), odd F with ONE stream too (its last row is stored from registers), odd F with S > 1 and F = 1 the
    register / shared-memory store path; P >= 1024 adds several accumulation chains (read-modify-write of the
    output) and several column passes."""
    case = ti.pfb_case(P, M, F, real=True, streams=S, seed=650 + P + F)
    got = _run_pfb(tina, case)
    assert got.shape == (S, F, P // 2 + 1)
    for s in range(S):
        ref = oracle.pfb(case.x[s], P, M, case.window)
        assert rel_l2_rows(got[s], ref) <= TOL_FP32
        assert np.all(got[s][:, 0].imag == 0) and np.all(got[s][:, P // 2].imag == 0)


@pytest.mark.parametrize("P,M,F,real,S", [(32, 1, 1, False, 1), (64, 16, 1, True, 3), (32, 4, 257, False, 5),
                                           (4096, 2, 130, False, 1), (8192, 2, 131, True, 1), (1024, 16, 513, False, 1)])
def test_pfb_tensor_path_edges(tina, oracle, P, M, F, real, S):
    """Single frame, ragged pair tiles, several streams, the largest contraction lengths (K = 8192:
    eight accumulation chains, 16 column passes)."""
    case = ti.pfb_case(P, M, F, real=real, streams=S, seed=680 + P + F)
    got = _run_pfb(tina, case)
    assert tina.last_path() == 2
    for s in range(S):
        assert rel_l2_rows(got[s], oracle.pfb(case.x[s], P, M, case.window)) <= TOL_FP32


@pytest.mark.parametrize("P,M,F,real,S", [(64, 32, 70, True, 2), (128, 17, 131, False, 2), (256, 64, 40, False, 1),
                                           (1024, 32, 300, False, 2), (4096, 24, 131, True, 1), (128, 33, 260, True, 2),
                                           (96, 20, 50, False, 1), (2048, 48, 257, False, 1)])
def test_pfb_many_taps(tina, oracle, P, M, F, real, S):
    """16 < M <= 64.  Where the column-paired kernel tiles the shape (P a multiple of 64; real kind P >= 128) the PFB
    stays ONE fused launch, the taps processed in groups of 16 inside the kernel (M not a multiple of 16: the last
    group's missing taps read as zeros); other shapes take the subfilter kernel into a stream-ordered temporary
    followed by the contraction (two launches).  Several streams, ragged tiles, several accumulation chains."""
    rng = np.random.default_rng(690 + P)
    case = ti.pfb_case(P, M, F, real=real, streams=S, seed=691 + P, window=ti.random_taps(rng, P * M))
    launches = tina.launch_count()
    got = _run_pfb(tina, case)
    fused = P % 64 == 0 and (P >= 128 or not real)
    if fused:
        assert tina.last_kernel() == ("pfb_symt_kernel<real, tap groups>" if real else "pfb_symt_kernel<tap groups>")
        assert tina.launch_count() - launches <= 2          # the kernel (+ the one-off twiddle plan)
    else:
        assert not tina.last_kernel().endswith("tap groups>")
    for s in range(S):
        assert rel_l2_rows(got[s], oracle.pfb(case.x[s], P, M, case.window)) <= TOL_FP32


@pytest.mark.parametrize("P,M,F,real,S", [(320, 5, 300, False, 1), (192, 3, 257, False, 2), (8192, 1, 40, False, 1),
                                           (320, 4, 200, True, 1), (256, 16, 100, True, 2), (128, 1, 513, True, 1),
                                           (1024, 16, 700, False, 3), (4096, 8, 300, True, 1), (64, 16, 1000, False, 1)])
def test_pfb_column_paired_kernel_shapes(tina, oracle, P, M, F, real, S):
    """Shapes that exercise the column-paired kernel's tiling (tina_sym.cu): a last pass narrower than 128 bins
    (P = 320, 192), one 32-element chunk per pass (P = 64), the longest contraction (P = 8192: eight accumulation
    chains with add-reduce epilogues), M below / at the unrolled tap counts, several streams, ragged frame tiles;
    both variants (TMA-staged input, and register-window producers where they exist) give the oracle's result."""
    rng = np.random.default_rng(640 + P + M)
    case = ti.pfb_case(P, M, F, real=real, streams=S, seed=641 + P + F, window=ti.random_taps(rng, P * M))
    got = _run_pfb(tina, case)
    assert tina.last_kernel().startswith("pfb_symt_kernel")
    for s in range(S):
        ref = oracle.pfb(case.x[s], P, M, case.window)
        assert rel_l2_rows(got[s], ref) <= TOL_FP32
        if real:
            assert np.all(got[s][:, 0].imag == 0) and np.all(got[s][:, P // 2].imag == 0)


def test_pfb_column_paired_variants_agree(tina, oracle, tina_env):
    """TINA_SYM_V1 (register-window producers) and TINA_NO_SYM (round-1 block-form kernel) stay correct."""
    case = ti.pfb_case(1024, 16, 300, streams=2, seed=655)
    ref = [oracle.pfb(case.x[s], 1024, 16, case.window) for s in range(2)]
    for env, name in (({"TINA_SYM_V1": 1}, "pfb_sym_kernel"), ({"TINA_NO_SYM": 1}, "pfb_umma_kernel")):
        tina_env(**env)
        got = _run_pfb(tina, case)
        assert tina.last_kernel() == name
        for s in range(2):
            assert rel_l2_rows(got[s], ref[s]) <= TOL_FP32
        tina_env(**{k: 0 for k in env})


@pytest.mark.parametrize("P,M,F,S", [(64, 4, 200, 1), (128, 16, 257, 2), (320, 5, 300, 1), (192, 3, 257, 2), (1024, 16, 700, 3),
                                     (1024, 1, 130, 1), (2048, 2, 300, 2), (4096, 8, 131, 1), (8192, 2, 40, 1)])
def test_pfb_row_paired_kernel(tina, oracle, tina_env, P, M, F, S):
    """TINA_SYM_FOLD=1: the complex kind with the row pairs (p, P - p) of the Fourier matrix folded as well
    (pfb_symf_kernel, tina_symf.cu): narrow last passes (P = 320, 192), two chunks per pass (P = 64), the unpaired
    samples p = 0 and p = P/2, the Nyquist bin through the extra matrix rows, several accumulation chains (P >= 4096),
    several streams and ragged tiles; DFT batches (no window) forward and inverse, single pass too."""
    import torch
    tina_env(TINA_SYM_FOLD=1)
    rng = np.random.default_rng(1640 + P + M)
    case = ti.pfb_case(P, M, F, real=False, streams=S, seed=1641 + P + F, window=ti.random_taps(rng, P * M))
    got = _run_pfb(tina, case)
    assert tina.last_kernel() == "pfb_symf_kernel"
    for s in range(S):
        ref = oracle.pfb(case.x[s], P, M, case.window)
        assert rel_l2_rows(got[s], ref) <= TOL_FP32
    if M <= 4:
        x = ti.noise_complex(np.random.default_rng(P), 300 * P).reshape(300, P)
        Z = tina.dft(_cuda(x)); xb = tina.dft(Z, inverse=True); torch.cuda.synchronize()
        assert tina.last_kernel() == "pfb_symf_kernel"
        assert rel_l2_rows(Z.cpu().numpy(), oracle.dft(x)) <= TOL_FP32
        assert rel_l2_rows(xb.cpu().numpy(), x.astype(np.complex128)) <= 2 * TOL_FP32
        Zb = tina.dft(_cuda(x), prec=1); torch.cuda.synchronize()
        assert rel_l2_rows(Zb.cpu().numpy(), oracle.dft(x)) <= TOL_BF16


@pytest.mark.parametrize("P,M,S,F,real", [(1024, 16, 4, 2100, False), (2048, 8, 1, 4099, True), (256, 4, 4, 16384, False), (512, 40, 2, 1500, False)])
def test_pfb_repeated_launches_bit_identical(tina, P, M, S, F, real):
    """300 back-to-back launches on the same buffers give bit-identical results (the ring / barrier protocols of the
    fused kernels, the early hand-back of the input slot and the add-reduce order of later accumulation chains are
    deterministic; a race would show up as a differing launch)."""
    import torch
    n = (F + M - 1) * P
    g = torch.Generator(device="cuda").manual_seed(P + M)
    x = torch.randn(S, n, device="cuda", generator=g) if real else torch.view_as_complex(torch.randn(S, n, 2, device="cuda", generator=g))
    w = torch.randn(M, P, device="cuda", generator=g)
    out = tina.pfb(x, P, M, w); torch.cuda.synchronize()
    ref = out.clone()
    for it in range(300):
        out = tina.pfb(x, P, M, w, out=out)
        if it % 50 == 49:
            torch.cuda.synchronize()
            assert torch.equal(torch.view_as_real(out), torch.view_as_real(ref)), it


@pytest.mark.parametrize("C,L,K,per_channel", [(64, 128 * 1024, 64, False), (70, 128 * 130, 33, True), (3, 128 * 2049, 193, False)])
def test_fir_repeated_launches_bit_identical(tina, C, L, K, per_channel):
    """300 back-to-back launches of fir_umma_kernel on the same buffers give bit-identical results: its operand slots in
    tensor memory (tcgen05.st by the producers, read by tcgen05.mma), the two producer groups on alternate chunks, the
    three accumulator stages and the per-channel rebuild of the resident band matrix are deterministic; a race would
    show up as a differing launch."""
    import torch
    g = torch.Generator(device="cuda").manual_seed(C + K)
    x = torch.randn(C, L, device="cuda", generator=g)
    a = torch.randn((C, K) if per_channel else (K,), device="cuda", generator=g)
    run = tina.fir_multi if per_channel else tina.fir
    out = run(x, a); torch.cuda.synchronize()
    assert tina.last_kernel().startswith("fir_umma_kernel")
    ref = out.clone()
    for it in range(300):
        out = run(x, a, out=out)
        if it % 50 == 49:
            torch.cuda.synchronize()
            assert torch.equal(out, ref), it


def test_pfb_complex_multichain_batched(tina, oracle):
    """Complex kind, K = 4096: four accumulation chains (TMA add-reduce epilogue), 8 column passes,
    ragged last tile, 2 streams."""
    P, M, F, S = 2048, 2, 300, 2
    case = ti.pfb_case(P, M, F, streams=S, seed=660)
    got = _run_pfb(tina, case)
    for s in range(S):
        assert rel_l2_rows(got[s], oracle.pfb(case.x[s], P, M, case.window)) <= TOL_FP32


def test_pfb_shared_fir_clusters(tina, oracle, tina_env):
    """Opt-in SHARE mode (TINA_SHARE=1): clusters of four CTAs compute the subfilter stage once per two
    column passes and exchange the A tiles with bulk shared-memory-to-shared-memory copies."""
    tina_env(TINA_SHARE=1)
    for (P, M, F, real, S) in [(1024, 16, 300, False, 2), (2048, 4, 259, True, 1), (512, 8, 700, False, 1)]:
        case = ti.pfb_case(P, M, F, real=real, streams=S, seed=670 + P)
        got = _run_pfb(tina, case)
        for s in range(S):
            assert rel_l2_rows(got[s], oracle.pfb(case.x[s], P, M, case.window)) <= TOL_FP32


def test_pfb_m1_rect_is_blocked_dft(tina, oracle):
    import torch
    P, F = 128, 256
    case = ti.pfb_case(P, 1, F, seed=700, window=np.ones(P, np.float32))
    got = _run_pfb(tina, case)[0]
    blocks = _cuda(case.x[0].reshape(F, P))
    Z = tina.dft(blocks); torch.cuda.synchronize()
    assert np.array_equal(got, Z.cpu().numpy())
    assert rel_l2_rows(got, oracle.dft(case.x[0].reshape(F, P))) <= TOL_FP32


def test_config1_pfb_full(tina, oracle):
    case = ti.config1()
    got = _run_pfb(tina, case)
    ref = oracle.pfb(case.x[0], case.P, case.M, case.window)
    assert got.shape == (1, 4096, 16)
    assert rel_l2_rows(got[0], ref) <= TOL_FP32


def test_config4_full_size_sampled(tina, oracle):
    """c4 at full size, in the launch configuration bench.py times (one tina_pfb_batched call over the
    8 streams): first 16, last 16 and 96 seeded frames of every stream against the oracle; tone bins
    dominate (P9); error over the non-tone bins reported against the looser bound of SURVEY 8(c)."""
    case = ti.config4()
    got = _run_pfb(tina, case)
    assert got.shape == (8, 8192, 1024)
    worst, worst_nt = 0.0, 0.0
    for s in range(8):
        fr = ti.sample_frames(8192, 96, ti.SEED_BASE + 40 + s)
        ref = oracle.pfb(case.x[s], 1024, 16, case.window, frames=fr)
        g = got[s][fr]
        worst = max(worst, rel_l2_rows(g, ref))
        mask = np.ones(1024, bool); mask[case.tone_bins[s]] = False
        worst_nt = max(worst_nt, rel_l2_rows(g[:, mask], ref[:, mask]))
        top3 = np.argsort(np.abs(ref).mean(axis=0))[-3:]
        assert set(top3.tolist()) == set(case.tone_bins[s].tolist())
    assert worst <= TOL_FP32
    assert worst_nt <= 1.3e-4          # 1e-5 of the frame norm, which the tones inflate ~12x


@pytest.mark.parametrize("prec,tol", [(0, TOL_FP32), (1, TOL_BF16)])
def test_config5_full_size_sampled(tina, oracle, prec, tol):
    """c5 at full size (2^27 real samples, P=4096, M=8): fp32-accurate and single-pass bf16 runs, first 16,
    last 16 and 64 seeded frames against the oracle; Im X[0] = Im X[P/2] = 0."""
    case = ti.config5()
    got = _run_pfb(tina, case, prec=prec)[0]
    assert got.shape == (32761, 2049)
    fr = ti.sample_frames(32761, 64, ti.SEED_BASE + 50)
    ref = oracle.pfb(case.x[0], 4096, 8, case.window, frames=fr)
    assert rel_l2_rows(got[fr], ref) <= tol
    assert np.all(got[:, 0].imag == 0) and np.all(got[:, 2048].imag == 0)


@pytest.mark.parametrize("M,F,S", [(16, 130, 1), (4, 7, 2), (8, 257, 1), (1, 64, 1), (16, 1, 1)])
def test_pfb_fft_factorised_stage(tina, oracle, M, F, S):
    """tina_pfb_fft_batched (two-stage 32 x 32 Fourier stage on the tensor cores) gives the same result as
    the oracle's direct O(P^2) DFT, within the fp32 contract; ragged groups of 4 frames, several streams."""
    rng = np.random.default_rng(40 + M)
    case = ti.pfb_case(1024, M, F, streams=S, seed=41 + M + F, window=ti.random_taps(rng, 1024 * M))
    import torch
    out = tina.pfb_fft(_cuda(case.x), 1024, M, _cuda(case.window)); torch.cuda.synchronize()
    got = out.cpu().numpy()
    assert got.shape == (S, F, 1024)
    for s in range(S):
        assert rel_l2_rows(got[s], oracle.pfb(case.x[s], 1024, M, case.window)) <= TOL_FP32
    with pytest.raises(tina.TinaError) as e:
        tina.pfb_fft(_cuda(case.x[:, : (F + M - 1) * 512]), 512, M, _cuda(case.window[: 512 * M]))
    assert e.value.status == 3


@pytest.mark.parametrize("M,F,S", [(8, 130, 1), (4, 7, 2), (6, 33, 1), (1, 16, 1), (8, 1, 1), (8, 4, 3)])
def test_pfb_fft_factorised_stage_real(tina, oracle, M, F, S):
    """Real kind, P = 4096 = 64 x 64 (the config-5 shape): factorised Fourier stage against the oracle's direct DFT;
    ragged groups of 4 frames, M below the unrolled tap count, several streams; Im X[0] = Im X[P/2] = 0."""
    rng = np.random.default_rng(60 + M)
    case = ti.pfb_case(4096, M, F, real=True, streams=S, seed=61 + M + F, window=ti.random_taps(rng, 4096 * M))
    import torch
    out = tina.pfb_fft(_cuda(case.x), 4096, M, _cuda(case.window)); torch.cuda.synchronize()
    got = out.cpu().numpy()
    assert got.shape == (S, F, 2049)
    for s in range(S):
        ref = oracle.pfb(case.x[s], 4096, M, case.window)
        assert rel_l2_rows(got[s], ref) <= TOL_FP32
        assert np.abs(got[s][:, 2048] - ref[:, 2048]).max() <= 1e-5 * np.linalg.norm(ref, axis=1).max()
    assert np.all(got[..., 2048].imag == 0)
    with pytest.raises(tina.TinaError) as e:                 # M > 8 is not covered by the real-kind factorised kernel
        tina.pfb_fft(_cuda(np.zeros((1, 4096 * 12), np.float32)), 4096, 9, _cuda(np.ones(4096 * 9, np.float32)))
    assert e.value.status == 3


def test_pfb_fft_real_warp_specialised_variant(tina, oracle, tina_env):
    """Opt-in warp-specialised real-kind kernel (TINA_CTR_WS=1; slower than the default, kept as a measured experiment):
    same contract, enough frames for the two-group operand ring and both accumulator slots to wrap several times."""
    import torch
    tina_env(TINA_CTR_WS=1)
    for (M, F, S) in [(8, 4 * 148 * 5 + 3, 1), (4, 7, 2), (8, 1, 1), (5, 1300, 2)]:
        rng = np.random.default_rng(160 + M)
        case = ti.pfb_case(4096, M, F, real=True, streams=S, seed=161 + M + F, window=ti.random_taps(rng, 4096 * M))
        out = tina.pfb_fft(_cuda(case.x), 4096, M, _cuda(case.window)); torch.cuda.synchronize()
        got = out.cpu().numpy()
        assert got.shape == (S, F, 2049)
        fr = ti.sample_frames(F, min(F, 48), 77 + F)
        for s in range(S):
            ref = oracle.pfb(case.x[s], 4096, M, case.window, frames=fr)
            assert rel_l2_rows(got[s][fr], ref) <= TOL_FP32
        assert np.all(got[..., 2048].imag == 0)


def test_config5_full_size_factorised_sampled(tina, oracle):
    """c5 at full size through tina_pfb_fft_batched: first / last / seeded frames against the oracle."""
    import torch
    case = ti.config5()
    out = tina.pfb_fft(_cuda(case.x), 4096, 8, _cuda(case.window)); torch.cuda.synchronize()
    got = out.cpu().numpy()[0]
    assert got.shape == (32761, 2049)
    fr = ti.sample_frames(32761, 64, ti.SEED_BASE + 51)
    ref = oracle.pfb(case.x[0], 4096, 8, case.window, frames=fr)
    assert rel_l2_rows(got[fr], ref) <= TOL_FP32
    assert np.all(got[:, 2048].imag == 0)


def test_config4_full_size_factorised_sampled(tina, oracle):
    """c4 at full size through tina_pfb_fft_batched: seeded frames of every stream against the oracle."""
    import torch
    case = ti.config4()
    out = tina.pfb_fft(_cuda(case.x), 1024, 16, _cuda(case.window)); torch.cuda.synchronize()
    got = out.cpu().numpy()
    assert got.shape == (8, 8192, 1024)
    for s in (0, 3, 7):
        fr = ti.sample_frames(8192, 24, ti.SEED_BASE + 60 + s)
        ref = oracle.pfb(case.x[s], 1024, 16, case.window, frames=fr)
        assert rel_l2_rows(got[s][fr], ref) <= TOL_FP32


def test_pfb_fir_only(tina, oracle):
    import torch
    for real in (False, True):
        P, M, F = 64, 16, 100
        rng = np.random.default_rng(800)
        case = ti.pfb_case(P, M, F, real=real, streams=2, seed=801, window=ti.random_taps(rng, P * M))
        y = tina.pfb_fir(_cuda(case.x), P, M, _cuda(case.window)); torch.cuda.synchronize()
        y = y.cpu().numpy()
        for s in range(2):
            _, yref = oracle.pfb(case.x[s], P, M, case.window, return_subfiltered=True)
            assert rel_l2_rows(y[s], yref) <= TOL_FP32


@pytest.mark.parametrize("P,M,F,real,S", [(128, 3, 131, False, 2), (256, 8, 257, True, 1), (96, 5, 40, False, 1), (24, 4, 50, True, 2)])
def test_pfb_fir_only_shapes(tina, oracle, P, M, F, real, S):
    """Subfilter-only output over the register-window kernel (K % 64 == 0, M <= 16) and the generic one."""
    import torch
    rng = np.random.default_rng(810 + P)
    case = ti.pfb_case(P, M, F, real=real, streams=S, seed=811 + P, window=ti.random_taps(rng, P * M))
    y = tina.pfb_fir(_cuda(case.x), P, M, _cuda(case.window)); torch.cuda.synchronize()
    y = y.cpu().numpy()
    assert y.shape == (S, F, P)
    for s in range(S):
        _, yref = oracle.pfb(case.x[s], P, M, case.window, return_subfiltered=True)
        assert rel_l2_rows(y[s], yref) <= TOL_FP32


@pytest.mark.parametrize("P,M,F,real,S", [(64, 4, 300, False, 3), (128, 8, 2500, True, 1), (256, 4, 3000, False, 2),
                                           (16, 4, 1500, False, 1), (10, 2, 77, True, 2), (128, 8, 2501, True, 2),
                                           (6, 3, 1031, True, 3)])
def test_pfb_host_pipeline_matches_device_call(tina, oracle, P, M, F, real, S):
    """tina_pfb_batched_host (host buffers; pieces pipelined over copy / compute / copy streams) returns
    exactly what the device-pointer call returns, and that matches the oracle."""
    import torch
    case = ti.pfb_case(P, M, F, real=real, streams=S, seed=900 + P + F)
    xh = torch.from_numpy(case.x).pin_memory()
    wh = torch.from_numpy(case.window).pin_memory()
    got_h = tina.pfb_host(xh, P, M, wh).numpy()
    if case.x.shape[1] % (4 if real else 2) == 0 or S == 1:
        got_d = _run_pfb(tina, case)
    else:
        # streams that are not 16-byte aligned inside one batch: the device entry point refuses them
        # (ALIGNMENT), the host entry point stages every stream into its own padded slot
        got_d = np.stack([tina.pfb(_cuda(case.x[s]), P, M, _cuda(case.window)).cpu().numpy() for s in range(S)])
    assert np.array_equal(got_h, got_d)
    ref = oracle.pfb(case.x[S - 1], P, M, case.window)
    assert rel_l2_rows(got_h[S - 1], ref) <= TOL_FP32


# ------------------------------------------------------------------ per-channel FIR taps
@pytest.mark.parametrize("C,L,K", [(1, 64, 64), (5, 9000, 7), (64, 40000, 64), (3, 4097 + 15, 16), (7, 300, 300), (2, 70001, 129)])
def test_fir_multi_per_channel_taps(tina, oracle, C, L, K):
    """tina_fir_multi: channel c is filtered with ITS row of asymmetric random taps (Eq. (15) per channel;
    the 'multiple FIR filters' of PAPER.md:233)."""
    import torch
    rng = np.random.default_rng(170 + C + K)
    x = ti.noise_real(rng, C * L).reshape(C, L)
    a = rng.standard_normal((C, K)).astype(np.float32)
    y = tina.fir_multi(_cuda(x), _cuda(a))
    torch.cuda.synchronize()
    ref = oracle.fir_multi(x, a)
    assert y.shape == ref.shape
    assert rel_l2_rows(y.cpu().numpy(), ref) <= TOL_FP32
    # impulse response of every channel = its own tap row, exactly (fp32 FMA with one non-zero term)
    xi = np.zeros((C, 2 * K - 1), np.float32); xi[:, K - 1] = 1
    yi = tina.fir_multi(_cuda(xi), _cuda(a)); torch.cuda.synchronize()
    assert np.array_equal(yi.cpu().numpy(), a)


def test_fir_multi_is_pfb_subfilter_stage(tina, oracle):
    """the subfilter stage of the PFB = P FIR filters, one per branch, taps w[p::P]."""
    import torch
    P, M, F = 96, 5, 300
    rng = np.random.default_rng(181)
    case = ti.pfb_case(P, M, F, real=True, seed=182, window=ti.random_taps(rng, P * M))
    branches = np.ascontiguousarray(case.x[0].reshape(F + M - 1, P).T)
    taps = np.ascontiguousarray(case.window.reshape(M, P).T)
    y = tina.fir_multi(_cuda(branches), _cuda(taps)); torch.cuda.synchronize()
    _, ysub = oracle.pfb(case.x[0], P, M, case.window, return_subfiltered=True)
    assert rel_l2_rows(y.cpu().numpy(), ysub.T) <= TOL_FP32


# ------------------------------------------------------------------ adversarial inputs
def _bin_check(got, ref, k):
    """|error| of bin k against max(|ref_k|, rms bin magnitude of the frame): a wrong DC / Nyquist
    handling is O(1) on this scale, the split-precision error a few 1e-6."""
    rms = np.linalg.norm(ref, axis=1) / np.sqrt(ref.shape[1])
    scale = np.maximum(np.abs(ref[:, k]), rms)
    scale = np.where(scale == 0, 1.0, scale)
    return float((np.abs(got[:, k] - ref[:, k]) / scale).max())


@pytest.mark.parametrize("kind", ti.ADVERSARIAL_KINDS)
@pytest.mark.parametrize("P,M,F,real,route", [(1024, 16, 140, False, "dense"), (1024, 16, 140, False, "fft"),
                                               (4096, 8, 40, True, "dense"), (4096, 8, 40, True, "fft"),
                                               (2048, 4, 70, False, "dense"), (256, 8, 300, False, "dense")])
def test_pfb_adversarial_inputs(tina, oracle, kind, P, M, F, real, route):
    """The bf16 hi/lo split and the truncating tensor-core accumulator are data dependent; N(0,1) inputs do
    not exercise them.  Same 1e-5 per-frame contract on: constant input (every product of the DC column has
    the same sign), DC offset 100 + noise, one tone of amplitude 1e4 over unit noise, inputs scaled by 1e+-20,
    a window with one tap 1e4 times the rest; plus a per-bin check of DC and Nyquist."""
    import torch
    case = ti.adversarial_case(kind, P, M, F, real=real, seed=7000 + P + len(kind))
    x, w = _cuda(case.x), _cuda(case.window)
    out = tina.pfb(x, P, M, w) if route == "dense" else tina.pfb_fft(x, P, M, w)
    torch.cuda.synchronize()
    got = out.cpu().numpy()[0]
    assert np.all(np.isfinite(got.view(np.float32)))
    ref = oracle.pfb(case.x[0], P, M, case.window)
    assert rel_l2_rows(got, ref) <= TOL_FP32
    assert _bin_check(got, ref, 0) <= 5e-5
    assert _bin_check(got, ref, P // 2) <= 5e-5
    if real:
        assert np.all(got[:, 0].imag == 0) and np.all(got[:, P // 2].imag == 0)


@pytest.mark.parametrize("kind", ["constant", "dc_offset", "scale_up", "scale_down"])
def test_dft_adversarial_inputs(tina, oracle, kind):
    """Standalone DFT / IDFT on the same adversarial data (N = 256 and 2048: one and two accumulation chains)."""
    import torch
    for N, B in ((256, 300), (2048, 40)):
        case = ti.adversarial_case(kind, N, 1, B, seed=7100 + N)
        x = case.x[0].reshape(B, N)
        Z = tina.dft(_cuda(x)); Xi = tina.dft(_cuda(x), inverse=True)
        torch.cuda.synchronize()
        assert rel_l2_rows(Z.cpu().numpy(), oracle.dft(x)) <= TOL_FP32
        assert rel_l2_rows(Xi.cpu().numpy(), oracle.dft(x, inverse=True)) <= TOL_FP32


# ------------------------------------------------------------------ threads / devices
def test_two_host_threads_concurrent_calls(tina, oracle):
    """Two host threads call the library concurrently on their own streams (plan cache, per-device state and
    options are mutex-guarded; everything else is re-entrant): both get correct results."""
    import threading
    import torch
    cases = [ti.pfb_case(256, 8, 700, seed=8100), ti.pfb_case(512, 4, 300, real=True, seed=8101)]
    refs = [oracle.pfb(c.x[0], c.P, c.M, c.window) for c in cases]
    tina.clear_plan_cache()
    outs, errs = [None, None], []

    def work(i):
        try:
            torch.cuda.set_device(0)
            st = torch.cuda.Stream()
            c = cases[i]
            with torch.cuda.stream(st):
                x, w = _cuda(c.x), _cuda(c.window)
                for _ in range(20):
                    o = tina.pfb(x, c.P, c.M, w, stream=st)
                st.synchronize()
            outs[i] = o.cpu().numpy()[0]
        except Exception as e:      # noqa: BLE001
            errs.append(e)

    th = [threading.Thread(target=work, args=(i,)) for i in range(2)]
    [t.start() for t in th]; [t.join() for t in th]
    assert not errs, errs
    for i in range(2):
        assert rel_l2_rows(outs[i], refs[i]) <= TOL_FP32


def test_second_device_in_one_process(tina, oracle):
    """State is kept per CUDA device: the same process can use a second GPU (skipped on one-GPU boxes)."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("one CUDA device")
    case = ti.pfb_case(1024, 16, 300, seed=8200)
    ref = oracle.pfb(case.x[0], 1024, 16, case.window)
    for dev in (0, 1):
        with torch.cuda.device(dev):
            x = torch.from_numpy(case.x).cuda(dev); w = torch.from_numpy(case.window).cuda(dev)
            out = tina.pfb(x, 1024, 16, w); torch.cuda.synchronize(dev)
            assert rel_l2_rows(out.cpu().numpy()[0], ref) <= TOL_FP32
            y = tina.fir(torch.ones((2, 4096), device=f"cuda:{dev}"), torch.ones(8, device=f"cuda:{dev}"))
            torch.cuda.synchronize(dev)
            assert np.allclose(y.cpu().numpy(), 8.0)


def test_out_shape_is_checked(tina):
    """A caller-supplied out= of the wrong shape is refused before any kernel runs."""
    import torch
    x = torch.zeros((2, 64 * 10), dtype=torch.complex64, device="cuda")
    w = torch.ones(64 * 4, dtype=torch.float32, device="cuda")
    with pytest.raises(ValueError):
        tina.pfb(x, 64, 4, w, out=torch.empty((2, 6, 64), dtype=torch.complex64, device="cuda"))
    with pytest.raises(ValueError):
        tina.fir(torch.zeros((2, 100), device="cuda"), torch.ones(5, device="cuda"), out=torch.empty((2, 90), device="cuda"))
    with pytest.raises(ValueError):
        tina.dft(torch.zeros((4, 32), dtype=torch.complex64, device="cuda"), out=torch.empty((4, 16), dtype=torch.complex64, device="cuda"))


def test_error_paths(tina):
    import torch
    x = torch.zeros(64, dtype=torch.complex64, device="cuda")
    w = torch.ones(64, dtype=torch.float32, device="cuda")
    with pytest.raises(tina.TinaError) as e:
        tina.pfb(x[:48], 16, 4, w)               # 3 blocks, M=4 -> F=0: too short
    assert e.value.status == 2
    with pytest.raises(tina.TinaError) as e:
        tina.pfb(torch.zeros(10, dtype=torch.float32, device="cuda"), 5, 1,
                 torch.ones(5, dtype=torch.float32, device="cuda"))       # odd P, real kind
    assert e.value.status == 2
    with pytest.raises(tina.TinaError) as e:
        tina.dft(torch.zeros((1, 16384), dtype=torch.complex64, device="cuda"))
    assert e.value.status == 3


# ---------------------------------------------------------------- section 3 arithmetic blocks
@pytest.mark.parametrize("n", [0, 1, 5, 1023, 4096, (1 << 20) + 3])
def test_arith_mul_add(tina, oracle, n):
    """Eq. (6) / (10): one float32 rounding per element (the oracle's float64 value rounded to float32 is the exact
    expected result, so the comparison is bit-exact); unaligned views take the scalar path; in-place is allowed."""
    import torch
    rng = np.random.default_rng(900 + n % 97)
    a = rng.standard_normal(n + 1).astype(np.float32)
    b = rng.standard_normal(n + 1).astype(np.float32)
    for off in (0, 1):                                       # off = 1: 4-byte-aligned views
        ad, bd = _cuda(a)[off:off + n], _cuda(b)[off:off + n]
        ah, bh = a[off:off + n], b[off:off + n]
        got_m = tina.mul(ad, bd); got_a = tina.add(ad, bd); torch.cuda.synchronize()
        assert np.array_equal(got_m.cpu().numpy(), oracle.mul(ah, bh).astype(np.float32))
        assert np.array_equal(got_a.cpu().numpy(), oracle.add(ah, bh).astype(np.float32))
    if n:
        ad = _cuda(a[:n].copy())
        tina.mul(ad, _cuda(b[:n].copy()), out=ad); torch.cuda.synchronize()
        assert np.array_equal(ad.cpu().numpy(), oracle.mul(a[:n], b[:n]).astype(np.float32))


@pytest.mark.parametrize("rows,n", [(1, 0), (1, 1), (3, 1000), (1, 4096 * 37 + 11), (257, 513), (2, 1 << 22), (4096, 64)])
def test_arith_sum(tina, oracle, rows, n):
    """Eq. (11): |got - ref| <= 1e-6 sum|x| + one float32 rounding of the result."""
    import torch
    rng = np.random.default_rng(910 + rows)
    x = (rng.standard_normal((rows, n)) + 0.25).astype(np.float32)
    got = tina.summation(_cuda(x)); torch.cuda.synchronize()
    ref = oracle.summation(x)
    tol = 1e-6 * np.abs(x).sum(axis=1, dtype=np.float64) + 6e-8 * np.abs(ref) + 1e-30
    assert np.all(np.abs(got.cpu().numpy().astype(np.float64) - ref) <= tol)
    if n:
        one = tina.summation(_cuda(x[0])); torch.cuda.synchronize()
        assert abs(float(one) - ref[0]) <= tol[0]


@pytest.mark.parametrize("M,L,N", [(1, 1, 1), (2, 3, 2), (128, 16, 128), (129, 17, 131), (300, 1000, 70), (64, 4096, 256),
                                   (5, 0, 7), (1000, 64, 1000)])
def test_arith_matmul(tina, oracle, M, L, N):
    """Eq. (7) against the float64 triple loop: |Z - Zref|(m, n) <= 1e-5 |X(m, :)| |Y(:, n)| (fp32 FMA chains of length L:
    the bound is L eps / 2 in the worst case, sqrt(L) eps typically); ragged tiles; L = 0 gives zeros."""
    import torch
    rng = np.random.default_rng(920 + M + N)
    X = rng.standard_normal((M, L)).astype(np.float32)
    Y = rng.standard_normal((L, N)).astype(np.float32)
    got = tina.matmul(_cuda(X), _cuda(Y)); torch.cuda.synchronize()
    ref = oracle.matmul(X, Y)
    bound = 1e-5 * np.outer(np.linalg.norm(X.astype(np.float64), axis=1), np.linalg.norm(Y.astype(np.float64), axis=0)) + 1e-30
    assert got.shape == (M, N)
    assert np.all(np.abs(got.cpu().numpy().astype(np.float64) - ref) <= bound)
    if (M, L, N) == (2, 3, 2):                               # the hand-worked example of the oracle pin
        Z = tina.matmul(_cuda(np.array([[1, 2, 3], [4, 5, 6]], np.float32)), _cuda(np.array([[7, 8], [9, 10], [11, 12]], np.float32)))
        assert Z.cpu().numpy().tolist() == [[58.0, 64.0], [139.0, 154.0]]


def test_arith_error_paths(tina):
    import torch
    L = tina.lib()
    x = torch.zeros(16, device="cuda")
    assert L.tina_mul(x.data_ptr(), x.data_ptr(), x.data_ptr(), -1, None) == 2
    assert L.tina_add(None, x.data_ptr(), x.data_ptr(), 4, None) == 1
    assert L.tina_sum(x.data_ptr(), -1, 4, x.data_ptr(), None) == 2
    assert L.tina_matmul(x.data_ptr(), x.data_ptr(), x.data_ptr(), 2, 2, 2, None) == 2      # aliasing
    assert L.tina_matmul(None, x.data_ptr(), x.data_ptr(), 2, 2, 2, None) == 1
