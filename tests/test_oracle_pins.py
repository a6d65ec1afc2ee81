"""Pins for the float64 oracle (oracle/tina_oracle.c) -- CPU only.

None of these re-type the oracle's formula: each checks the oracle against a
value the paper prints, a closed form, an invariant, a library routine it must
reduce to, or a brute-force single-expression evaluation on tiny inputs.
Pin numbers P1..P12 follow SURVEY.md section 8(c) / DESIGN.md.
"""
import cmath
import math
import os

import numpy as np
import pytest

import tina_inputs as ti

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
TOL = 1e-12


def _rows(path):
    with open(path) as fh:
        return [[float(t) for t in ln.split()] for ln in fh if ln.strip() and not ln.startswith("#")]


# ---------------------------------------------------------------- FIR / unfold
def test_P2_unfold_paper_example(oracle):
    """X=[1,2,3,4], window 2 -> [[1,2],[2,3],[3,4]], shape (I-J+1) x J."""
    rows = _rows(os.path.join(GOLDEN, "unfold_example.txt"))
    x, J, Y = np.array(rows[0], np.float32), int(rows[1][0]), np.array(rows[2:])
    got = oracle.unfold(x, J)
    assert got.shape == (len(x) - J + 1, J) == Y.shape
    assert np.array_equal(got, Y)


def test_P1_fir_impulse_response_is_taps_in_order(oracle):
    """Eq. (15): x = delta[n-(K-1)] -> y = a[0..K-1] (asymmetric taps; pins R1-R3)."""
    rng = np.random.default_rng(1)
    for K in (1, 2, 5, 64):
        a = ti.random_taps(rng, K)
        x = np.zeros(2 * K - 1, np.float32)
        x[K - 1] = 1.0
        y = oracle.fir(x, a)
        assert y.shape == (K,)
        assert np.array_equal(y, a.astype(np.float64))


def test_P2_fir_is_unfold_dot_flipped_taps_and_numpy_convolve(oracle):
    """valid length L-K+1; y = unfold(x,K) . a[::-1]; equals numpy.convolve(x,a,'valid')."""
    rng = np.random.default_rng(2)
    x = ti.noise_real(rng, 3 * 257).reshape(3, 257)
    a = ti.random_taps(rng, 17)
    y = oracle.fir(x, a)
    assert y.shape == (3, 257 - 17 + 1)
    for c in range(3):
        U = oracle.unfold(x[c], 17)
        assert np.allclose(y[c], U @ a[::-1].astype(np.float64), rtol=0, atol=1e-12)
        assert np.allclose(y[c], np.convolve(x[c].astype(np.float64), a.astype(np.float64), "valid"),
                           rtol=0, atol=1e-12)


def test_fir_single_tap_and_shared_taps(oracle):
    """K=1 is a scale; all channels share one tap vector (R13)."""
    rng = np.random.default_rng(3)
    x = ti.noise_real(rng, 40).reshape(4, 10)
    y = oracle.fir(x, np.array([2.5], np.float32))
    assert np.array_equal(y, 2.5 * x.astype(np.float64))
    a = ti.random_taps(rng, 3)
    y = oracle.fir(x, a)
    for c in range(4):
        assert np.array_equal(y[c], oracle.fir(x[c], a))


def test_fir_multi_per_channel_taps(oracle):
    """Per-channel taps (PAPER.md:233 'multiple FIR filters'; Eq. (15) per channel).  Pins that do
    not re-type the formula: (i) channel c's impulse response is ITS tap row, in order; (ii) each
    channel equals numpy.convolve with its own taps; (iii) rows of taps are not mixed up: a channel
    whose taps are all zero gives zeros; (iv) the PFB subfilter stage (Eq. (20)) is ONE fir_multi
    call over the P branches with taps w[p::P] (the statement of PAPER.md:233)."""
    rng = np.random.default_rng(31)
    C, K, L = 5, 7, 90
    a = rng.standard_normal((C, K)).astype(np.float32)
    a[3] = 0.0
    x = np.zeros((C, 2 * K - 1), np.float32)
    x[:, K - 1] = 1.0
    assert np.array_equal(oracle.fir_multi(x, a), a.astype(np.float64))
    x = ti.noise_real(rng, C * L).reshape(C, L)
    y = oracle.fir_multi(x, a)
    assert y.shape == (C, L - K + 1)
    for c in range(C):
        assert np.allclose(y[c], np.convolve(x[c].astype(np.float64), a[c].astype(np.float64), "valid"),
                           rtol=0, atol=1e-12)
    assert np.array_equal(y[3], np.zeros(L - K + 1))
    P, M, F = 8, 3, 11
    c4 = _small_case(P, M, F, real=True, seed=12)
    _, ysub = oracle.pfb(c4.x[0], P, M, c4.window, return_subfiltered=True)
    branches = np.ascontiguousarray(c4.x[0][: (F + M - 1) * P].reshape(F + M - 1, P).T)   # [P][NB]
    taps = np.ascontiguousarray(c4.window.reshape(M, P).T)                                # [P][M] = w[p::P]
    assert np.allclose(oracle.fir_multi(branches, taps).T, ysub, rtol=0, atol=1e-12)


# ---------------------------------------------------------------- DFT / IDFT
def test_dft4_textbook_golden(oracle):
    rows = _rows(os.path.join(GOLDEN, "dft4_textbook.txt"))
    x = np.array(rows[0], np.float32).astype(np.complex64)
    Z = np.array(rows[1]) + 1j * np.array(rows[2])
    assert np.allclose(oracle.dft(x), Z, rtol=0, atol=1e-14)


@pytest.mark.parametrize("N", [1, 2, 3, 8, 12, 256])
def test_P3_dft_of_impulses(oracle, N):
    """DFT(delta) = all-ones (unnormalised forward); DFT(delta[n-1])[k] = exp(-2 pi i k/N) (sign)."""
    d0 = np.zeros(N, np.complex64); d0[0] = 1
    assert np.array_equal(oracle.dft(d0), np.ones(N, np.complex128))
    if N > 1:
        d1 = np.zeros(N, np.complex64); d1[1] = 1
        want = np.array([cmath.exp(-2j * math.pi * k / N) for k in range(N)])
        assert np.allclose(oracle.dft(d1), want, rtol=0, atol=1e-15)


@pytest.mark.parametrize("N,k0", [(8, 3), (64, 63), (256, 17), (12, 5)])
def test_P4_bin_aligned_tone_single_bin(oracle, N, k0):
    """x[n] = exp(+2 pi i k0 n/N) -> Z[k0] = N, others 0."""
    n = np.arange(N)
    x = np.exp(2j * np.pi * ((k0 * n) % N) / N)          # complex128 input path
    Z = oracle.dft(x)
    want = np.zeros(N, np.complex128); want[k0] = N
    assert np.allclose(Z, want, rtol=0, atol=1e-12 * N)


def test_P5_roundtrip_parseval_and_numpy_fft(oracle):
    rng = np.random.default_rng(5)
    for N in (2, 7, 16, 256):
        x = ti.noise_complex(rng, 3 * N).reshape(3, N)
        Z = oracle.dft(x)
        assert np.allclose(oracle.dft(Z, inverse=True), x.astype(np.complex128), rtol=0, atol=1e-12)
        assert np.allclose((np.abs(Z) ** 2).sum(1), N * (np.abs(x.astype(np.complex128)) ** 2).sum(1),
                           rtol=1e-13)
        assert np.allclose(Z, np.fft.fft(x.astype(np.complex128), axis=1), rtol=0, atol=1e-11)
        assert np.allclose(oracle.dft(x, inverse=True), np.fft.ifft(x.astype(np.complex128), axis=1),
                           rtol=0, atol=1e-13)


# ---------------------------------------------------------------- PFB
def _small_case(P, M, F, real=False, seed=0):
    rng = np.random.default_rng(seed)
    w = ti.random_taps(rng, P * M)                      # random ASYMMETRIC window
    return ti.pfb_case(P, M, F, real=real, seed=seed + 1, window=w)


def test_pfb_num_frames(oracle):
    assert oracle.pfb_num_frames(65584, 16, 4) == 4096          # config 1
    assert oracle.pfb_num_frames((8192 + 15) * 1024, 1024, 16) == 8192   # config 4
    assert oracle.pfb_num_frames(1 << 27, 4096, 8) == 32761    # config 5
    assert oracle.pfb_num_frames(16 * 7 + 5, 16, 4) == 4        # tail ignored (R8)
    assert oracle.pfb_num_frames(16 * 3, 16, 4) == 0


@pytest.mark.parametrize("real", [False, True])
def test_P6_subfilter_stage_is_P_independent_firs(oracle, real):
    """PAPER.md:233 'combining multiple FIR filters as detailed in Section 4.3':
    y[:,p] == FIR(x[p::P], taps = w[p::P]) in valid mode (pins R4, R5, R6)."""
    P, M, F = 8, 3, 11
    c = _small_case(P, M, F, real=real, seed=10)
    x = c.x[0]
    _, y = oracle.pfb(x, P, M, c.window, return_subfiltered=True)
    assert y.shape == (F, P)
    for p in range(P):
        taps = c.window[p::P]
        if real:
            want = oracle.fir(x[p::P], taps)
        else:
            want = oracle.fir(x.real[p::P].copy(), taps) + 1j * oracle.fir(x.imag[p::P].copy(), taps)
        assert np.allclose(y[:, p], want, rtol=0, atol=1e-12)


def test_P7_M1_rect_window_is_blocked_dft(oracle):
    P, F = 16, 9
    c = ti.pfb_case(P, 1, F, seed=20, window=np.ones(P, np.float32))
    X = oracle.pfb(c.x[0], P, 1, c.window)
    blocks = c.x[0].reshape(F, P)
    assert np.allclose(X, oracle.dft(blocks), rtol=0, atol=1e-12)
    assert np.allclose(X, np.fft.fft(blocks.astype(np.complex128), axis=1), rtol=0, atol=1e-11)


def test_P8_weighted_overlap_add_identity(oracle):
    """X[f][k] = bin k*M of the (M*P)-point DFT of w~ (.) x[fP .. fP+MP),
    w~[n] = w[(M-1-n//P) P + n%P]  -- an independent route through one long library FFT."""
    P, M, F = 8, 3, 6
    c = _small_case(P, M, F, seed=30)
    x = c.x[0].astype(np.complex128)
    X = oracle.pfb(c.x[0], P, M, c.window)
    n = np.arange(M * P)
    wt = c.window.astype(np.float64)[(M - 1 - n // P) * P + n % P]
    for f in range(F):
        long_fft = np.fft.fft(wt * x[f * P: f * P + M * P])
        assert np.allclose(X[f], long_fft[::M], rtol=0, atol=1e-11)


def test_P9_pure_tone_closed_form(oracle):
    """x[n] = A exp(2 pi i k0 n/P): every frame identical; X[f][k0] = A sum_j w[j];
    X[f][k] = A sum_p g[p] exp(-2 pi i p (k-k0)/P), g[p] = sum_m w[mP+p]."""
    P, M, F, k0, A = 16, 4, 5, 5, 10.0
    w = ti.pfb_window(P, M)
    n = np.arange((F + M - 1) * P)
    x = (A * np.exp(2j * np.pi * ((k0 * n) % P) / P)).astype(np.complex64)
    X = oracle.pfb(x, P, M, w)
    g = w.astype(np.float64).reshape(M, P).sum(0)
    p = np.arange(P)
    want = np.array([A * (g * np.exp(-2j * np.pi * p * (k - k0) / P)).sum() for k in range(P)])
    for f in range(F):
        assert np.allclose(X[f], want, rtol=0, atol=2e-5)   # x itself was rounded to complex64
    assert abs(X[0, k0] - A * w.astype(np.float64).sum()) < 2e-5


def test_P10_linearity_and_block_delay(oracle):
    P, M, F = 8, 3, 7
    c1, c2 = _small_case(P, M, F, seed=40), _small_case(P, M, F, seed=41)
    w = c1.window
    xa, xb = c1.x[0], c2.x[0]
    Xa, Xb = oracle.pfb(xa, P, M, w), oracle.pfb(xb, P, M, w)
    xs = (2 * xa + xb).astype(np.complex64)             # exact in fp32? not always -> compare via f64 route
    Xs = oracle.pfb(xs, P, M, w)
    # linearity checked against the *rounded* sum's own decomposition error bound
    assert np.allclose(Xs, 2 * Xa + Xb, rtol=0, atol=1e-4)
    # delaying the input by P samples shifts frames by one
    xd = np.concatenate([np.zeros(P, np.complex64), xa])
    Xd = oracle.pfb(xd, P, M, w)
    assert Xd.shape[0] == F + 1
    assert np.array_equal(Xd[1:], Xa)


def test_P11_real_input_half_spectrum(oracle):
    P, M, F = 8, 3, 6
    c = _small_case(P, M, F, real=True, seed=50)
    xr = c.x[0]
    Xh, y = oracle.pfb(xr, P, M, c.window, return_subfiltered=True)
    assert Xh.shape == (F, P // 2 + 1)
    Xc = oracle.pfb(xr.astype(np.complex64), P, M, c.window)
    assert np.allclose(Xh, Xc[:, : P // 2 + 1], rtol=0, atol=1e-13)
    # Hermitian symmetry of the full spectrum
    for k in range(1, P):
        assert np.allclose(Xc[:, k], np.conj(Xc[:, P - k]), rtol=0, atol=1e-12)
    # Nyquist bin = sum_p (-1)^p y[f][p]
    sign = (-1.0) ** np.arange(P)
    assert np.allclose(Xh[:, P // 2].real, (y * sign).sum(1), rtol=0, atol=1e-12)
    assert np.allclose(Xh[:, P // 2].imag, 0, atol=1e-12)


@pytest.mark.parametrize("P", [2, 4, 8])
@pytest.mark.parametrize("M", [1, 2, 3])
@pytest.mark.parametrize("F", [1, 2, 5])
def test_P12_brute_force_single_expression(oracle, P, M, F):
    """Pure-python evaluation of X[f][k] = sum_{n<MP} w~[n] x[fP+n] exp(-2 pi i n k/P)."""
    c = _small_case(P, M, F, seed=60 + P * 100 + M * 10 + F)
    x = [complex(v) for v in c.x[0]]
    w = [float(v) for v in c.window]
    X = oracle.pfb(c.x[0], P, M, c.window)
    assert X.shape == (F, P)
    for f in range(F):
        for k in range(P):
            acc = 0j
            for n in range(M * P):
                wt = w[(M - 1 - n // P) * P + n % P]
                acc += wt * x[f * P + n] * cmath.exp(-2j * math.pi * n * k / P)
            assert abs(acc - X[f, k]) < 1e-11


def test_pfb_frame_subset_matches_full(oracle):
    P, M, F = 8, 4, 40
    c = _small_case(P, M, F, seed=70)
    X = oracle.pfb(c.x[0], P, M, c.window)
    sel = np.array([0, 3, 39, 17], np.int64)
    assert np.array_equal(oracle.pfb(c.x[0], P, M, c.window, frames=sel), X[sel])


def test_config4_tone_bins_dominate(oracle):
    """The c4 recipe at reduced size: 3 tones of amplitude 10 -> |X[k_t]| ~ 10 * sum(w) (P9)."""
    c = ti.pfb_case(64, 4, 8, seed=ti.SEED_BASE + 4, tones=3)
    X = oracle.pfb(c.x[0], 64, 4, c.window)
    sw = float(c.window.astype(np.float64).sum())
    for k in c.tone_bins[0]:
        assert abs(abs(X[2, k]) - 10 * sw) < 0.15 * 10 * sw


# ---------------------------------------------------------------- section 3 arithmetic blocks
def test_arith_mul_add_closed_forms(oracle):
    """Eq. (6) / (10) on values whose products and sums are exact in binary: powers of two and small integers."""
    a = np.array([1, 2, -3, 0.5, 1024, -0.25, 7, 0], np.float32)
    b = np.array([4, -0.5, 3, 8, 2 ** -10, -16, 0, 5], np.float32)
    assert oracle.mul(a, b).tolist() == [4.0, -1.0, -9.0, 4.0, 1.0, 4.0, 0.0, 0.0]
    assert oracle.add(a, b).tolist() == [5.0, 1.5, 0.0, 8.5, 1024 + 2 ** -10, -16.25, 7.0, 5.0]
    rng = np.random.default_rng(5)
    x, y = rng.standard_normal(1000).astype(np.float32), rng.standard_normal(1000).astype(np.float32)
    assert np.array_equal(oracle.add(x, y), oracle.add(y, x))                 # commutative
    assert np.array_equal(oracle.mul(x, np.ones_like(x)), x.astype(np.float64))   # K = 1 is the identity (Eq. (10) step)
    assert oracle.mul(x, y).dtype == np.float64 and oracle.mul(x.reshape(10, 100), y.reshape(10, 100)).shape == (10, 100)


def test_arith_sum_gauss_and_cancellation(oracle):
    """Eq. (11): 1 + 2 + ... + n = n (n + 1) / 2; a sum whose naive float32 accumulation fails; math.fsum."""
    import math
    n = 4096
    assert oracle.summation(np.arange(1, n + 1, dtype=np.float32)) == n * (n + 1) / 2
    x = np.array([1e8, 1.0, -1e8, 1.0] * 100, np.float32)
    assert oracle.summation(x) == 200.0
    rng = np.random.default_rng(6)
    r = rng.standard_normal((3, 5000)).astype(np.float32)
    got = oracle.summation(r)
    for i in range(3):
        assert abs(got[i] - math.fsum(float(v) for v in r[i])) <= 1e-12 * np.abs(r[i]).sum()
    assert oracle.summation(np.zeros((2, 0), np.float32)).tolist() == [0.0, 0.0]


def test_arith_matmul_textbook_and_dft(oracle):
    """Eq. (7): a 2x3 by 3x2 product worked by hand; identity / permutation; (XY)^T = Y^T X^T; and the cross-pin the
    paper itself draws (section 4.1): the DFT is a matrix product with the Fourier matrix, so the real and imaginary
    parts of oracle.dft must equal oracle.matmul against cos / -sin matrices built here with numpy."""
    X = np.array([[1, 2, 3], [4, 5, 6]], np.float32)
    Y = np.array([[7, 8], [9, 10], [11, 12]], np.float32)
    assert oracle.matmul(X, Y).tolist() == [[58.0, 64.0], [139.0, 154.0]]
    rng = np.random.default_rng(7)
    A = rng.standard_normal((5, 7)).astype(np.float32)
    B = rng.standard_normal((7, 4)).astype(np.float32)
    assert np.array_equal(oracle.matmul(A, np.eye(7, dtype=np.float32)), A.astype(np.float64))
    perm = np.eye(7, dtype=np.float32)[:, ::-1]
    assert np.array_equal(oracle.matmul(A, perm), A[:, ::-1].astype(np.float64))
    np.testing.assert_allclose(oracle.matmul(A, B).T, oracle.matmul(B.T.copy(), A.T.copy()), rtol=0, atol=1e-14)
    brute = [[sum(float(A[m, l]) * float(B[l, n]) for l in range(7)) for n in range(4)] for m in range(5)]
    np.testing.assert_allclose(oracle.matmul(A, B), brute, rtol=0, atol=1e-14)
    N = 16
    x = rng.standard_normal((3, N)).astype(np.float32)
    ang = 2 * np.pi * np.outer(np.arange(N), np.arange(N)) / N
    C, S = np.cos(ang).astype(np.float32), (-np.sin(ang)).astype(np.float32)
    Z = oracle.dft(x.astype(np.complex64))
    np.testing.assert_allclose(oracle.matmul(x, C), Z.real, atol=2e-6)      # float32 twiddles: ~N * 6e-8 * |x|
    np.testing.assert_allclose(oracle.matmul(x, S), Z.imag, atol=2e-6)
