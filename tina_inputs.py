"""Seeded synthetic inputs for the five BASELINE.json configs (and small test shapes).

This module serves BOTH the oracle-side tests and the CUDA-side tests/bench, and
therefore holds none of the method's arithmetic: no FIR, no DFT, no PFB -- only
random draws (numpy PCG64 ``default_rng(seed)``, ``standard_normal(float32)``)
and the closed-form filter *coefficients*, which are inputs to both sides
(SURVEY.md section 8(c) readings R9, R10).

The paper measures on "32 bit floating point input data generated randomly"
(PAPER.md:214); no public dataset is involved.  The shapes follow BASELINE.json
``configs`` (radio-astronomy PFB shapes); these synthetic inputs stand in for
the paper's random data.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

SEED_BASE = 24081600  # paper id 2408.16551 -> 240816, + config index


def noise_real(rng: np.random.Generator, n: int) -> np.ndarray:
    return rng.standard_normal(n, dtype=np.float32)


def noise_complex(rng: np.random.Generator, n: int) -> np.ndarray:
    """iid N(0,1) real and imaginary parts: real array drawn first, then imaginary."""
    re = rng.standard_normal(n, dtype=np.float32)
    im = rng.standard_normal(n, dtype=np.float32)
    out = np.empty(n, dtype=np.complex64)
    out.real = re
    out.imag = im
    return out


def pfb_window(P: int, M: int) -> np.ndarray:
    """Prototype filter of length P*M: sinc (first null at +-P samples) x symmetric Hann.

    w[j] = sinc((j - (PM-1)/2) / P) * (0.5 - 0.5 cos(2 pi j / (PM-1))), float64 -> float32,
    no gain normalisation (reading R9).  M*P == 1 degenerates to [1].
    """
    n = P * M
    if n == 1:
        return np.ones(1, dtype=np.float32)
    j = np.arange(n, dtype=np.float64)
    w = np.sinc((j - (n - 1) / 2.0) / P) * (0.5 - 0.5 * np.cos(2.0 * np.pi * j / (n - 1)))
    return w.astype(np.float32)


def lowpass_taps(K: int = 64, fc: float = 0.25) -> np.ndarray:
    """K-tap windowed-sinc lowpass, cutoff fc cycles/sample, Hamming, unit DC gain (R10)."""
    k = np.arange(K, dtype=np.float64)
    a = 2.0 * fc * np.sinc(2.0 * fc * (k - (K - 1) / 2.0))
    a *= 0.54 - 0.46 * np.cos(2.0 * np.pi * k / (K - 1))
    a /= a.sum()
    return a.astype(np.float32)


def random_taps(rng: np.random.Generator, K: int) -> np.ndarray:
    """Asymmetric random taps (pins the convolution direction, reading R1)."""
    return rng.standard_normal(K, dtype=np.float32)


@dataclass
class PfbCase:
    name: str
    x: np.ndarray          # [S, n_samples] complex64 or float32
    window: np.ndarray     # [P*M] float32
    P: int
    M: int
    real: bool
    n_frames: int
    tone_bins: np.ndarray | None = None   # [S, 3] for config 4

    @property
    def n_streams(self) -> int:
        return self.x.shape[0]


def pfb_case(P: int, M: int, n_frames: int, real: bool = False, streams: int = 1,
             seed: int = 0, tones: int = 0, tone_amp: float = 10.0,
             name: str = "custom", window: np.ndarray | None = None) -> PfbCase:
    """S streams of (n_frames + M - 1) * P samples, iid N(0,1) (+ optional bin-centred tones).

    Tones (config 4): after ALL noise draws, per stream ``tones`` bins drawn without
    replacement from [0,P) and phases uniform [0, 2 pi); each adds
    tone_amp * exp(2 pi i k n / P + i phi) to the complex stream.
    """
    rng = np.random.default_rng(seed)
    n = (n_frames + M - 1) * P
    if real:
        x = np.stack([noise_real(rng, n) for _ in range(streams)])
    else:
        x = np.stack([noise_complex(rng, n) for _ in range(streams)])
    bins = None
    if tones:
        if real:
            raise ValueError("tones are defined for the complex kind only")
        bins = np.empty((streams, tones), dtype=np.int64)
        # phase of the tone depends on n mod P only (bin-centred): build one period.
        p = np.arange(P, dtype=np.float64)
        for s in range(streams):
            bins[s] = rng.choice(P, size=tones, replace=False)
            phis = rng.uniform(0.0, 2.0 * np.pi, size=tones)
            period = np.zeros(P, dtype=np.complex128)
            for k, phi in zip(bins[s], phis):
                period += tone_amp * np.exp(1j * (2.0 * np.pi * ((k * p) % P) / P + phi))
            period = period.astype(np.complex64)
            x[s] = (x[s].reshape(-1, P) + period[None, :]).reshape(-1)
    w = pfb_window(P, M) if window is None else np.asarray(window, dtype=np.float32)
    return PfbCase(name, x, w, P, M, real, n_frames, bins)


ADVERSARIAL_KINDS = ("constant", "dc_offset", "big_tone", "scale_up", "scale_down", "big_tap")


def adversarial_case(kind: str, P: int, M: int, n_frames: int, real: bool = False, streams: int = 1,
                     seed: int = 0) -> PfbCase:
    """Inputs chosen to stress data-dependent mechanisms of an implementation (operand splitting,
    accumulator rounding) -- still only draws and closed-form signals, no filtering or transforms:
      constant    x = 1 (real) or 1 + 0.5i (complex): every product has the same sign
      dc_offset   100 + N(0,1)
      big_tone    one bin-centred tone / cosine of amplitude 1e4 over unit noise
      scale_up    N(0,1) * 1e20          scale_down  N(0,1) * 1e-20
      big_tap     random window with one tap 1e4 times the rest (data N(0,1))
    The window is random and asymmetric (as in the small parity shapes) except where stated."""
    if kind not in ADVERSARIAL_KINDS:
        raise ValueError(kind)
    rng = np.random.default_rng(seed)
    case = pfb_case(P, M, n_frames, real=real, streams=streams, seed=seed + 1,
                    window=random_taps(rng, P * M))
    x = case.x
    if kind == "constant":
        x[...] = 1.0 if real else np.complex64(1.0 + 0.5j)
    elif kind == "dc_offset":
        x += np.float32(100.0)
    elif kind == "big_tone":
        k0 = int(rng.integers(1, P // 2))
        n = np.arange(P, dtype=np.float64)
        ph = 2.0 * np.pi * ((k0 * n) % P) / P + 0.3
        period = 1e4 * (np.cos(ph) if real else np.exp(1j * ph))
        period = period.astype(x.dtype)
        for s in range(streams):
            x[s] = (x[s].reshape(-1, P) + period[None, :]).reshape(-1)
    elif kind == "scale_up":
        x *= np.float32(1e20)
    elif kind == "scale_down":
        x *= np.float32(1e-20)
    elif kind == "big_tap":
        j = int(rng.integers(0, P * M))
        case.window[j] *= np.float32(1e4)
    case.name = f"adv_{kind}"
    return case


# ---- the five BASELINE.json configs -------------------------------------------------

def config1() -> PfbCase:
    """c1: PFB complex, P=16, M=4, 4096 spectra (65,584 samples)."""
    return pfb_case(16, 4, 4096, seed=SEED_BASE + 1, name="c1_pfb_P16_M4")


def config2(B: int = 65536, N: int = 256):
    """c2: DFT batch B x N complex64 iid N(0,1)."""
    rng = np.random.default_rng(SEED_BASE + 2)
    return noise_complex(rng, B * N).reshape(B, N)


def config3(C: int = 64, L: int = 1 << 20, K: int = 64):
    """c3: FIR, C channels x L float32, K-tap Hamming lowpass; also asymmetric random taps."""
    rng = np.random.default_rng(SEED_BASE + 3)
    x = noise_real(rng, C * L).reshape(C, L)
    taps = lowpass_taps(K, 0.25)
    taps_asym = random_taps(np.random.default_rng(SEED_BASE + 3 + 1000), K)
    return x, taps, taps_asym


def config4(streams: int = 8, n_frames: int = 8192) -> PfbCase:
    """c4 (headline): 8 streams x 8192 spectra x P=1024, M=16, noise + 3 tones of amplitude 10."""
    return pfb_case(1024, 16, n_frames, streams=streams, seed=SEED_BASE + 4, tones=3,
                    name="c4_pfb_P1024_M16")


def config5(n_samples: int = 1 << 27) -> PfbCase:
    """c5: one real stream of 2^27 samples, P=4096, M=8, half spectrum."""
    P, M = 4096, 8
    n_frames = n_samples // P - M + 1
    return pfb_case(P, M, n_frames, real=True, seed=SEED_BASE + 5, name="c5_pfb_real_P4096_M8")


def sample_frames(n_frames: int, n_random: int, seed: int, edge: int = 16) -> np.ndarray:
    """First ``edge``, last ``edge`` and ``n_random`` seeded frames without replacement (sorted)."""
    if n_frames <= 2 * edge + n_random:
        return np.arange(n_frames, dtype=np.int64)
    rng = np.random.default_rng(seed)
    mid = rng.choice(np.arange(edge, n_frames - edge), size=n_random, replace=False)
    return np.sort(np.concatenate([np.arange(edge), mid, np.arange(n_frames - edge, n_frames)])).astype(np.int64)
