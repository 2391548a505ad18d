"""CPU oracle for the F-engine -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

PAPER.md:49-52 (Sec. 2, Eq. 1): "For a discrete time signal s[n] of N samples ... the Discrete Fourier Transform is
first applied to obtain the spectra S[k]":

    S[k] = sum_{n=0}^{N-1} s[n] exp(-j (2 pi / N) k n)

with the paper's FFT length N = 256 ("An FFT length of 256 is used across all tests") applied to
consecutive, non-overlapping blocks of each input stream's 8-bit real samples.  The oracle is the
definition written out: one fp64 matrix product with the DFT matrix exp(-2 pi j k n / N); no FFT algorithm, no
scaling (Eq. 1 has none), no windowing.

Readings:
  F1  the samples are real, so S[N-k] = conj(S[k]); the N/2 channels k = 0 .. N/2-1 are kept (the Nyquist bin is
      dropped), which is what the X-engine consumes as its channel axis;
  F2  spectrum a of stream m is computed from samples [a N, (a+1) N) of that stream;
  F3  output order [spectrum a][channel k][stream m] = the X-engine's input layout [T][C][N*P].

Layouts:  s [n_stream, n_spectra * N] int8  ->  S [n_spectra, N/2, n_stream] complex128 (unrounded).
Only tests/, __graft_entry__.smoke() and bench.py's CPU legs may import this module.
"""
import numpy as np

FFT_LEN = 256


def dft_matrix(n_fft=FFT_LEN, n_chan=None):
    """exp(-j 2 pi k n / N) for k < n_chan, n < N (Eq. 1), fp64; the angle is reduced exactly in integers first."""
    n_chan = n_fft // 2 if n_chan is None else n_chan
    kn = (np.arange(n_chan)[:, None] * np.arange(n_fft)[None, :]) % n_fft
    ang = -2.0 * np.pi * kn / n_fft
    return np.cos(ang) + 1j * np.sin(ang)


def fengine(s, n_fft=FFT_LEN):
    s = np.ascontiguousarray(s)
    if s.ndim != 2 or s.dtype != np.int8 or s.shape[1] % n_fft:
        raise ValueError("s must be int8 [n_stream, n_spectra * %d]" % n_fft)
    n_stream, n_total = s.shape
    n_spec = n_total // n_fft
    blocks = s.reshape(n_stream, n_spec, n_fft).astype(np.float64)          # [m][a][n]
    W = dft_matrix(n_fft)                                                   # [k][n]
    S = np.einsum("kn,man->akm", W, blocks)                                 # Eq. 1, per block
    return np.ascontiguousarray(S)


def to_xengine_input(S):
    """Round the spectra to complex fp16 in the X-engine's [T, C, M, 2] (re, im) layout (round to nearest even)."""
    out = np.empty(S.shape + (2,), dtype=np.float16)
    out[..., 0] = S.real.astype(np.float16)
    out[..., 1] = S.imag.astype(np.float16)
    return out


def quantise_ci8(S, scale):
    """Requantised int8 codes of the spectra: clip(rint(S * scale), -127, 127) per component, rint = round half to even,
    in the X-engine's [T, C, M, 2] layout.  Also returns the distance of every scaled component from the nearest
    rounding tie (k + 0.5), so that a comparison can tell a genuine mismatch from a tie decided in lower precision."""
    y = np.stack([S.real, S.imag], axis=-1) * float(scale)
    codes = np.clip(np.rint(y), -127, 127).astype(np.int8)
    tie_dist = np.abs(np.abs(y - np.floor(y)) - 0.5)
    return codes, tie_dist
