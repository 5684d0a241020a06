"""ORACLE (test infrastructure only) — NEXT-4: the front end of the pipeline, PAPER.md:79-87 (Sec. II A) and
PAPER.md:354 (Sec. IV C): FIR down-sampling, frequency-domain whitening (Eq. 1) against a running median PSD of
the immediate past, and amplitude gating with 0.25 s of zero padding on either side.

Plain numpy float64, one step after the other in the paper's order; numpy.fft is the library primitive for the
Fourier transforms.  The paper gives the method in words only; the readings (W1-W6):
  W1  down-sampling by an integer factor R with a causal FIR h of N_FIR taps ("in time-domain using
      a finite impulse response (FIR) filter", :354 N_FIR-D ~ 192): y[m] = sum_j h[j] x[R m + R - 1 - j], x[n<0] = 0.
      The taps are an INPUT (the generator supplies a Kaiser-windowed sinc).
  W2  the stream is processed in hops of H output samples ("segment length ... two seconds");
      block c is the 2H samples [hop c-1 | hop c] (hop -1 = zeros), windowed with the periodic Hann window
      w[n] = sin^2(pi n / 2H), whose half-overlapped copies sum to one ("overlapping 4-second blocks").
  W3  Eq. 1 per block: D = FFT(w d), D_w[k] = D[k] / sqrt(S_n(f_k) f_s / 2), d_w-block = IFFT(D_w); the
      whitened stream is the overlap-add of the blocks, so hop c-1 is complete after block c.  The factor
      f_s / 2 makes noise of one-sided PSD S_n come out with unit variance (E n n* = S_n / 2).
  W4  S_n(f_k) for block c = median over the periodograms of the n_hist most recent PAST blocks (PAPER.md:83:
      "tracking the geometric median PSD from overlapping 4-second blocks of immediate past data spanning 56
      seconds": n_hist = 27 blocks of 4 s at a 2-s hop), divided by the bias of the median of n exponential
      variates b(n) = sum_{i=1}^{n} (-1)^(i+1) / i (odd n; n even uses n - 1 blocks); periodogram of a block
      P[k] = 2 |D[k]|^2 / (f_s sum w^2).  Block 0 has no past: its whitened block is zero.
  W5  gating: a whitened sample with |d_w| > threshold and every sample within `pad` samples of
      one is replaced by zero.
  W6  the front end emits hop c-1 shifted by the gate's look-ahead: call c returns the gated samples
      t in [(c-1) H - pad, c H - pad) (zeros before t = 0): 0.25 s + one hop of latency, as PAPER.md:354 lists.
"""
import numpy as np


def median_bias(n):
    """Bias of the sample median of n (odd) independent exponential variates relative to their mean."""
    n = int(n)
    return float(sum((-1.0) ** (i + 1) / i for i in range(1, n + 1)))


def downsample(x, taps, R):
    """W1.  x float [n_in] (n_in a multiple of R) from the start of the stream -> y [n_in / R]."""
    x = np.asarray(x, dtype=np.float64)
    h = np.asarray(taps, dtype=np.float64)
    n_out = len(x) // R
    y = np.zeros(n_out)
    xp = np.concatenate([np.zeros(len(h)), x])             # x[n < 0] = 0
    hr = h[::-1]
    for m in range(n_out):
        i = R * m + R - 1 + len(h)                          # position of x[R m + R - 1] in xp
        y[m] = np.dot(hr, xp[i - len(h) + 1:i + 1])         # sum_j h[j] x[R m + R - 1 - j]
    return y


def hann_periodic(n):
    return np.sin(np.pi * np.arange(n) / n) ** 2


def whiten_stream(d, H, fs, n_hist, psd_true=None):
    """W2-W4 over a whole stream d [n_hops * H].  Returns (d_w [n_hops * H] complete up to the last hop but one
    — the last hop is only half overlap-added —, S [n_hops][H + 1] the PSD used for each block, P the periodograms).
    With psd_true [H + 1] given, that PSD is used for every block instead of the running median."""
    d = np.asarray(d, dtype=np.float64)
    n_hops = len(d) // H
    N = 2 * H
    w = hann_periodic(N)
    sw2 = float(np.sum(w * w))
    out = np.zeros((n_hops + 1) * H)
    P = np.zeros((n_hops, H + 1))
    S = np.zeros((n_hops, H + 1))
    dp = np.concatenate([np.zeros(H), d])                  # hop -1 = zeros
    for c in range(n_hops):
        blk = dp[c * H:c * H + N] * w
        D = np.fft.rfft(blk)
        P[c] = 2.0 * np.abs(D) ** 2 / (fs * sw2)
        if psd_true is not None:
            S[c] = psd_true
        else:
            n = min(c, n_hist)
            if n % 2 == 0:
                n -= 1
            if n < 1:
                continue                                    # block 0: no past, nothing emitted
            S[c] = np.median(P[c - n:c], axis=0) / median_bias(n)
        Dw = D / np.sqrt(S[c] * fs / 2.0)
        out[c * H:c * H + N] += np.fft.irfft(Dw, N)
    # out is indexed from hop -1: drop it
    return out[H:H + n_hops * H], S, P


def gate_mask(dw, threshold, pad):
    """W5.  True where the sample is zeroed."""
    dw = np.asarray(dw, dtype=np.float64)
    bad = np.abs(dw) > threshold
    m = np.zeros(len(dw), bool)
    for i in np.nonzero(bad)[0]:
        m[max(0, i - pad):i + pad + 1] = True
    return m


def frontend(x_raw, taps, R, H, fs, n_hist, threshold, pad):
    """The whole front end over a stream from its start: x_raw [n_det][n_hops * H * R] -> per call c the H samples
    W6 describes, concatenated: out [n_det][n_hops * H]; also the whitened (ungated) stream for reference."""
    x_raw = np.asarray(x_raw)
    n_det = x_raw.shape[0]
    n_hops = x_raw.shape[1] // (H * R)
    out = np.zeros((n_det, n_hops * H))
    dws = np.zeros((n_det, n_hops * H))
    for I in range(n_det):
        y = downsample(x_raw[I].astype(np.float32), np.asarray(taps, np.float32), R)
        dw, _, _ = whiten_stream(y, H, fs, n_hist)
        dws[I] = dw
        # call c (c = 0 .. n_hops-1) emits t in [(c-1)H - pad, cH - pad).  Gating a sample t needs the whitened stream
        # on [t - pad, t + pad], i.e. up to cH - 1: all of it complete after block c (hop c-1 is closed by block c, and
        # later blocks never touch it), so the mask of the complete part of the stream is the mask every call sees.
        n_done = (n_hops - 1) * H                            # the last hop is only half overlap-added: never emitted
        m = gate_mask(dw[:n_done], threshold, pad)
        for c in range(n_hops):
            t0, t1 = (c - 1) * H - pad, c * H - pad
            for t in range(max(t0, 0), t1):
                out[I, c * H + (t - t0)] = 0.0 if m[t] else dw[t]
    return out, dws
