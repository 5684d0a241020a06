"""O11 (NEXT-3, second half) — sub-sample alignment of the SNR series by interpolation.

ORACLE / TEST INFRASTRUCTURE (see spiir_oracle.c header): plain float64 numpy, shares no code with
the CUDA path.  The paper aligns the detectors' SNR series at integer samples ("Time offsets of SNRs
from different detectors"); SURVEY.md §8(f) NEXT-3 asks for a fractional-delay
interpolation of z with a 4-tap interpolator.  Reading X7: around every candidate the
window z[k - H .. k + H] of each detector is resampled R times finer with the cubic Lagrange
interpolator through the four neighbouring samples (nodes -1, 0, 1, 2 around the interval that holds
the new point); the coherent search then runs unchanged on those windows with a delay table built at
R times the sampling rate.
"""
import numpy as np


def lagrange4(mu):
    """Weights of the samples at nodes -1, 0, 1, 2 for the point at 0 <= mu < 1: the cubic through the
    four samples, L_m(mu) = prod_{n != m} (mu - n) / (m - n)."""
    nodes = (-1.0, 0.0, 1.0, 2.0)
    w = []
    for m in nodes:
        p = 1.0
        for n in nodes:
            if n != m:
                p *= (mu - n) / (m - n)
        w.append(p)
    return np.array(w)


def upsample_windows(z, ring_len, k_newest, trig_valid, trig_row, trig_det, trig_k, R, H):
    """z complex [D][rows][ring_len] (ring: sample k lives at k mod ring_len, defined for
    max(0, k_newest - ring_len + 1) <= k <= k_newest).  Returns
      out   complex128 [D][n_slots][2 R H + 1]: out[I][s][u] = z_I(row_s, k_s - H + u / R)
      valid int32 [n_slots]: 1 iff the slot is valid and k_s - H - 1 .. k_s + H + 1 lie in the ring
    (slots that are not valid are all zero).  In the windows the candidate sits at sample R H."""
    z = np.asarray(z)
    D = z.shape[0]
    n = len(trig_k)
    R, H = int(R), int(H)
    Lw = 2 * R * H + 1
    out = np.zeros((D, n, Lw), np.complex128)
    valid = np.zeros(n, np.int32)
    k_old = max(0, int(k_newest) - int(ring_len) + 1)
    W = [lagrange4(r / R) for r in range(R)]
    for s in range(n):
        k = int(trig_k[s])
        if not trig_valid[s] or k - H - 1 < k_old or k + H + 1 > k_newest:
            continue
        valid[s] = 1
        row = int(trig_row[s])
        for I in range(D):
            for u in range(Lw):
                q, r = divmod(u, R)
                base = k - H + q
                if r == 0:
                    out[I, s, u] = z[I, row, base % ring_len]
                else:
                    acc = 0.0
                    for m in range(4):
                        acc = acc + W[r][m] * complex(z[I, row, (base - 1 + m) % ring_len])
                    out[I, s, u] = acc
    return out, valid
