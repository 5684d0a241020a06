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


def upsample_windows(z, ring_len, k_newest, trig_valid, trig_row, trig_det, trig_k, R, H,
                     n_slides=0, step=0, slide_mult=None):
    """z complex [D][rows][ring_len] (ring: sample k lives at k mod ring_len, defined for
    max(0, k_newest - ring_len + 1) <= k <= k_newest).  Returns
      out   complex128 [D][n_rows][2 R H + 1]: out[I][w][u] = z_I(row_s, c_I - H + u / R)
      valid int32 [n_rows]: 1 iff the slot is valid and c_I - H - 1 .. c_I + H + 1 lie in the ring for every I
    (rows that are not valid are all zero).  Foreground (n_slides = 0): one row per slot, c_I = k_s.  Time slides
    (O7): row w = s n_slides + (slide - 1), c_I = k_s - slide step slide_mult[I] for I other than the
    trigger detector.  In the windows the candidate sits at sample R H."""
    z = np.asarray(z)
    D = z.shape[0]
    n = len(trig_k)
    R, H = int(R), int(H)
    S1 = max(1, int(n_slides))
    Lw = 2 * R * H + 1
    out = np.zeros((D, n * S1, Lw), np.complex128)
    valid = np.zeros(n * S1, np.int32)
    k_old = max(0, int(k_newest) - int(ring_len) + 1)
    W = [lagrange4(r / R) for r in range(R)]
    for s in range(n):
        for si in range(S1):
            w = s * S1 + si
            T = int(trig_det[s])
            cen = [int(trig_k[s]) - ((si + 1) * int(step) * int(slide_mult[I]) if (n_slides and I != T) else 0)
                   for I in range(D)]
            if not trig_valid[s] or any(c - H - 1 < k_old or c + H + 1 > k_newest for c in cen):
                continue
            valid[w] = 1
            row = int(trig_row[s])
            for I in range(D):
                for u in range(Lw):
                    q, r = divmod(u, R)
                    base = cen[I] - H + q
                    if r == 0:
                        out[I, w, u] = z[I, row, base % ring_len]
                    else:
                        acc = 0.0
                        for m in range(4):
                            acc = acc + W[r][m] * complex(z[I, row, (base - 1 + m) % ring_len])
                        out[I, w, u] = acc
    return out, valid
