"""ORACLE (test infrastructure only) — NEXT-2: ranking statistic and false-alarm probability from the
time-slide background, PAPER.md:202-225 (Sec. II D 1, Eq. 13-15).

Plain numpy, written out from the definitions, no cumulative-sum tricks:
  * selection of coherent events: rho_C >= rho_I + sqrt(2);
  * P(rho_C, xi_C^2 | n): a 2-D histogram of the selected background events;
  * R(rho', xi') = sum over bins with rho >= rho' and xi^2 <= xi' of P (Eq. 13, at bin granularity);
  * FAP(R') = sum over bins with R < R' of P (Eq. 14);   FAR = FAP * N_b / T_b (Eq. 15).
The paper gives no binning.  Reading X3: both axes are binned uniformly in the pseudo-logarithm
u(x) = e + (m - 1) of x = m 2^e (m in [1, 2)), read off the float32 bit pattern, so that the bin of an event
is decided by the same few float32 operations on both sides (no transcendental function).
Counts are integers; R and FAP are compared as integer counts (exact), and reported as count / N_b.
"""
import numpy as np

SQRT2_F32 = np.float32(1.41421356)


def pseudo_log2(x):
    """u(x) = (bits(x) - bits(1.0)) * 2^-23 in float32 for float32 x > 0 (piecewise-linear log2)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    d = x.view(np.int32).astype(np.int64) - 0x3F800000
    return (d.astype(np.int32).astype(np.float32) * np.float32(2.0 ** -23)).astype(np.float32)


def bin_index(x, u_min, u_max, n):
    """Bin of x on an axis of n uniform bins in u over [u_min, u_max); outside values go to the edge bins,
    x <= 0 to bin 0.  All arithmetic in float32: floor((u - u_min) * scale), scale = float32(n / (u_max - u_min))."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    scale = np.float32(np.float32(n) / (np.float32(u_max) - np.float32(u_min)))
    u = pseudo_log2(np.where(x > 0, x, np.float32(1.0)))
    t = np.floor((u - np.float32(u_min)).astype(np.float32) * scale).astype(np.float32)
    b = np.clip(t, 0, n - 1).astype(np.int64)
    return np.where(x > 0, b, 0)


def select(snr_trig, coh2, used):
    """rho_C >= rho_I + sqrt(2), in float32 (sqrtf, one add, one compare)."""
    rho_c = np.sqrt(np.asarray(coh2, np.float32)).astype(np.float32)
    return (np.asarray(used) != 0) & (rho_c >= (np.asarray(snr_trig, np.float32) + SQRT2_F32).astype(np.float32))


def histogram(bins, snr_trig, coh2, xi2_c, used):
    """H[n_rho][n_xi] int64 of the selected events; bins = (n_rho, n_xi, u_rho_min, u_rho_max, u_xi_min, u_xi_max)."""
    n_rho, n_xi, r0, r1, x0, x1 = bins
    sel = select(snr_trig, coh2, used)
    i = bin_index(np.asarray(coh2, np.float32)[sel], r0, r1, n_rho)
    j = bin_index(np.asarray(xi2_c, np.float32)[sel], x0, x1, n_xi)
    H = np.zeros((n_rho, n_xi), np.int64)
    for a, b in zip(i, j):
        H[a, b] += 1
    return H


def rank_counts(H):
    """C[i][j] = sum_{i' >= i, j' <= j} H[i'][j']  (Eq. 13 times N_b), written as the double sum it is."""
    n_rho, n_xi = H.shape
    Cc = np.zeros_like(H)
    for i in range(n_rho):
        for j in range(n_xi):
            Cc[i, j] = H[i:, :j + 1].sum()
    return Cc


def fap_counts(H, Cc):
    """F[i][j] = sum over bins (i', j') with C[i'][j'] < C[i][j] of H[i'][j']  (Eq. 14 times N_b)."""
    F = np.zeros_like(H)
    flatC, flatH = Cc.reshape(-1), H.reshape(-1)
    for b in range(flatC.size):
        F.reshape(-1)[b] = flatH[flatC < flatC[b]].sum()
    return F


def candidates(bins, H, snr_trig, coh2, xi2_c, used, background_seconds):
    """Per foreground candidate: (R, FAP, FAR, selected).  R = C/N_b, FAP = F/N_b, FAR = FAP N_b / T_b."""
    n_rho, n_xi, r0, r1, x0, x1 = bins
    Cc = rank_counts(H)
    F = fap_counts(H, Cc)
    nb = int(H.sum())
    sel = select(snr_trig, coh2, used)
    i = bin_index(coh2, r0, r1, n_rho)
    j = bin_index(xi2_c, x0, x1, n_xi)
    R = np.where(sel, Cc[i, j] / max(nb, 1), 0.0)
    fap = np.where(sel, F[i, j] / max(nb, 1), 0.0)
    far = np.where(sel, F[i, j] / float(background_seconds), 0.0)            # FAP * N_b / T_b
    return R, fap, far, sel.astype(np.int32)
