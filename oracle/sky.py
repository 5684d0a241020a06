"""O5 — the per-direction look-up table of the coherent search, in float64 numpy.

ORACLE / TEST INFRASTRUCTURE (see spiir_oracle.c header).  Follows PAPER.md:169
(HEALPix pixel centres as sky directions), PAPER.md:173 (tables of U and of the
detectors' time offsets per direction), PAPER.md:417-428 (G+, Gx)
(Eq. 27: G_sigma = U Lambda V^T), with readings A18, A20-A23 of DESIGN.md.
numpy.linalg.svd is the library primitive for the decomposition.
"""
import numpy as np

C_LIGHT = 299792458.0


def healpix_ring_centres(nside):
    """(theta, phi) of the 12 nside^2 pixel centres in RING order (ref. [46] of the
    paper).  Written pixel by pixel from the defining formulas."""
    N = int(nside)
    npix = 12 * N * N
    ncap = 2 * N * (N - 1)
    theta = np.zeros(npix)
    phi = np.zeros(npix)
    for p in range(npix):
        if p < ncap:                                         # north polar cap
            ph = (p + 1) / 2.0
            i = int(np.floor(np.sqrt(ph - np.sqrt(np.floor(ph))))) + 1
            j = p + 1 - 2 * i * (i - 1)
            z = 1.0 - i * i / (3.0 * N * N)
            f = (j - 0.5) * np.pi / (2.0 * i)
        elif p < npix - ncap:                                # equatorial belt
            pp = p - ncap
            i = pp // (4 * N) + N
            j = pp % (4 * N) + 1
            fodd = 0.5 if (i + N) % 2 == 0 else 1.0          # rings alternate by half a pixel
            z = (2 * N - i) * 2.0 / (3.0 * N)
            f = (j - fodd) * np.pi / (2.0 * N)
        else:                                                # south polar cap
            ps = npix - p
            ph = ps / 2.0
            i = int(np.floor(np.sqrt(ph - np.sqrt(np.floor(ph))))) + 1
            j = 4 * i + 1 - (ps - 2 * i * (i - 1))
            z = -1.0 + i * i / (3.0 * N * N)
            f = (j - 0.5) * np.pi / (2.0 * i)
        theta[p] = np.arccos(z)
        phi[p] = f
    return theta, phi


def g_sigma(theta, phi, resp, sigma, gmst):
    """G_sigma [P][D][2] = sigma_I (G_I^+, G_I^x) at psi = 0 (Eq. 27), and the
    Earth-fixed unit vectors n [P][3] towards the sources."""
    lam = phi - gmst
    st, ct = np.sin(theta), np.cos(theta)
    n = np.stack([st * np.cos(lam), st * np.sin(lam), ct], axis=1)
    X = np.stack([np.sin(lam), -np.cos(lam), np.zeros_like(lam)], axis=1)
    Y = np.stack([-ct * np.cos(lam), -ct * np.sin(lam), st], axis=1)
    ep = np.einsum("pi,pj->pij", X, X) - np.einsum("pi,pj->pij", Y, Y)
    ec = np.einsum("pi,pj->pij", X, Y) + np.einsum("pi,pj->pij", Y, X)
    gp = np.einsum("dij,pij->pd", resp, ep)
    gc = np.einsum("dij,pij->pd", resp, ec)
    sig = np.asarray(sigma, float)[None, :]
    return np.stack([sig * gp, sig * gc], axis=2), n


def sky_table(nside, pos, resp, sigma, gmst, fs):
    """Returns (U2 float64 [P][D][2], delay int32 [P][D]).

    U2 = first two left singular vectors of G_sigma (I = diag(1,1,0..) keeps two
    columns).  delay_I = rint(-(r_I . n)/c * fs), per detector
    against the geocentre; differences are taken at use (A18)."""
    theta, phi = healpix_ring_centres(nside)
    G, n = g_sigma(theta, phi, np.asarray(resp, float), sigma, gmst)
    U, S, Vt = np.linalg.svd(G, full_matrices=True)
    U2 = np.ascontiguousarray(U[:, :, :2])
    tau = -(n @ np.asarray(pos, float).T) / C_LIGHT
    delay = np.rint(tau * fs).astype(np.int32)
    return U2, delay


# ----------------------------------------------------------------------------- O10 (NEXT-3)
# "we sample U every half hour up to 24 hours and refreshed every day ...  Time offsets of SNRs
# from different detectors are sampled at the same interval along with U.  The pipeline will
# calculate the coherent SNR using the U and offset sample that are closest in the time to the
# triggering candidate".
SIDEREAL_DAY_S = 86164.0905          # one turn of the Earth against the stars, in seconds


def table_set(nside, pos, resp, sigma, gmst0, interval_s, n_sets, fs):
    """Set i is the table of `sky_table` at time t0 + i interval_s, i.e. at sidereal angle
    gmst0 + 2 pi i interval_s / SIDEREAL_DAY_S (reading X6).  Returns (U2 [n][P][D][2], delay [n][P][D])."""
    U, dl = [], []
    for i in range(int(n_sets)):
        gm = gmst0 + 2.0 * np.pi * (i * float(interval_s)) / SIDEREAL_DAY_S
        u, d = sky_table(nside, pos, resp, sigma, gm, fs)
        U.append(u)
        dl.append(d)
    return np.stack(U), np.stack(dl)


def nearest_table(t, t0, interval_s, n_sets):
    """Index of the set closest in time to t, by exhaustive comparison; the earlier one on an exact
    tie; -1 when t is further than interval_s / 2 from every set (the tables are stale: PAPER.md:173
    refreshes them every day) — reading X6."""
    times = t0 + np.arange(int(n_sets)) * float(interval_s)
    dist = np.abs(float(t) - times)
    i = int(np.argmin(dist))                                  # first minimum = earlier set
    return i if dist[i] <= 0.5 * float(interval_s) else -1
