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
