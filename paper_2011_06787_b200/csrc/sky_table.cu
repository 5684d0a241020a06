// Host-side look-up table build (float64; "tables of U and of the
// time offsets ... prepared every day").  Not on the hot path.
//
//   directions : HEALPix RING pixel centres (pixelisation of ref. [46])
//   G+ , Gx    : D_I : e+ , D_I : ex at psi = 0 (Eq. 17-18)
//   U2         : first two left singular vectors of G_sigma = [sigma_I G+_I, sigma_I Gx_I]
//                (Eq. 27; I = diag(1,1,0..) keeps two columns)
//   delay      : rint(-(r_I . n) / c * fs) per detector against the geocentre
//
// The N_d x 2 SVD is done in closed form through the 2 x 2 eigenproblem of
// G^T G (U_j = G v_j / sqrt(lambda_j)); only the projector U2 U2^T is unique.
#include <cmath>

#include "spiir_internal.cuh"

namespace {

const double kPi = 3.14159265358979323846;
const double kC = 299792458.0;

// centre (z = cos theta, phi) of RING pixel p
void ring_centre(long nside, long p, double* z, double* phi) {
  const long npix = 12 * nside * nside, ncap = 2 * nside * (nside - 1);
  if (p < ncap) {                                   // north polar cap: ring i has 4 i pixels
    long i = (long)std::floor(0.5 * (1.0 + std::sqrt(1.0 + 2.0 * (double)p)));
    while (2 * i * (i - 1) > p) --i;                // guard the float sqrt at ring edges
    while (2 * i * (i + 1) <= p) ++i;
    const long j = p - 2 * i * (i - 1);             // 0-based position in the ring
    *z = 1.0 - (double)(i * i) / (3.0 * nside * nside);
    *phi = ((double)j + 0.5) * kPi / (2.0 * i);
  } else if (p < npix - ncap) {                     // equatorial belt: every ring has 4 nside pixels
    const long q = p - ncap;
    const long i = q / (4 * nside) + nside, j = q % (4 * nside);
    const double shift = ((i + nside) % 2 == 0) ? 0.5 : 0.0;
    *z = (double)(2 * nside - i) * 2.0 / (3.0 * nside);
    *phi = ((double)j + shift) * kPi / (2.0 * nside);
  } else {                                          // south cap: mirror image, rings counted from the pole
    const long q = npix - 1 - p;                    // 0-based from the end
    long i = (long)std::floor(0.5 * (1.0 + std::sqrt(1.0 + 2.0 * (double)q)));
    while (2 * i * (i - 1) > q) --i;
    while (2 * i * (i + 1) <= q) ++i;
    const long jr = q - 2 * i * (i - 1);            // position counted backwards
    const long j = 4 * i - 1 - jr;
    *z = -1.0 + (double)(i * i) / (3.0 * nside * nside);
    *phi = ((double)j + 0.5) * kPi / (2.0 * i);
  }
}

}  // namespace

extern "C" int spiir_sky_table_build(int32_t nside, int32_t n_det, const double* pos, const double* resp,
                                     const double* sigma, double gmst, double fs, float* u2, int32_t* delay) {
  SPIIR_REQUIRE(nside >= 1 && nside <= 8192, "nside %d out of range", nside);
  SPIIR_REQUIRE(n_det >= 2 && n_det <= SPIIR_MAX_DET, "n_det %d out of range", n_det);
  SPIIR_REQUIRE(pos && resp && sigma && u2 && delay, "a pointer is NULL");
  SPIIR_REQUIRE(fs > 0.0, "fs_hz must be positive");
  const long npix = 12L * nside * nside;
  for (long p = 0; p < npix; ++p) {
    double cz, phi;
    ring_centre(nside, p, &cz, &phi);
    const double sz = std::sqrt(std::fmax(0.0, 1.0 - cz * cz));
    const double lam = phi - gmst;                                  // Earth-fixed longitude of the source
    const double n[3] = {sz * std::cos(lam), sz * std::sin(lam), cz};
    const double X[3] = {std::sin(lam), -std::cos(lam), 0.0};
    const double Y[3] = {-cz * std::cos(lam), -cz * std::sin(lam), sz};
    double G[SPIIR_MAX_DET][2];
    for (int I = 0; I < n_det; ++I) {
      const double* D = resp + 9 * I;
      double gp = 0.0, gc = 0.0;
      for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c) {
          gp += D[3 * r + c] * (X[r] * X[c] - Y[r] * Y[c]);
          gc += D[3 * r + c] * (X[r] * Y[c] + Y[r] * X[c]);
        }
      G[I][0] = sigma[I] * gp;
      G[I][1] = sigma[I] * gc;
      const double tau = -(pos[3 * I] * n[0] + pos[3 * I + 1] * n[1] + pos[3 * I + 2] * n[2]) / kC;
      delay[p * n_det + I] = (int32_t)std::nearbyint(tau * fs);     // round-half-even (default mode)
    }
    // eigen-decomposition of the symmetric 2 x 2 matrix M = G^T G
    double A = 0, Bm = 0, C = 0;
    for (int I = 0; I < n_det; ++I) { A += G[I][0] * G[I][0]; Bm += G[I][0] * G[I][1]; C += G[I][1] * G[I][1]; }
    const double half = 0.5 * (A - C), rad = std::hypot(half, Bm);
    const double l1 = 0.5 * (A + C) + rad, l2 = 0.5 * (A + C) - rad;
    double v1[2];
    if (rad > 0.0) {
      // eigenvector of l1: (Bm, l1 - A) or (l1 - C, Bm), whichever is longer
      const double ax = Bm, ay = l1 - A, bx = l1 - C, by = Bm;
      if (ax * ax + ay * ay >= bx * bx + by * by) { v1[0] = ax; v1[1] = ay; } else { v1[0] = bx; v1[1] = by; }
      const double nv = std::hypot(v1[0], v1[1]);
      v1[0] /= nv; v1[1] /= nv;
    } else { v1[0] = 1.0; v1[1] = 0.0; }
    const double v2[2] = {-v1[1], v1[0]};
    double U[SPIIR_MAX_DET][2];
    double n1 = 0, n2 = 0;
    for (int I = 0; I < n_det; ++I) {
      U[I][0] = G[I][0] * v1[0] + G[I][1] * v1[1];
      U[I][1] = G[I][0] * v2[0] + G[I][1] * v2[1];
      n1 += U[I][0] * U[I][0]; n2 += U[I][1] * U[I][1];
    }
    SPIIR_REQUIRE(n1 > 0.0, "pixel %ld: the network has no response (all sigma zero?)", p);
    for (int I = 0; I < n_det; ++I) U[I][0] /= std::sqrt(n1);
    if (n2 > 1e-24 * n1 && l2 > 0.0) {
      // remove any residual overlap with the first vector, then normalise
      double dot = 0; for (int I = 0; I < n_det; ++I) dot += U[I][0] * U[I][1];
      n2 = 0; for (int I = 0; I < n_det; ++I) { U[I][1] -= dot * U[I][0]; n2 += U[I][1] * U[I][1]; }
      for (int I = 0; I < n_det; ++I) U[I][1] /= std::sqrt(n2);
    } else {
      // rank one: complete the plane with the coordinate axis least aligned with U1
      int best = 0;
      for (int I = 1; I < n_det; ++I) if (std::fabs(U[I][0]) < std::fabs(U[best][0])) best = I;
      n2 = 0;
      for (int I = 0; I < n_det; ++I) { U[I][1] = (I == best ? 1.0 : 0.0) - U[best][0] * U[I][0]; n2 += U[I][1] * U[I][1]; }
      for (int I = 0; I < n_det; ++I) U[I][1] /= std::sqrt(n2);
    }
    for (int I = 0; I < n_det; ++I) {
      u2[(p * n_det + I) * 2] = (float)U[I][0];
      u2[(p * n_det + I) * 2 + 1] = (float)U[I][1];
    }
  }
  return SPIIR_OK;
}

// NEXT-3: the tables sampled along the Earth's rotation, and the nearest-in-time set.
extern "C" int spiir_sky_table_set_build(int32_t nside, int32_t n_det, const double* pos, const double* resp,
                                         const double* sigma, double gmst0, double interval_s, int32_t n_sets,
                                         double fs, float* u2, int32_t* delay) {
  SPIIR_REQUIRE(n_sets >= 1 && n_sets <= 4096, "n_sets %d out of range", n_sets);
  SPIIR_REQUIRE(interval_s > 0.0, "interval_s must be positive");
  const double kSiderealDay = 86164.0905;
  const size_t npix = (size_t)12 * nside * nside;
  for (int i = 0; i < n_sets; ++i) {
    const double gm = gmst0 + 2.0 * kPi * ((double)i * interval_s) / kSiderealDay;
    const int rc = spiir_sky_table_build(nside, n_det, pos, resp, sigma, gm, fs, u2 + (size_t)i * npix * n_det * 2,
                                         delay + (size_t)i * npix * n_det);
    if (rc) return rc;
  }
  return SPIIR_OK;
}

extern "C" int spiir_sky_table_nearest(double t, double t0, double interval_s, int32_t n_sets, int32_t* index) {
  SPIIR_REQUIRE(index != nullptr, "index is NULL");
  SPIIR_REQUIRE(n_sets >= 1 && interval_s > 0.0, "bad n_sets / interval_s");
  *index = -1;
  double x = (t - t0) / interval_s;
  SPIIR_REQUIRE(x == x, "t_s / t0_s is not a number");
  x = x < -1.0 ? -1.0 : (x > (double)n_sets ? (double)n_sets : x);
  long i = (long)std::ceil(x - 0.5);                      // nearest; x = i + 1/2 goes to the earlier set i
  i = i < 0 ? 0 : (i > n_sets - 1 ? n_sets - 1 : i);
  // settle the last ulp by the distances themselves, as the definition does
  while (i > 0 && std::fabs(t - (t0 + (double)(i - 1) * interval_s)) <= std::fabs(t - (t0 + (double)i * interval_s))) --i;
  while (i < n_sets - 1 && std::fabs(t - (t0 + (double)(i + 1) * interval_s)) < std::fabs(t - (t0 + (double)i * interval_s))) ++i;
  if (std::fabs(t - (t0 + (double)i * interval_s)) > 0.5 * interval_s) return SPIIR_OK;
  *index = (int32_t)i;
  return SPIIR_OK;
}
