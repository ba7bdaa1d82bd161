// Host-side derivation of the geometry-only constants (O1).
//
// Everything is computed in double from the float geometry fields and rounded once to float.
// The least-squares maps P (x-z, Eq. 1) and Q (y-z straight line, L215) exist because
// the layer z positions are constants: the fit of each hit pattern is one fixed matrix.  They are
// obtained here from a thin QR factorisation (modified Gram-Schmidt, re-orthogonalised) of the
// column-scaled design matrix.
#pragma once
#include <cmath>
#include <cstring>

#include "../../include/lhcb.h"

namespace lhcb {

// pinv = R^-1 Q^T of the n x m matrix A (row-major), m <= 3, n <= 6.  out is m x n row-major.
inline bool qr_pinv(int n, int m, const double* A, double* out) {
  double scale[3], Qm[3][6], R[3][3] = {{0}};
  for (int j = 0; j < m; ++j) {
    scale[j] = 0;
    for (int i = 0; i < n; ++i) scale[j] = std::fmax(scale[j], std::fabs(A[i * m + j]));
    if (scale[j] == 0) return false;
    for (int i = 0; i < n; ++i) Qm[j][i] = A[i * m + j] / scale[j];
  }
  for (int j = 0; j < m; ++j) {
    for (int pass = 0; pass < 2; ++pass)              // two passes: orthogonal to working precision
      for (int k = 0; k < j; ++k) {
        double dot = 0;
        for (int i = 0; i < n; ++i) dot += Qm[k][i] * Qm[j][i];
        R[k][j] += dot;
        for (int i = 0; i < n; ++i) Qm[j][i] -= dot * Qm[k][i];
      }
    double nrm = 0;
    for (int i = 0; i < n; ++i) nrm += Qm[j][i] * Qm[j][i];
    nrm = std::sqrt(nrm);
    if (!(nrm > 1e-12)) return false;
    R[j][j] = nrm;
    for (int i = 0; i < n; ++i) Qm[j][i] /= nrm;
  }
  // back substitution: R X = Q^T, column by column of Q^T (i.e. per hit i)
  for (int i = 0; i < n; ++i) {
    double x[3];
    for (int j = m - 1; j >= 0; --j) {
      double v = Qm[j][i];
      for (int k = j + 1; k < m; ++k) v -= R[j][k] * x[k];
      x[j] = v / R[j][j];
    }
    for (int j = 0; j < m; ++j) out[j * n + i] = x[j] / scale[j];
  }
  return true;
}

inline double g_of(double zb, double d) { return zb * zb * (1.0 + d * zb); }

inline int resolve_capacity(int v, int dflt) { return v > 0 ? v : dflt; }

inline void resolve_defaults(lhcb_geom_t& g) {
  g.max_seeds_per_half = resolve_capacity(g.max_seeds_per_half, 256);
  g.max_xz_cand_per_half = resolve_capacity(g.max_xz_cand_per_half, 1024);
  g.max_long_per_event = resolve_capacity(g.max_long_per_event, 256);
  g.max_hits_per_half = resolve_capacity(g.max_hits_per_half, 6144);
  g.max_triplets_per_half = resolve_capacity(g.max_triplets_per_half, 4096);
  g.max_match_cand_per_event = resolve_capacity(g.max_match_cand_per_event, 384);
  g.max_velo_per_event = resolve_capacity(g.max_velo_per_event, 512);
  g.max_ut_per_event = resolve_capacity(g.max_ut_per_event, 6144);
}

inline int derive(const lhcb_geom_t& g, lhcb_derived_t& D) {
  std::memset(&D, 0, sizeof(D));
  int nx = 0, nu = 0;
  for (int l = 0; l < 12; ++l) {
    if (l > 0 && !(g.scifi_z[l] > g.scifi_z[l - 1])) return LHCB_ERR_BAD_GEOMETRY;
    if (g.scifi_tan_alpha[l] == 0.0f) {
      if (nx < 6) { D.xl[nx] = l; D.slot_of_layer[l] = nx; }
      ++nx;
    } else {
      if (nu < 6) { D.ul[nu] = l; D.slot_of_layer[l] = nu; }
      ++nu;
    }
  }
  if (nx != 6 || nu != 6) return LHCB_ERR_BAD_GEOMETRY;
  if (g.min_x_hits < 5 || g.min_x_hits > 6 || g.min_uv_hits < 2 || g.min_uv_hits > 6) return LHCB_ERR_BAD_GEOMETRY;
  if (!(g.sigma_hit > 0) || !(g.kappa_cx != 0) || !(g.kick_pt != 0) || g.gamma_ab[1] == 0)
    return LHCB_ERR_BAD_GEOMETRY;
  for (int pp = 0; pp < 2; ++pp) {                           // first layer of each UV pass: a stereo layer
    const int lf = g.uv_first_layer[pp];
    if (lf < 0 || lf >= 12 || g.scifi_tan_alpha[lf] == 0.0f) return LHCB_ERR_BAD_GEOMETRY;
  }
  if (g.min_ut_hits < 1 || g.min_ut_hits > 4) return LHCB_ERR_BAD_GEOMETRY;
  if (!(g.y_max > 0) || !(g.y_min < 0) || !(g.y_half_tol >= 0)) return LHCB_ERR_BAD_GEOMETRY;
  const double zref = g.z_ref, dr = g.d_ratio;
  for (int l = 0; l < 12; ++l) {
    const double z = g.scifi_z[l], zb = z - zref, ta = g.scifi_tan_alpha[l];
    D.zb[l] = (float)zb;
    D.gz[l] = (float)g_of(zb, dr);
    D.tan_a[l] = (float)ta;
    D.inv_tan[l] = ta != 0.0 ? (float)(1.0 / ta) : 0.0f;
    D.inv_z[l] = (float)(1.0 / z);
    D.zt[l] = (float)(z * ta);
    D.ywin_a[0][l] = (float)(-(double)g.y_half_tol * ta);
    D.ywin_b[0][l] = (float)((double)g.y_max * ta);
    D.ywin_a[1][l] = (float)((double)g.y_min * ta);
    D.ywin_b[1][l] = (float)((double)g.y_half_tol * ta);
  }
  for (int it = 0; it < 2; ++it) {
    const int l1 = g.iter_layers[it][0], l2 = g.iter_layers[it][1], l3 = g.iter_layers[it][2];
    for (int l : {l1, l2, l3})
      if (l < 0 || l >= 12 || g.scifi_tan_alpha[l] != 0.0f) return LHCB_ERR_BAD_GEOMETRY;
    if (!(l1 < l2 && l2 < l3)) return LHCB_ERR_BAD_GEOMETRY;
    const double z1 = g.scifi_z[l1], z2 = g.scifi_z[l2], z3 = g.scifi_z[l3];
    const double a = g.inv_p_a, b = g.inv_p_b, pmin = g.p_min;
    const double g1 = g_of(z1 - zref, dr), g2 = g_of(z2 - zref, dr), g3 = g_of(z3 - zref, dr);
    const double root = std::sqrt(a * a + 4.0 * b / pmin);
    const double dx3 = (z3 - z1) / (2.0 * z1 * b) * (root - a);                  // Eq. 8
    const double ratio = z1 / (z3 - z1);
    const double acorr = (double)g.alpha0 / (ratio * (pmin - (double)g.alpha1));  // Eq. 9-10
    const double K = (g2 - g1) - (z2 - z1) / (z3 - z1) * (g3 - g1);              // reading A3
    if (!std::isfinite(dx3) || !std::isfinite(acorr) || !std::isfinite(K) || K == 0.0)
      return LHCB_ERR_BAD_GEOMETRY;                          // e.g. p_min below the real root of Eq. 8
    D.l1[it] = l1; D.l2[it] = l2; D.l3[it] = l3;
    D.dx3max[it] = (float)dx3;
    D.alpha_corr[it] = (float)acorr;
    D.r13[it] = (float)((z3 + acorr) / z1);                                        // Eq. 11
    D.inv_dz13[it] = (float)(1.0 / (z3 - z1));
    D.z1[it] = (float)z1;
    D.dz12[it] = (float)(z2 - z1);
    D.K[it] = (float)K;
    D.inv_K[it] = (float)(1.0 / K);
    D.G13[it] = (float)((g3 - g1) / (z3 - z1));
  }
  D.a = g.inv_p_a; D.b = g.inv_p_b; D.kappa = g.kappa_cx;
  D.inv_kappa = (float)(1.0 / (double)g.kappa_cx);
  D.f_lo = g.cx_band[0]; D.f_hi = g.cx_band[1]; D.d_lo = g.cx_band[2]; D.d_hi = g.cx_band[3];
  D.tol_x = g.tol_x_ext; D.tol_uv = g.tol_uv; D.chi2x_max = g.chi2x_max; D.chi2y_max = g.chi2y_max;
  const double s2 = (double)g.sigma_hit * (double)g.sigma_hit;
  for (int n = 0; n <= 6; ++n) {
    D.wx[n] = n > 3 ? (float)(1.0 / (s2 * (n - 3))) : 0.0f;
    D.wy[n] = n > 2 ? (float)(1.0 / (s2 * (n - 2))) : 0.0f;
  }
  // x-z map per pattern
  for (int pat = 0; pat <= 6; ++pat) {
    double A[18], out[18];
    int n = 0, slot[6];
    for (int s = 0; s < 6; ++s) {
      if (pat == 1 + s) continue;
      const double zb = (double)g.scifi_z[D.xl[s]] - zref;
      A[n * 3] = 1.0; A[n * 3 + 1] = zb; A[n * 3 + 2] = g_of(zb, dr);
      slot[n++] = s;
    }
    if (!qr_pinv(n, 3, A, out)) return LHCB_ERR_BAD_GEOMETRY;
    for (int r = 0; r < 3; ++r)
      for (int i = 0; i < n; ++i) D.P[pat][r][slot[i]] = (float)out[r * n + i];
  }
  // y-z map per stereo-slot mask (rows tan(alpha)*[1, zb])
  for (int mask = 0; mask < 64; ++mask) {
    double A[12], out[12];
    int n = 0, slot[6];
    for (int s = 0; s < 6; ++s)
      if (mask >> s & 1) {
        const double zb = (double)g.scifi_z[D.ul[s]] - zref, ta = g.scifi_tan_alpha[D.ul[s]];
        A[n * 2] = ta; A[n * 2 + 1] = ta * zb;
        slot[n++] = s;
      }
    if (n < 2) continue;
    if (!qr_pinv(n, 2, A, out)) return LHCB_ERR_BAD_GEOMETRY;
    for (int r = 0; r < 2; ++r)
      for (int i = 0; i < n; ++i) D.Q[mask][r][slot[i]] = (float)out[r * n + i];
  }
  {
    const double zb = (double)g.z_scifi_state - zref;
    D.zbS = (float)zb; D.gS = (float)g_of(zb, dr); D.gpS = (float)(2.0 * zb + 3.0 * dr * zb * zb);
  }
  D.zS = g.z_scifi_state; D.zV = g.z_velo;
  D.dzyS = (float)((double)g.z_match_y - (double)g.z_scifi_state);
  D.dzyV = (float)((double)g.z_match_y - (double)g.z_velo);
  for (int i = 0; i < 5; ++i) D.mag[i] = g.mag[i];
  for (int i = 0; i < 4; ++i) D.presel[i] = g.presel[i];
  const double t0 = g.match_tol[0], t1 = g.match_tol[1], t2 = g.match_tol[2], t3 = g.match_tol[3],
               t4 = g.match_tol[4], t5 = g.match_tol[5];
  D.cx0 = (float)(t0 * t1 * t1); D.cx1 = (float)(t0 * t2 * t2);                   // Eq. 23
  D.cy0 = (float)(t3 * t4 * t4); D.cy1 = (float)(t3 * t5 * t5);
  D.inv_tol_tx = (float)(1.0 / (double)g.match_tol[6]); D.inv_tol_ty = g.match_tol[7];
  D.chi2m_max = g.chi2_match_max;
  D.inv_KB = (float)(1.0 / (double)g.kick_pt);
  D.Ag = g.gamma_ab[0]; D.Bg = g.gamma_ab[1]; D.inv_Bg = (float)(1.0 / (double)g.gamma_ab[1]);
  for (int i = 0; i < 4; ++i) {
    const double dz = (double)g.ut_z[i] - (double)g.z_velo;
    D.ut_dz[i] = (float)dz; D.ut_dz2[i] = (float)(dz * dz); D.ut_dz4[i] = (float)(dz * dz * dz * dz);
    D.ut_tan[i] = g.ut_tan_alpha[i];
    for (int k = 0; k < 4; ++k) { D.ut_loose[i][k] = g.ut_loose[i][k]; D.ut_tight[i][k] = g.ut_tight[i][k]; }
  }
  D.ut_y_tol = g.ut_y_tol;
  return LHCB_OK;
}

}  // namespace lhcb
