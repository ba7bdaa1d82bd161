/*
 * oracle.c -- plain, slow, single-threaded CPU oracle of the LHCb HLT1 Seeding + Matching path.
 *
 * TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code, header, table or
 * constant generator with the CUDA path under paper_2606_14480_b200/ and neither includes the other.
 *
 * What it is: the paper's algorithm written out step by step (PAPER.md sections 3 and 4), in the
 * order and notation of the paper, with the readings DESIGN.md lists (A1..A21) where the paper is
 * silent or garbled.  Searches are linear scans with the literal predicate; there is no binary
 * search, no blocking, no fusion.  Steps are labelled O1..O14 as in DESIGN.md.
 *
 * Two builds of this one file: -DREAL=float ("f32 spec mode": every operation rounds to float in
 * the order DESIGN.md "Arithmetic specification" fixes, no FMA contraction; this build decides
 * parity with the CUDA path) and -DREAL=double (truth-recovery checks).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): closed forms of tests/golden/closed_forms.txt,
 * K identity, brute-force triplet enumeration, 3-point parabola vs polynomial interpolation,
 * fits vs numpy.linalg.lstsq, noise-free recovery in f64, clone-kill worked examples and
 * invariants, UV invariants, field-off matching, UT noise-free recovery, one-to-one selection.
 * Parity unpinned by the paper (pinned only by DESIGN.md readings): third-hit band (A4),
 * chi2 cut values (A6), min stereo hits and first stereo layers (A9), UT hypothesis rule (A13),
 * chi2-ranked final selection standing in for the NN (A14).
 *
 * Units: mm, MeV, q/p in 1/MeV.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifndef REAL
#define REAL float
#endif

#define NL 12
#define NX 6
#define NUT 4
#define NO_HIT 0xFFFFFFFFu

/* ------------------------------------------------------------------------------------------ */
/* Geometry as handed over by the caller (all double; the f32 build rounds every value to float
 * first, because the f32 specification takes float geometry: DESIGN.md "Arithmetic"). */
typedef struct {
  double scifi_z[NL], scifi_tan_alpha[NL];
  double z_ref, d_ratio;
  double p_min, inv_p_a, inv_p_b, alpha0, alpha1;
  int32_t iter_layers[2][3];
  double kappa_cx;
  double cx_band[4];
  double tol_x_ext, tol_uv;
  int32_t min_x_hits, min_uv_hits;
  int32_t uv_first_layer[2];
  double sigma_hit, chi2x_max, chi2y_max;
  double y_min, y_max, y_half_tol;
  double z_velo, z_scifi_state, z_match_y;
  double mag[5], gamma_ab[2], kick_pt;
  int32_t polarity;
  double presel[4], match_tol[8], chi2_match_max;
  double ut_z[NUT], ut_tan_alpha[NUT], ut_loose[NUT][4], ut_tight[NUT][4], ut_y_tol;
  int32_t min_ut_hits, ut_enabled;
} orc_geom_t;

typedef struct {
  orc_geom_t g;              /* (rounded) geometry */
  int xl[NX], ul[NX];        /* x-layer and stereo-layer indices, ascending z */
  int slot_of_layer[NL];     /* layer -> slot in xl[] or ul[] */
  /* O1 per-layer */
  REAL zb[NL], gz[NL], tan_a[NL], inv_tan[NL], inv_z[NL], zt[NL];
  /* O1 per-iteration */
  int l1[2], l2[2], l3[2];
  REAL dx3max[2], alpha_corr[2], r13[2], inv_dz13[2], z1[2], dz12[2], K[2], inv_K[2], G13[2];
  REAL a, b, kappa, inv_kappa, f_lo, f_hi, d_lo, d_hi, tol_x, tol_uv, chi2x_max, chi2y_max;
  REAL wx[NX + 1], wy[NX + 1];   /* 1/(sigma^2 * ndf) by number of hits */
  REAL P[1 + NX][3][NX];         /* x-z pseudo-inverse: pattern 0 = all six, 1+k = slot k missing */
  REAL Q[64][2][NX];             /* y-z pseudo-inverse by stereo-slot bitmask */
  REAL ywin_a[2][NL], ywin_b[2][NL];
  REAL zbS, gS, gpS;
  /* matching */
  REAL zS, zV, dzyS, dzyV, mag[5], presel[4], cx0, cx1, cy0, cy1, inv_tol_tx, inv_tol_ty, chi2m_max;
  REAL inv_KB, Ag, Bg, inv_Bg, ut_dz[NUT], ut_dz2[NUT], ut_dz4[NUT], ut_tan[NUT], ut_y_tol;
  REAL ut_loose[NUT][4], ut_tight[NUT][4];
  /* Hough-cluster UV seeding (L217, reading A20): off unless orc_set_uv_hough(ctx, 1) */
  int uv_hough;
  REAL hough_tlo[2], hough_invw, hough_w;   /* t_y bins per half: b = floor((t - tlo) * invw), 64 bins of width w */
} orc_ctx;

enum { C_T1 = 0, C_PAIRS, C_TRIPLETS, C_EXT_OK, C_FIT_OK, C_XZ_KEPT, C_UV_FIRST, C_UV_STEPS,
       C_YFITS, C_SEEDS, C_SV_PAIRS, C_PRESEL, C_CHI2_OK, C_UT_STEPS, C_UT_HYP, C_LONG, C_N };

static REAL rabs(REAL v) { return (REAL)fabs((double)v); }
static REAL rmin(REAL a, REAL b) { return a < b ? a : b; }
static REAL rmax(REAL a, REAL b) { return a > b ? a : b; }
static uint32_t f32bits(float f) { uint32_t u; memcpy(&u, &f, 4); return u; }

static double rnd(double v) { return sizeof(REAL) == 4 ? (double)(float)v : v; }

/* Least-squares pseudo-inverse (A^T A)^-1 A^T of an n x m design matrix (m <= 3), in long double
 * with column scaling and Gaussian elimination with partial pivoting.  out is m x n. */
static void pinv_cols(int n, int m, const double* A /* n x m */, double* out /* m x n */) {
  long double s[3], N[3][3], R[3][NX];
  int i, j, k;
  for (j = 0; j < m; j++) {
    s[j] = 0;
    for (i = 0; i < n; i++) { long double v = fabsl((long double)A[i * m + j]); if (v > s[j]) s[j] = v; }
    if (s[j] == 0) s[j] = 1;
  }
  for (j = 0; j < m; j++)
    for (k = 0; k < m; k++) {
      N[j][k] = 0;
      for (i = 0; i < n; i++) N[j][k] += ((long double)A[i * m + j] / s[j]) * ((long double)A[i * m + k] / s[k]);
    }
  for (j = 0; j < m; j++)
    for (i = 0; i < n; i++) R[j][i] = (long double)A[i * m + j] / s[j];
  for (k = 0; k < m; k++) {                    /* eliminate */
    int piv = k;
    for (j = k + 1; j < m; j++) if (fabsl(N[j][k]) > fabsl(N[piv][k])) piv = j;
    if (piv != k) {
      for (j = 0; j < m; j++) { long double t = N[k][j]; N[k][j] = N[piv][j]; N[piv][j] = t; }
      for (i = 0; i < n; i++) { long double t = R[k][i]; R[k][i] = R[piv][i]; R[piv][i] = t; }
    }
    for (j = 0; j < m; j++) {
      if (j == k) continue;
      long double f = N[j][k] / N[k][k];
      int c;
      for (c = 0; c < m; c++) N[j][c] -= f * N[k][c];
      for (i = 0; i < n; i++) R[j][i] -= f * R[k][i];
    }
  }
  for (j = 0; j < m; j++)
    for (i = 0; i < n; i++) out[j * n + i] = (double)(R[j][i] / N[j][j] / s[j]);
}

/* O1: everything that depends on the geometry only.  Derived constants are computed in double
 * from the (rounded) geometry and rounded once to REAL. */
int orc_init(const orc_geom_t* gin, orc_ctx* C) {
  int i, k, it, nx = 0, nu = 0;
  orc_geom_t* g = &C->g;
  memset(C, 0, sizeof(*C));
  *g = *gin;
  {                                            /* f32 spec mode: the geometry itself is float */
    double* dp;
#define RND_ARR(arr) for (dp = (double*)(arr), i = 0; i < (int)(sizeof(arr) / sizeof(double)); i++) dp[i] = rnd(dp[i])
#define RND(v) (v) = rnd(v)
    RND_ARR(g->scifi_z); RND_ARR(g->scifi_tan_alpha); RND(g->z_ref); RND(g->d_ratio);
    RND(g->p_min); RND(g->inv_p_a); RND(g->inv_p_b); RND(g->alpha0); RND(g->alpha1); RND(g->kappa_cx);
    RND_ARR(g->cx_band); RND(g->tol_x_ext); RND(g->tol_uv); RND(g->sigma_hit); RND(g->chi2x_max);
    RND(g->chi2y_max); RND(g->y_min); RND(g->y_max); RND(g->y_half_tol); RND(g->z_velo);
    RND(g->z_scifi_state); RND(g->z_match_y); RND_ARR(g->mag); RND_ARR(g->gamma_ab); RND(g->kick_pt);
    RND_ARR(g->presel); RND_ARR(g->match_tol); RND(g->chi2_match_max); RND_ARR(g->ut_z);
    RND_ARR(g->ut_tan_alpha); RND_ARR(g->ut_loose); RND_ARR(g->ut_tight); RND(g->ut_y_tol);
#undef RND_ARR
#undef RND
  }
  for (i = 0; i < NL; i++) {
    if (g->scifi_tan_alpha[i] == 0.0) { if (nx < NX) { C->xl[nx] = i; C->slot_of_layer[i] = nx; } nx++; }
    else { if (nu < NX) { C->ul[nu] = i; C->slot_of_layer[i] = nu; } nu++; }
  }
  if (nx != NX || nu != NX) return -1;
  if (g->min_x_hits < NX - 1 || g->min_uv_hits < 2) return -3;   /* one missing x layer at most */
  for (i = 0; i < NL; i++) {
    double zb = g->scifi_z[i] - g->z_ref, ta = g->scifi_tan_alpha[i];
    C->zb[i] = (REAL)zb;
    C->gz[i] = (REAL)(zb * zb * (1.0 + g->d_ratio * zb));          /* Eq. 1 */
    C->tan_a[i] = (REAL)ta;
    C->inv_tan[i] = ta != 0.0 ? (REAL)(1.0 / ta) : (REAL)0;
    C->inv_z[i] = (REAL)(1.0 / g->scifi_z[i]);
    C->zt[i] = (REAL)(g->scifi_z[i] * ta);
    /* first-layer window of O8: y in [-y_half_tol, y_max] (upper half), mirrored (lower half) */
    C->ywin_a[0][i] = (REAL)(-g->y_half_tol * ta); C->ywin_b[0][i] = (REAL)(g->y_max * ta);
    C->ywin_a[1][i] = (REAL)(g->y_min * ta);       C->ywin_b[1][i] = (REAL)(g->y_half_tol * ta);
  }
  for (it = 0; it < 2; it++) {
    int l1 = g->iter_layers[it][0], l2 = g->iter_layers[it][1], l3 = g->iter_layers[it][2];
    double z1 = g->scifi_z[l1], z2 = g->scifi_z[l2], z3 = g->scifi_z[l3];
    double a = g->inv_p_a, b = g->inv_p_b;
    double g1 = 0, g2 = 0, g3 = 0, zb;
    double dx3, kk, ac, K;
    if (g->scifi_tan_alpha[l1] != 0 || g->scifi_tan_alpha[l2] != 0 || g->scifi_tan_alpha[l3] != 0) return -2;
    zb = z1 - g->z_ref; g1 = zb * zb * (1.0 + g->d_ratio * zb);
    zb = z2 - g->z_ref; g2 = zb * zb * (1.0 + g->d_ratio * zb);
    zb = z3 - g->z_ref; g3 = zb * zb * (1.0 + g->d_ratio * zb);
    dx3 = (z3 - z1) / (2.0 * z1 * b) * (-a + sqrt(a * a + 4.0 * b / g->p_min));     /* Eq. 8 */
    kk = z1 / (z3 - z1);
    ac = g->alpha0 / (kk * (g->p_min - g->alpha1));                                  /* Eq. 9-10 */
    K = (g2 - g1) - (z2 - z1) / (z3 - z1) * (g3 - g1);                               /* A3 */
    C->l1[it] = l1; C->l2[it] = l2; C->l3[it] = l3;
    C->dx3max[it] = (REAL)dx3; C->alpha_corr[it] = (REAL)ac;
    C->r13[it] = (REAL)((z3 + ac) / z1);                                             /* Eq. 11 */
    C->inv_dz13[it] = (REAL)(1.0 / (z3 - z1)); C->z1[it] = (REAL)z1; C->dz12[it] = (REAL)(z2 - z1);
    C->K[it] = (REAL)K; C->inv_K[it] = (REAL)(1.0 / K); C->G13[it] = (REAL)((g3 - g1) / (z3 - z1));
  }
  C->a = (REAL)g->inv_p_a; C->b = (REAL)g->inv_p_b; C->kappa = (REAL)g->kappa_cx;
  C->inv_kappa = (REAL)(1.0 / g->kappa_cx);
  C->f_lo = (REAL)g->cx_band[0]; C->f_hi = (REAL)g->cx_band[1];
  C->d_lo = (REAL)g->cx_band[2]; C->d_hi = (REAL)g->cx_band[3];
  C->tol_x = (REAL)g->tol_x_ext; C->tol_uv = (REAL)g->tol_uv;
  C->chi2x_max = (REAL)g->chi2x_max; C->chi2y_max = (REAL)g->chi2y_max;
  for (i = 0; i <= NX; i++) {
    C->wx[i] = i > 3 ? (REAL)(1.0 / (g->sigma_hit * g->sigma_hit * (i - 3))) : (REAL)0;
    C->wy[i] = i > 2 ? (REAL)(1.0 / (g->sigma_hit * g->sigma_hit * (i - 2))) : (REAL)0;
  }
  /* O6: x-z least squares is a fixed linear map per hit pattern (z is constant per layer) */
  for (k = 0; k <= NX; k++) {
    double A[NX * 3], out[3 * NX];
    int n = 0, slot[NX], s, r;
    for (s = 0; s < NX; s++) {
      if (k == 1 + s) continue;
      double zb = g->scifi_z[C->xl[s]] - g->z_ref;
      A[n * 3 + 0] = 1.0; A[n * 3 + 1] = zb; A[n * 3 + 2] = zb * zb * (1.0 + g->d_ratio * zb);
      slot[n++] = s;
    }
    pinv_cols(n, 3, A, out);
    for (r = 0; r < 3; r++) for (i = 0; i < n; i++) C->P[k][r][slot[i]] = (REAL)out[r * n + i];
  }
  /* O9: rows tan(alpha_i) * [1, zb_i]; theta = -Q m */
  for (k = 0; k < 64; k++) {
    double A[NX * 2], out[2 * NX];
    int n = 0, slot[NX], s, r;
    for (s = 0; s < NX; s++) if (k >> s & 1) {
      double zb = g->scifi_z[C->ul[s]] - g->z_ref, ta = g->scifi_tan_alpha[C->ul[s]];
      A[n * 2 + 0] = ta; A[n * 2 + 1] = ta * zb; slot[n++] = s;
    }
    if (n < 2) continue;
    pinv_cols(n, 2, A, out);
    for (r = 0; r < 2; r++) for (i = 0; i < n; i++) C->Q[k][r][slot[i]] = (REAL)out[r * n + i];
  }
  {
    double zb = g->z_scifi_state - g->z_ref;
    C->zbS = (REAL)zb; C->gS = (REAL)(zb * zb * (1.0 + g->d_ratio * zb));
    C->gpS = (REAL)(2.0 * zb + 3.0 * g->d_ratio * zb * zb);
  }
  /* matching constants */
  C->zS = (REAL)g->z_scifi_state; C->zV = (REAL)g->z_velo;
  C->dzyS = (REAL)(g->z_match_y - g->z_scifi_state); C->dzyV = (REAL)(g->z_match_y - g->z_velo);
  for (i = 0; i < 5; i++) C->mag[i] = (REAL)g->mag[i];
  for (i = 0; i < 4; i++) C->presel[i] = (REAL)g->presel[i];
  C->cx0 = (REAL)(g->match_tol[0] * g->match_tol[1] * g->match_tol[1]);     /* Eq. 23 */
  C->cx1 = (REAL)(g->match_tol[0] * g->match_tol[2] * g->match_tol[2]);
  C->cy0 = (REAL)(g->match_tol[3] * g->match_tol[4] * g->match_tol[4]);
  C->cy1 = (REAL)(g->match_tol[3] * g->match_tol[5] * g->match_tol[5]);
  C->inv_tol_tx = (REAL)(1.0 / g->match_tol[6]); C->inv_tol_ty = (REAL)g->match_tol[7];
  C->chi2m_max = (REAL)g->chi2_match_max;
  C->inv_KB = (REAL)(1.0 / g->kick_pt);
  C->Ag = (REAL)g->gamma_ab[0]; C->Bg = (REAL)g->gamma_ab[1]; C->inv_Bg = (REAL)(1.0 / g->gamma_ab[1]);
  for (i = 0; i < NUT; i++) {
    double dz = g->ut_z[i] - g->z_velo;
    C->ut_dz[i] = (REAL)dz; C->ut_dz2[i] = (REAL)(dz * dz); C->ut_dz4[i] = (REAL)(dz * dz * dz * dz);
    C->ut_tan[i] = (REAL)g->ut_tan_alpha[i];
    for (k = 0; k < 4; k++) { C->ut_loose[i][k] = (REAL)g->ut_loose[i][k]; C->ut_tight[i][k] = (REAL)g->ut_tight[i][k]; }
  }
  C->ut_y_tol = (REAL)g->ut_y_tol;
  {                                                         /* A20: t_y = y / z range of each half over the stereo layers */
    double zmin = g->scifi_z[C->ul[0]], tol = fabs(g->y_half_tol);
    double ylo[2], yhi[2]; int h;
    ylo[0] = -tol; yhi[0] = g->y_max; ylo[1] = g->y_min; yhi[1] = tol;
    for (h = 0; h < 2; h++) C->hough_tlo[h] = (REAL)rnd(ylo[h] / zmin);
    C->hough_w = (REAL)rnd((yhi[0] - ylo[0]) / zmin / 64.0);
    C->hough_invw = (REAL)rnd(64.0 / ((yhi[0] - ylo[0]) / zmin));
    C->uv_hough = 0;
  }
  return 0;
}

size_t orc_ctx_size(void) { return sizeof(orc_ctx); }
int orc_real_size(void) { return (int)sizeof(REAL); }

/* ------------------------------------------------------------------------------------------ */
/* small growable arrays */
typedef struct { int it; uint32_t i1, i2, i3; } trip_t;          /* global hit indices */
typedef struct {
  REAL ax, bx, cx, chi2; int nx, it; uint32_t hit[NX]; uint64_t key; int keep;
} cand_t;
typedef struct {
  int event, half; REAL st[5], par[7]; uint32_t hit[NL]; int nx, nuv;
} seed_t;
#define VEC(T) struct { T* p; size_t n, cap; }
typedef VEC(trip_t) vtrip;
typedef VEC(cand_t) vcand;
typedef VEC(seed_t) vseed;
#define PUSH(v, val) do { if ((v)->n == (v)->cap) { (v)->cap = (v)->cap ? 2 * (v)->cap : 256; \
  (v)->p = realloc((v)->p, (v)->cap * sizeof(*(v)->p)); } (v)->p[(v)->n++] = (val); } while (0)

/* closest hit to xp in [b, e) with |x - xp| <= tol; ties -> lower index (A15).  -1 if none. */
static int64_t closest_hit(const REAL* hx, uint32_t b, uint32_t e, REAL xp, REAL tol) {
  int64_t best = -1; REAL bd = 0; uint32_t i;
  for (i = b; i < e; i++) {
    REAL d = rabs(hx[i] - xp);
    if (d <= tol && (best < 0 || d < bd)) { best = i; bd = d; }
  }
  return best;
}

/* O5 exact parabola through the three seed hits (d_ratio fixed) */
static void parabola3(const orc_ctx* C, int it, REAL x1, REAL x2, REAL x3, REAL* t13o, REAL* ax, REAL* bx, REAL* cx) {
  REAL t13 = (x3 - x1) * C->inv_dz13[it];                    /* Eq. 4 */
  REAL x2c = x1 + C->dz12[it] * t13;                         /* Eq. 12 */
  REAL c = (x2 - x2c) * C->inv_K[it];                        /* Eq. 13 with A3 */
  REAL b = t13 - c * C->G13[it];
  REAL a = (x1 - b * C->zb[C->l1[it]]) - c * C->gz[C->l1[it]];
  *t13o = t13; *ax = a; *bx = b; *cx = c;
}

static REAL xz_at(const orc_ctx* C, REAL ax, REAL bx, REAL cx, int layer) {
  return (ax + bx * C->zb[layer]) + cx * C->gz[layer];       /* Eq. 1 */
}

/* O6: least-squares fit of Eq. 1 to the attached x hits, as a correction to (ax3,bx3,cx3).
 * r[s] = x_hit - x_parabola3 at slot s (present slots only).  Returns chi2/ndf. */
static REAL fit_xz(const orc_ctx* C, int pattern, const REAL* r, int nx, REAL* ax, REAL* bx, REAL* cx) {
  REAL d[3], ssq = 0; int k, s, first;
  for (k = 0; k < 3; k++) {
    REAL acc = 0; first = 1;
    for (s = 0; s < NX; s++) {
      if (pattern == 1 + s) continue;
      if (first) { acc = C->P[pattern][k][s] * r[s]; first = 0; }
      else acc = acc + C->P[pattern][k][s] * r[s];
    }
    d[k] = acc;
  }
  first = 1;
  for (s = 0; s < NX; s++) {
    REAL rr;
    if (pattern == 1 + s) continue;
    rr = r[s] - ((d[0] + d[1] * C->zb[C->xl[s]]) + d[2] * C->gz[C->xl[s]]);
    if (first) { ssq = rr * rr; first = 0; } else ssq = ssq + rr * rr;
  }
  *ax = *ax + d[0]; *bx = *bx + d[1]; *cx = *cx + d[2];
  return ssq * C->wx[nx];
}

/* Eq. 15 with reading A8: 64-bit lexicographic key.  High word: f32 bits of m*1000*chi2; low word:
 * f32 bits of |cx| with its last bit replaced by the iteration, so that the same hit set found by
 * both iterations (identical fit up to rounding) is still ordered and only one copy survives. */
static uint64_t clone_key(REAL chi2, REAL cx, int nx, int it) {
  REAL score = (REAL)1000 * chi2;
  if (nx == 5) score = (REAL)10 * score;
  return ((uint64_t)f32bits((float)score) << 32) | ((f32bits((float)rabs(cx)) & ~1u) | (uint32_t)(it & 1));
}

/* O7: two-pass O(n) clone kill over the candidates [c0, c1) of one half.  table is indexed by
 * (global hit index - base). */
static void clone_kill(cand_t* c, size_t n, uint32_t base, uint32_t nhits) {
  uint64_t* table = malloc((nhits ? nhits : 1) * sizeof(uint64_t));
  size_t i; int s;
  for (i = 0; i < nhits; i++) table[i] = ~(uint64_t)0;
  for (i = 0; i < n; i++)                                   /* pass 1: min score per hit */
    for (s = 0; s < NX; s++)
      if (c[i].hit[s] != NO_HIT && c[i].key < table[c[i].hit[s] - base]) table[c[i].hit[s] - base] = c[i].key;
  for (i = 0; i < n; i++) {                                 /* pass 2: vote */
    int own = 0;
    for (s = 0; s < NX; s++)
      if (c[i].hit[s] != NO_HIT && table[c[i].hit[s] - base] == c[i].key) own++;
    c[i].keep = (own >= 3) || (own >= 2 && c[i].nx == 6);
  }
  free(table);
}

/* O9: straight-line y fit in measurement space.  m[s] = x_hit - x_pred for present stereo slots. */
static REAL fit_y(const orc_ctx* C, int mask, const REAL* m, int n, REAL* ay, REAL* by) {
  REAL th[2], ssq = 0; int k, s, first;
  for (k = 0; k < 2; k++) {
    REAL acc = 0; first = 1;
    for (s = 0; s < NX; s++) {
      if (!(mask >> s & 1)) continue;
      if (first) { acc = C->Q[mask][k][s] * m[s]; first = 0; }
      else acc = acc + C->Q[mask][k][s] * m[s];
    }
    th[k] = -acc;
  }
  first = 1;
  for (s = 0; s < NX; s++) {
    REAL rr;
    if (!(mask >> s & 1)) continue;
    rr = m[s] + C->tan_a[C->ul[s]] * (th[0] + th[1] * C->zb[C->ul[s]]);
    if (first) { ssq = rr * rr; first = 0; } else ssq = ssq + rr * rr;
  }
  *ay = th[0]; *by = th[1];
  return ssq * C->wy[n];
}

/* One event-half.  zoff: the 13 zone offsets of this half (global hit indices). */
static void seed_half(const orc_ctx* C, const uint32_t* zoff, const REAL* hx, int pol, int event, int half,
                      vtrip* trips, vcand* cands, vseed* seeds, uint64_t* cnt) {
  size_t cand0 = cands->n, ci;
  int it, s;
  for (it = 0; it < 2; it++) {                                                  /* S6 / L78 */
    int l1 = C->l1[it], l2 = C->l2[it], l3 = C->l3[it];
    uint32_t i1, i2, i3;
    for (i1 = zoff[l1]; i1 < zoff[l1 + 1]; i1++) {                              /* O2 */
      REAL x1 = hx[i1];
      REAL c = x1 * C->r13[it];                                                 /* Eq. 11 */
      REAL lo = c - C->dx3max[it], hi = c + C->dx3max[it];
      cnt[C_T1]++;
      for (i3 = zoff[l3]; i3 < zoff[l3 + 1]; i3++) {
        REAL x3 = hx[i3], t13, x0, s0, invp, x2c, kinv, cxp, ca, cb, cxlo, cxhi, e1, e2, lo2, hi2;
        if (!(lo <= x3 && x3 <= hi)) continue;
        cnt[C_PAIRS]++;
        t13 = (x3 - x1) * C->inv_dz13[it];                                      /* O3, Eq. 4 */
        x0 = x1 - C->z1[it] * t13;                                              /* Eq. 3 */
        s0 = x0 >= (REAL)0 ? (REAL)1 : (REAL)-1;
        invp = C->a * rabs(x0) + C->b * (x0 * x0);                              /* Eq. 5 */
        x2c = x1 + C->dz12[it] * t13;                                           /* O4, Eq. 12 */
        kinv = C->kappa * invp;
        cxp = s0 > 0 ? -kinv : kinv;                                            /* A3 */
        ca = C->f_lo * cxp; cb = C->f_hi * cxp;                                 /* A4 */
        cxlo = rmin(ca, cb) - C->d_lo; cxhi = rmax(ca, cb) + C->d_hi;
        e1 = x2c + C->K[it] * cxlo; e2 = x2c + C->K[it] * cxhi;
        lo2 = rmin(e1, e2); hi2 = rmax(e1, e2);
        for (i2 = zoff[l2]; i2 < zoff[l2 + 1]; i2++) {
          REAL x2 = hx[i2], ax, bx, cx, tt, r[NX], chi2;
          cand_t cd; int nx = 0, pattern = 0;
          if (!(lo2 <= x2 && x2 <= hi2)) continue;
          cnt[C_TRIPLETS]++;
          if (trips) { trip_t t = { it, i1, i2, i3 }; PUSH(trips, t); }
          parabola3(C, it, x1, x2, x3, &tt, &ax, &bx, &cx);                     /* O5 */
          for (s = 0; s < NX; s++) {
            int l = C->xl[s];
            REAL xp = xz_at(C, ax, bx, cx, l);
            int64_t h;
            if (l == l1) h = i1; else if (l == l2) h = i2; else if (l == l3) h = i3;
            else h = closest_hit(hx, zoff[l], zoff[l + 1], xp, C->tol_x);
            if (h < 0) { cd.hit[s] = NO_HIT; pattern = 1 + s; r[s] = 0; }
            else { cd.hit[s] = (uint32_t)h; r[s] = hx[h] - xp; nx++; }
          }
          if (nx < C->g.min_x_hits) continue;
          cnt[C_EXT_OK]++;
          chi2 = fit_xz(C, pattern, r, nx, &ax, &bx, &cx);                      /* O6 */
          if (chi2 > C->chi2x_max) continue;
          cnt[C_FIT_OK]++;
          cd.ax = ax; cd.bx = bx; cd.cx = cx; cd.chi2 = chi2; cd.nx = nx; cd.it = it;
          cd.key = clone_key(chi2, cx, nx, it); cd.keep = 0;
          PUSH(cands, cd);
        }
      }
    }
  }
  clone_kill(cands->p + cand0, cands->n - cand0, zoff[0], zoff[NL] - zoff[0]);  /* O7, A11 */

  for (ci = cand0; ci < cands->n; ci++) {                                       /* O8 */
    const cand_t* cd = &cands->p[ci];
    REAL xp[NX];
    int pp, best_n = 0, have = 0; REAL best_chi2 = 0, best_ay = 0, best_by = 0; uint32_t best_hit[NX];
    if (!cd->keep) continue;
    cnt[C_XZ_KEPT]++;
    for (s = 0; s < NX; s++) xp[s] = xz_at(C, cd->ax, cd->bx, cd->cx, C->ul[s]);
    if (C->uv_hough) {
      /* O8h (L217, reading A20): one-dimensional Hough transform in t_y over all six stereo layers.
       * Every hit inside its layer's window (Eq. 16, the half's y range) votes for the bin of t_y = y / z;
       * a layer counts once per bin ("bitwise").  A cluster is a bin together with its upper neighbour; its
       * population is the number of layers with a vote in it.  Up to eight clusters with population >=
       * min_uv_hits are taken, most populated first (then lower t_y); each is cut into four finer t_y
       * hypotheses; per hypothesis the closest hit within tol_uv (2 mm) of the straight line is attached in
       * every layer; fit and choice of the best combination as in the iterative version. */
      uint64_t vote[NX]; int pop[64], sel[8], nsel = 0, b, level, r, k;
      for (s = 0; s < NX; s++) {
        int l = C->ul[s]; uint32_t ih;
        REAL wa = xp[s] - C->ywin_a[half][l], wb = xp[s] - C->ywin_b[half][l];
        REAL wlo = rmin(wa, wb), whi = rmax(wa, wb);
        vote[s] = 0;
        for (ih = zoff[l]; ih < zoff[l + 1]; ih++) {
          REAL xh = hx[ih], t, tb;
          if (!(wlo <= xh && xh <= whi)) continue;
          cnt[C_UV_FIRST]++;
          t = ((xp[s] - xh) * C->inv_tan[l]) * C->inv_z[l];                     /* Eq. 16, A7 */
          tb = (t - C->hough_tlo[half]) * C->hough_invw;
          tb = rmin(rmax(tb, (REAL)0), (REAL)63);
          vote[s] |= (uint64_t)1 << (int)tb;
        }
      }
      for (b = 0; b < 64; b++) {
        pop[b] = 0;
        for (s = 0; s < NX; s++)
          pop[b] += (int)(((vote[s] >> b) & 1) | (b < 63 ? (vote[s] >> (b + 1)) & 1 : 0));
      }
      for (level = NX; level >= C->g.min_uv_hits && level >= 1; level--)
        for (b = 0; b < 64; b++)
          if (pop[b] == level && nsel < 8) sel[nsel++] = b;
      for (r = 0; r < nsel; r++)
        for (k = 0; k < 4; k++) {
          REAL f = (REAL)k * (REAL)0.5 + (REAL)0.25;
          REAL ty = C->hough_tlo[half] + ((REAL)sel[r] + f) * C->hough_w;
          REAL m[NX], ay, by, chi2y; uint32_t hit[NX]; int n = 0, mask = 0;
          for (s = 0; s < NX; s++) {
            int l = C->ul[s]; REAL xe; int64_t h;
            cnt[C_UV_STEPS]++;
            hit[s] = NO_HIT;
            xe = xp[s] - ty * C->zt[l];
            h = closest_hit(hx, zoff[l], zoff[l + 1], xe, C->tol_uv);           /* L217: the same 2 mm */
            if (h >= 0) { hit[s] = (uint32_t)h; m[s] = hx[h] - xp[s]; mask |= 1 << s; n++; }
          }
          if (n < C->g.min_uv_hits) continue;
          cnt[C_YFITS]++;
          chi2y = fit_y(C, mask, m, n, &ay, &by);
          if (chi2y > C->chi2y_max) continue;
          if (!have || n > best_n || (n == best_n && chi2y < best_chi2)) {      /* ties: earlier (cluster, k) */
            have = 1; best_n = n; best_chi2 = chi2y; best_ay = ay; best_by = by;
            memcpy(best_hit, hit, sizeof(hit));
          }
        }
    } else
    for (pp = 0; pp < 2; pp++) {
      int lf = C->g.uv_first_layer[pp], sf = C->slot_of_layer[lf];
      REAL wa = xp[sf] - C->ywin_a[half][lf], wb = xp[sf] - C->ywin_b[half][lf];
      REAL wlo = rmin(wa, wb), whi = rmax(wa, wb);
      uint32_t ih;
      for (ih = zoff[lf]; ih < zoff[lf + 1]; ih++) {
        REAL xh = hx[ih], y0, ty, m[NX], ay, by, chi2y; uint32_t hit[NX]; int n = 1, mask;
        if (!(wlo <= xh && xh <= whi)) continue;
        cnt[C_UV_FIRST]++;
        y0 = (xp[sf] - xh) * C->inv_tan[lf];                                    /* Eq. 16 */
        ty = y0 * C->inv_z[lf];                                                 /* A7 */
        for (s = 0; s < NX; s++) hit[s] = NO_HIT;
        hit[sf] = ih; m[sf] = xh - xp[sf]; mask = 1 << sf;
        for (s = 0; s < NX; s++) {
          int l = C->ul[s]; REAL xe; int64_t h;
          if (s == sf) continue;
          cnt[C_UV_STEPS]++;
          xe = xp[s] - ty * C->zt[l];
          h = closest_hit(hx, zoff[l], zoff[l + 1], xe, C->tol_uv);             /* L215: 2 mm */
          if (h >= 0) {
            REAL yl = (xp[s] - hx[h]) * C->inv_tan[l];
            ty = (REAL)0.5 * (ty + yl * C->inv_z[l]);                           /* A7: running average */
            hit[s] = (uint32_t)h; m[s] = hx[h] - xp[s]; mask |= 1 << s; n++;
          }
        }
        if (n < C->g.min_uv_hits) continue;
        cnt[C_YFITS]++;
        chi2y = fit_y(C, mask, m, n, &ay, &by);                                 /* O9 */
        if (chi2y > C->chi2y_max) continue;
        /* max n, then min chi2y, then earlier pass, then lower first-hit index: the scan order is
         * (pass, first hit) ascending, so "strictly better" keeps the earliest on ties */
        if (!have || n > best_n || (n == best_n && chi2y < best_chi2)) {
          have = 1; best_n = n; best_chi2 = chi2y; best_ay = ay; best_by = by;
          memcpy(best_hit, hit, sizeof(hit));
        }
      }
    }
    if (!have) continue;                                    /* fake x-z projection (L219) */
    {                                                       /* O10 */
      seed_t sd; REAL q;
      sd.event = event; sd.half = half; sd.nx = cd->nx; sd.nuv = best_n;
      sd.st[0] = (cd->ax + cd->bx * C->zbS) + cd->cx * C->gS;
      sd.st[1] = best_ay + best_by * C->zbS;
      sd.st[2] = cd->bx + cd->cx * C->gpS;
      sd.st[3] = best_by;
      q = cd->cx * C->inv_kappa;
      sd.st[4] = pol > 0 ? q : -q;
      sd.par[0] = cd->ax; sd.par[1] = cd->bx; sd.par[2] = cd->cx; sd.par[3] = best_ay; sd.par[4] = best_by;
      sd.par[5] = cd->chi2; sd.par[6] = best_chi2;
      for (s = 0; s < NL; s++) sd.hit[s] = NO_HIT;
      for (s = 0; s < NX; s++) { sd.hit[C->xl[s]] = cd->hit[s]; sd.hit[C->ul[s]] = best_hit[s]; }
      PUSH(seeds, sd);
      cnt[C_SEEDS]++;
    }
  }
}

/* Seeding over a batch.  Returns the number of seeds found (may exceed cap; only cap are written).
 * Outputs are row-major: state[n][5], par[n][7], hits[n][12]. */
int64_t orc_seeding(const orc_ctx* C, int n_events, const uint32_t* zone_off, const REAL* hit_x,
                    const int8_t* polarity, int64_t cap, int32_t* o_event, int32_t* o_half, REAL* o_state,
                    REAL* o_par, uint32_t* o_hits, uint8_t* o_nx, uint8_t* o_nuv, uint64_t* counters) {
  vcand cands = { 0 }; vseed seeds = { 0 };
  uint64_t cnt[C_N] = { 0 };
  int e, h; size_t i; int64_t n;
  for (e = 0; e < n_events; e++)
    for (h = 0; h < 2; h++) {
      cands.n = 0;
      seed_half(C, zone_off + (size_t)(e * 2 + h) * NL, hit_x, polarity ? polarity[e] : C->g.polarity, e, h,
                NULL, &cands, &seeds, cnt);
    }
  n = (int64_t)seeds.n;
  for (i = 0; i < seeds.n && (int64_t)i < cap; i++) {
    const seed_t* s = &seeds.p[i];
    o_event[i] = s->event; o_half[i] = s->half; o_nx[i] = (uint8_t)s->nx; o_nuv[i] = (uint8_t)s->nuv;
    memcpy(o_state + 5 * i, s->st, sizeof(s->st)); memcpy(o_par + 7 * i, s->par, sizeof(s->par));
    memcpy(o_hits + NL * i, s->hit, sizeof(s->hit));
  }
  if (counters) for (i = 0; i < C_N; i++) counters[i] += cnt[i];
  free(cands.p); free(seeds.p);
  return n;
}

/* Debug capture of one event-half: triplets (it, i1, i2, i3 global indices) and x-z candidates
 * (before the clone kill, with the keep flag). Returns counts through n_trip / n_cand. */
void orc_seeding_debug(const orc_ctx* C, const uint32_t* zone_off, const REAL* hit_x, int event, int half,
                       int64_t cap_t, int64_t* n_trip, int32_t* t_it, uint32_t* t_idx /* [cap][3] = i1,i2,i3 */,
                       int64_t cap_c, int64_t* n_cand, REAL* c_par /* [cap][4] ax,bx,cx,chi2 */,
                       uint32_t* c_hits /* [cap][6] */, int32_t* c_nx, int32_t* c_it, uint64_t* c_key,
                       int32_t* c_keep) {
  vtrip trips = { 0 }; vcand cands = { 0 }; vseed seeds = { 0 };
  uint64_t cnt[C_N] = { 0 }; size_t i;
  seed_half(C, zone_off + (size_t)(event * 2 + half) * NL, hit_x, C->g.polarity, event, half, &trips, &cands,
            &seeds, cnt);
  *n_trip = (int64_t)trips.n; *n_cand = (int64_t)cands.n;
  for (i = 0; i < trips.n && (int64_t)i < cap_t; i++) {
    t_it[i] = trips.p[i].it; t_idx[3 * i] = trips.p[i].i1; t_idx[3 * i + 1] = trips.p[i].i2; t_idx[3 * i + 2] = trips.p[i].i3;
  }
  for (i = 0; i < cands.n && (int64_t)i < cap_c; i++) {
    const cand_t* c = &cands.p[i];
    c_par[4 * i] = c->ax; c_par[4 * i + 1] = c->bx; c_par[4 * i + 2] = c->cx; c_par[4 * i + 3] = c->chi2;
    memcpy(c_hits + NX * i, c->hit, sizeof(c->hit));
    c_nx[i] = c->nx; c_it[i] = c->it; c_key[i] = c->key; c_keep[i] = c->keep;
  }
  free(trips.p); free(cands.p); free(seeds.p);
}

/* ------------------------------------------------------------------------------------------ */
/* Matching */
typedef struct { REAL dx, dy, dtx, dty, zm, chi2; int presel; } pair_t;

/* O11 + O12 for one (seed, VELO) pair */
static pair_t match_pair(const orc_ctx* C, const REAL* sd /* x,y,tx,ty */, REAL xV, REAL yV, REAL txV, REAL tyV) {
  pair_t r;
  REAL dtx = sd[2] - txV, dty = sd[3] - tyV, adtx = rabs(dtx);
  REAL zm = (((C->mag[0] + C->mag[1] * adtx) + C->mag[2] * (dtx * dtx)) + C->mag[3] * rabs(sd[0]))
            + C->mag[4] * (txV * txV);                                          /* Eq. 18 */
  REAL xs = sd[0] + (zm - C->zS) * sd[2], xv = xV + (zm - C->zV) * txV;         /* Eq. 17 */
  REAL ys = sd[1] + C->dzyS * sd[3], yv = yV + C->dzyV * tyV;                   /* L231 */
  r.dtx = dtx; r.dty = dty; r.zm = zm; r.dx = xs - xv; r.dy = ys - yv; r.chi2 = 0;
  r.presel = rabs(r.dx) < C->presel[0] && rabs(r.dy) < C->presel[1] && adtx < C->presel[2]
             && rabs(dty) < C->presel[3];                                       /* Eq. 21 */
  if (r.presel) {
    REAL tolx = C->cx0 + C->cx1 * (dtx * dtx);                                  /* Eq. 23 */
    REAL toly = C->cy0 + C->cy1 * (txV * txV + tyV * tyV);
    r.chi2 = (((r.dx * r.dx) / tolx + (r.dy * r.dy) / toly) + (dtx * dtx) * C->inv_tol_tx)
             + (dty * dty) * C->inv_tol_ty;                                     /* Eq. 22 */
  }
  return r;
}

static REAL ut_window(const orc_ctx* C, int layer, int tight, REAL invpG) {
  const REAL* w = tight ? C->ut_tight[layer] : C->ut_loose[layer];
  return rmin(rmax(w[0] + w[1] * invpG, w[2]), w[3]);                           /* L315 */
}

typedef struct { int n; uint32_t idx[NUT]; REAL gamma, ssq; } uthyp_t;

/* O13.  ut_off: the 5 offsets of this event's UT layers.  q0 = dtx / K_B (A10). */
static int ut_search(const orc_ctx* C, REAL xV, REAL yV, REAL txV, REAL tyV, REAL q0, const uint32_t* ut_off,
                     const REAL* ux, const REAL* uylo, const REAL* uyhi, uthyp_t* best, uint64_t* cnt) {
  REAL invpG = rabs(q0) * (REAL)1000;                       /* Table 2 is in GeV */
  REAL gamma0 = C->Ag + C->Bg * q0;                         /* Eq. 20 (polarity cancels) */
  int i0, have = 0;
  for (i0 = 0; i0 < NUT; i0++) {                            /* loose search, layer by layer (L309-311) */
    REAL yi = yV + tyV * C->ut_dz[i0];
    REAL xi = (xV + txV * C->ut_dz[i0]) + gamma0 * C->ut_dz2[i0];               /* Eq. 19 */
    REAL x0e = xi - yi * C->ut_tan[i0];
    REAL w = ut_window(C, i0, 0, invpG);
    REAL lo = x0e - w, hi = x0e + w;
    uint32_t j; int found = 0;
    if (NUT - i0 < C->g.min_ut_hits) break;                 /* cannot reach min_ut_hits any more (A12) */
    cnt[C_UT_STEPS]++;
    for (j = ut_off[i0]; j < ut_off[i0 + 1]; j++) {
      uthyp_t h; REAL num, den, dj[NUT], gam; int i, k;
      if (!(lo <= ux[j] && ux[j] <= hi)) continue;
      if (!(uylo[j] - C->ut_y_tol <= yi && yi <= uyhi[j] + C->ut_y_tol)) continue;
      found = 1; cnt[C_UT_HYP]++;
      /* every loose-window hit starts a hypothesis (A13) */
      for (k = 0; k < NUT; k++) h.idx[k] = NO_HIT;
      h.n = 1; h.idx[i0] = j;
      dj[i0] = ((ux[j] + yi * C->ut_tan[i0]) - xV) - txV * C->ut_dz[i0];
      num = dj[i0] * C->ut_dz2[i0]; den = C->ut_dz4[i0];
      gam = num / den;                                      /* refit gamma_x (L309) */
      for (i = i0 + 1; i < NUT; i++) {                      /* tight windows (L309) */
        REAL yt = yV + tyV * C->ut_dz[i];
        REAL xt = (xV + txV * C->ut_dz[i]) + gam * C->ut_dz2[i];
        REAL xe = xt - yt * C->ut_tan[i];
        REAL wt = ut_window(C, i, 1, invpG), tlo = xe - wt, thi = xe + wt, bd = 0;
        int64_t bj = -1; uint32_t jj;
        cnt[C_UT_STEPS]++;
        for (jj = ut_off[i]; jj < ut_off[i + 1]; jj++) {
          REAL dd;
          if (!(tlo <= ux[jj] && ux[jj] <= thi)) continue;
          if (!(uylo[jj] - C->ut_y_tol <= yt && yt <= uyhi[jj] + C->ut_y_tol)) continue;
          dd = rabs(ux[jj] - xe);
          if (bj < 0 || dd < bd) { bj = jj; bd = dd; }      /* closest; ties -> lower index */
        }
        if (bj >= 0) {
          h.idx[i] = (uint32_t)bj; h.n++;
          dj[i] = ((ux[bj] + yt * C->ut_tan[i]) - xV) - txV * C->ut_dz[i];
          num = num + dj[i] * C->ut_dz2[i]; den = den + C->ut_dz4[i];
          gam = num / den;
        }
      }
      h.gamma = gam; h.ssq = 0;
      for (i = 0, k = 0; i < NUT; i++) if (h.idx[i] != NO_HIT) {
        REAL res = dj[i] - gam * C->ut_dz2[i];
        h.ssq = k ? h.ssq + res * res : res * res; k = 1;
      }
      /* best: max n, min ssq, lowest first-hit index (scan order ascending) */
      if (!have || h.n > best->n || (h.n == best->n && h.ssq < best->ssq)) { *best = h; have = 1; }
    }
    if (found) break;                                       /* the first layer with loose hits seeds the search */
  }
  return have && best->n >= C->g.min_ut_hits;
}

/* ---- ghost-killing network (L344-348; reading A14b) -------------------------------------
 * A fully connected network 8 -> 32 -> 1 on (z_match, dx, dy, dtx, dty, chi2_match, eta_VELO, nHits_SciFi)
 * gives the "ghost probability".  The paper fixes the shape and the inputs, not the activation, the input
 * scaling or the weights: hidden ReLU, output logistic, inputs standardised as (v - mu) * isig, all passed
 * in by the caller as one packed array
 *   nn = mu[8], isig[8], W1[32][8], b1[32], W2[32], b2, cut (0.8), margin (0.05)          (339 values).
 * exp and log are spelled out (same single-rounded operations on both sides of the parity test, no libm):
 *   exp(y) = 2^n * P6(r),  n = floor(y log2(e) + 1/2),  r = (y - n c1) - n c2   (Cody-Waite),  |y| <= 87
 *   log(x) = e ln2 + s (2 + s^2 (2/3 + s^2 (2/5 + s^2 (2/7 + s^2 2/9)))),  x = m 2^e, m in [sqrt(1/2), sqrt 2),
 *            s = (m - 1) / (m + 1)                                                                          */
#define NN_IN 8
#define NN_HID 32
#define NN_SIZE (NN_IN + NN_IN + NN_HID * NN_IN + NN_HID + NN_HID + 3)

static REAL spec_exp(REAL y) {
  REAL n, r, p;
  if (y > (REAL)87.0) y = (REAL)87.0;
  if (y < (REAL)-87.0) y = (REAL)-87.0;
  n = (REAL)floor((double)(y * (REAL)1.44269504f + (REAL)0.5));
  r = (y - n * (REAL)0.693359375f) - n * (REAL)-2.12194440e-4f;
  p = (REAL)(1.0f / 720.0f);
  p = p * r + (REAL)(1.0f / 120.0f);
  p = p * r + (REAL)(1.0f / 24.0f);
  p = p * r + (REAL)(1.0f / 6.0f);
  p = p * r + (REAL)0.5;
  p = p * r + (REAL)1.0;
  p = p * r + (REAL)1.0;
  return (REAL)ldexp((double)p, (int)n);                   /* exact: |n| <= 126 */
}

static REAL spec_log(REAL x) {
  int e; REAL m, s, s2, q;
  m = (REAL)frexp((double)x, &e);                           /* exact: x = m 2^e, m in [1/2, 1) */
  if (m < (REAL)0.70710678f) { m = m * (REAL)2.0; e -= 1; }
  s = (m - (REAL)1.0) / (m + (REAL)1.0);
  s2 = s * s;
  q = (REAL)(2.0f / 9.0f);
  q = q * s2 + (REAL)(2.0f / 7.0f);
  q = q * s2 + (REAL)(2.0f / 5.0f);
  q = q * s2 + (REAL)(2.0f / 3.0f);
  q = q * s2 + (REAL)2.0;
  return (REAL)e * (REAL)0.69314718f + s * q;
}

/* pseudorapidity of a VELO segment from its slopes: eta = ln((1 + sqrt(1 + rho^2)) / rho), rho = tan(theta) */
static REAL eta_velo(REAL tx, REAL ty) {
  REAL rho2 = tx * tx + ty * ty;
  REAL rho = (REAL)sqrt((double)rho2);                      /* correctly rounded in either precision */
  REAL sh = (REAL)sqrt((double)((REAL)1.0 + rho2));
  if (rho < (REAL)1e-6f) rho = (REAL)1e-6f;
  return spec_log(((REAL)1.0 + sh) / rho);
}

static REAL ghost_prob(const REAL* nn, const REAL* in /* [8] */) {
  const REAL *mu = nn, *isig = nn + NN_IN, *W1 = nn + 2 * NN_IN, *b1 = W1 + NN_HID * NN_IN, *W2 = b1 + NN_HID;
  REAL u[NN_IN], t = W2[NN_HID];                            /* b2 */
  int j, k;
  for (k = 0; k < NN_IN; k++) u[k] = (in[k] - mu[k]) * isig[k];
  for (j = 0; j < NN_HID; j++) {
    REAL h = b1[j];
    for (k = 0; k < NN_IN; k++) h = h + W1[j * NN_IN + k] * u[k];
    if (h < 0) h = 0;
    t = t + W2[j] * h;
  }
  return (REAL)1.0 / ((REAL)1.0 + spec_exp(-t));
}

typedef struct { int seed, velo; REAL chi2, qop, ghost; int n_ut; uint32_t ut[NUT]; int alive; } mcand_t;
typedef VEC(mcand_t) vmc;

/* A21: order of two seeds whose candidates tie exactly in chi2_match (twin seeds: bit-identical states from
 * duplicate hits at the same x).  The seed whose twelve hit indices (layer 0 first, NO_HIT = largest) come
 * first in lexicographic order wins; seeds without hit lists (or with equal ones) fall back to the seed index.
 * Unlike the index, the hit list does not depend on the order in which the seeds were written. */
static int seed_before(const uint32_t* seed_hits, int a, int b) {
  if (seed_hits) {
    int l;
    for (l = 0; l < NL; l++) {
      uint32_t ha = seed_hits[(size_t)a * NL + l], hb = seed_hits[(size_t)b * NL + l];
      if (ha != hb) return ha < hb;
    }
  }
  return a < b;
}

/* Matching over a batch.  Seeds: per-event offsets seed_off[n_events+1] into state[n][5].
 * ut_off may be NULL (no UT).  Returns number of long tracks (only cap written). */
static int64_t matching_impl(const orc_ctx* C, int n_events, const uint32_t* seed_off, const REAL* state,
                     const uint32_t* velo_off, const REAL* vx, const REAL* vy, const REAL* vtx, const REAL* vty,
                     const uint32_t* ut_off, const REAL* ux, const REAL* uylo, const REAL* uyhi,
                     const int8_t* polarity, int64_t cap, int32_t* o_event, uint32_t* o_seed, uint32_t* o_velo,
                     uint32_t* o_ut /* [n][4] */, uint8_t* o_nut, REAL* o_qop, REAL* o_chi2, uint64_t* counters,
                     const uint8_t* seed_nhits /* per seed, NULL = 12 */, const REAL* nn /* NULL = A14 */,
                     REAL* o_ghost /* may be NULL */, const uint32_t* seed_hits /* [n][12] or NULL (A21) */) {
  uint64_t cnt[C_N] = { 0 };
  vmc mc = { 0 };
  int64_t n_out = 0; int e; size_t i;
  int use_ut = C->g.ut_enabled && ut_off != NULL;
  for (e = 0; e < n_events; e++) {
    int pol = polarity ? polarity[e] : C->g.polarity;
    uint32_t s, v;
    mc.n = 0;
    for (s = seed_off[e]; s < seed_off[e + 1]; s++)
      for (v = velo_off[e]; v < velo_off[e + 1]; v++) {
        pair_t pr; mcand_t m; REAL q0; int k;
        cnt[C_SV_PAIRS]++;
        pr = match_pair(C, state + 5 * (size_t)s, vx[v], vy[v], vtx[v], vty[v]);
        if (!pr.presel) continue;
        cnt[C_PRESEL]++;
        if (!(pr.chi2 < C->chi2m_max)) continue;                                /* L301 */
        cnt[C_CHI2_OK]++;
        q0 = pr.dtx * C->inv_KB;                                                /* A10 */
        m.seed = (int)s; m.velo = (int)v; m.chi2 = pr.chi2; m.alive = 1; m.n_ut = 0; m.ghost = 0;
        m.qop = pol > 0 ? q0 : -q0;
        for (k = 0; k < NUT; k++) m.ut[k] = NO_HIT;
        if (use_ut) {
          uthyp_t h; REAL q1;
          if (!ut_search(C, vx[v], vy[v], vtx[v], vty[v], q0, ut_off + (size_t)e * NUT, ux, uylo, uyhi, &h, cnt))
            continue;                                                           /* L311 */
          m.n_ut = h.n; memcpy(m.ut, h.idx, sizeof(m.ut));
          q1 = (h.gamma - C->Ag) * C->inv_Bg;
          m.qop = pol > 0 ? q1 : -q1;
        }
        if (nn) {                                                               /* L346: ghost probability */
          REAL in[NN_IN];
          in[0] = pr.zm; in[1] = pr.dx; in[2] = pr.dy; in[3] = pr.dtx; in[4] = pr.dty; in[5] = pr.chi2;
          in[6] = eta_velo(vtx[v], vty[v]);
          in[7] = (REAL)(seed_nhits ? seed_nhits[s] : 12);
          m.ghost = ghost_prob(nn, in);
        }
        PUSH(&mc, m);
      }
    if (nn) {
      /* O14b (L348): keep ghost probability < cut; then a track that shares its VELO or its SciFi segment
       * with another kept track is removed if its ghost probability is at least `margin` higher */
      const REAL cut = nn[NN_SIZE - 2], margin = nn[NN_SIZE - 1];
      for (i = 0; i < mc.n; i++) if (!(mc.p[i].ghost < cut)) mc.p[i].alive = 0;
      for (i = 0; i < mc.n; i++) {
        size_t j;
        if (!mc.p[i].alive) continue;
        for (j = 0; j < mc.n; j++) {
          if (j == i || !mc.p[j].alive) continue;             /* alive is 1 or 2 for tracks that passed the cut */
          if (mc.p[j].seed != mc.p[i].seed && mc.p[j].velo != mc.p[i].velo) continue;
          if (mc.p[i].ghost >= mc.p[j].ghost + margin) mc.p[i].alive = 2;   /* mark only: the comparison set stays fixed */
        }
      }
    } else {
    /* O14 (A14): each seed keeps its min (chi2, velo) candidate ... */
    for (i = 0; i < mc.n; i++) {
      size_t j;
      for (j = 0; j < mc.n; j++) {
        if (j == i || mc.p[j].seed != mc.p[i].seed) continue;
        if (mc.p[j].chi2 < mc.p[i].chi2 || (mc.p[j].chi2 == mc.p[i].chi2 && mc.p[j].velo < mc.p[i].velo))
          mc.p[i].alive = 0;
      }
    }
    /* ... then each VELO keeps the min (chi2, seed) among the survivors */
    for (i = 0; i < mc.n; i++) {
      size_t j; int lose = 0;
      if (!mc.p[i].alive) continue;
      for (j = 0; j < mc.n; j++) {
        if (j == i || !mc.p[j].alive || mc.p[j].velo != mc.p[i].velo) continue;
        if (mc.p[j].chi2 < mc.p[i].chi2 ||
            (mc.p[j].chi2 == mc.p[i].chi2 && seed_before(seed_hits, mc.p[j].seed, mc.p[i].seed)))
          lose = 1;
      }
      if (lose) mc.p[i].alive = 2;                          /* mark, do not change the survivor set mid-pass */
    }
    }
    for (i = 0; i < mc.n; i++) {
      const mcand_t* m = &mc.p[i];
      if (m->alive != 1) continue;
      cnt[C_LONG]++;
      if (n_out < cap) {
        o_event[n_out] = e; o_seed[n_out] = (uint32_t)m->seed; o_velo[n_out] = (uint32_t)m->velo;
        memcpy(o_ut + NUT * n_out, m->ut, sizeof(m->ut)); o_nut[n_out] = (uint8_t)m->n_ut;
        o_qop[n_out] = m->qop; o_chi2[n_out] = m->chi2;
        if (o_ghost) o_ghost[n_out] = m->ghost;
      }
      n_out++;
    }
  }
  if (counters) for (i = 0; i < C_N; i++) counters[i] += cnt[i];
  free(mc.p);
  return n_out;
}

int64_t orc_matching(const orc_ctx* C, int n_events, const uint32_t* seed_off, const REAL* state,
                     const uint32_t* velo_off, const REAL* vx, const REAL* vy, const REAL* vtx, const REAL* vty,
                     const uint32_t* ut_off, const REAL* ux, const REAL* uylo, const REAL* uyhi,
                     const int8_t* polarity, int64_t cap, int32_t* o_event, uint32_t* o_seed, uint32_t* o_velo,
                     uint32_t* o_ut /* [n][4] */, uint8_t* o_nut, REAL* o_qop, REAL* o_chi2, uint64_t* counters,
                     const uint32_t* seed_hits /* [n][12] or NULL: tie-break of reading A21 */) {
  return matching_impl(C, n_events, seed_off, state, velo_off, vx, vy, vtx, vty, ut_off, ux, uylo, uyhi, polarity, cap,
                       o_event, o_seed, o_velo, o_ut, o_nut, o_qop, o_chi2, counters, NULL, NULL, NULL, seed_hits);
}

/* The same with the ghost-killing network in place of the chi2 ranking (A14b).  nn: NN_SIZE packed values. */
int64_t orc_matching_nn(const orc_ctx* C, int n_events, const uint32_t* seed_off, const REAL* state,
                        const uint32_t* velo_off, const REAL* vx, const REAL* vy, const REAL* vtx, const REAL* vty,
                        const uint32_t* ut_off, const REAL* ux, const REAL* uylo, const REAL* uyhi,
                        const int8_t* polarity, int64_t cap, int32_t* o_event, uint32_t* o_seed, uint32_t* o_velo,
                        uint32_t* o_ut, uint8_t* o_nut, REAL* o_qop, REAL* o_chi2, uint64_t* counters,
                        const uint8_t* seed_nhits, const REAL* nn, REAL* o_ghost) {
  return matching_impl(C, n_events, seed_off, state, velo_off, vx, vy, vtx, vty, ut_off, ux, uylo, uyhi, polarity, cap,
                       o_event, o_seed, o_velo, o_ut, o_nut, o_qop, o_chi2, counters, seed_nhits, nn, o_ghost, NULL);
}

/* Hough-cluster UV seeding (reading A20) on / off; the default is the iterative version (L204) */
void orc_set_uv_hough(orc_ctx* C, int on) { C->uv_hough = on ? 1 : 0; }
void orc_hough_constants(const orc_ctx* C, double* out /* tlo0, tlo1, w, invw */) {
  out[0] = C->hough_tlo[0]; out[1] = C->hough_tlo[1]; out[2] = C->hough_w; out[3] = C->hough_invw;
}

/* probes of the network arithmetic (pins) */
double orc_spec_exp(double y) { return (double)spec_exp((REAL)y); }
double orc_spec_log(double x) { return (double)spec_log((REAL)x); }
double orc_eta_velo(double tx, double ty) { return (double)eta_velo((REAL)tx, (REAL)ty); }
double orc_ghost_prob(const double* nn, const double* in) {
  REAL w[NN_SIZE], v[NN_IN]; int i;
  for (i = 0; i < NN_SIZE; i++) w[i] = (REAL)nn[i];
  for (i = 0; i < NN_IN; i++) v[i] = (REAL)in[i];
  return (double)ghost_prob(w, v);
}

/* ------------------------------------------------------------------------------------------ */
/* Thin exported probes of the very functions used above (for the pins in tests/). */
void orc_constants(const orc_ctx* C, double* out /* [16] */) {
  int it;
  for (it = 0; it < 2; it++) {
    out[it] = C->dx3max[it]; out[2 + it] = C->alpha_corr[it]; out[4 + it] = C->K[it]; out[6 + it] = C->r13[it];
  }
}
void orc_pinv_xz(const orc_ctx* C, int pattern, double* out /* [3][6] */) {
  int k, s; for (k = 0; k < 3; k++) for (s = 0; s < NX; s++) out[k * NX + s] = C->P[pattern][k][s];
}
void orc_pinv_y(const orc_ctx* C, int mask, double* out /* [2][6] */) {
  int k, s; for (k = 0; k < 2; k++) for (s = 0; s < NX; s++) out[k * NX + s] = C->Q[mask][k][s];
}
void orc_momentum(const orc_ctx* C, int it, double x1, double x3, double* out /* t13,x0,s,invp,x2c,lo2,hi2 */) {
  REAL X1 = (REAL)x1, X3 = (REAL)x3;
  REAL t13 = (X3 - X1) * C->inv_dz13[it], x0 = X1 - C->z1[it] * t13;
  REAL s0 = x0 >= (REAL)0 ? (REAL)1 : (REAL)-1;
  REAL invp = C->a * rabs(x0) + C->b * (x0 * x0), x2c = X1 + C->dz12[it] * t13, kinv = C->kappa * invp;
  REAL cxp = s0 > 0 ? -kinv : kinv, ca = C->f_lo * cxp, cb = C->f_hi * cxp;
  REAL cxlo = rmin(ca, cb) - C->d_lo, cxhi = rmax(ca, cb) + C->d_hi;
  REAL e1 = x2c + C->K[it] * cxlo, e2 = x2c + C->K[it] * cxhi;
  out[0] = t13; out[1] = x0; out[2] = s0; out[3] = invp; out[4] = x2c; out[5] = rmin(e1, e2); out[6] = rmax(e1, e2);
}
void orc_parabola3(const orc_ctx* C, int it, double x1, double x2, double x3, double* out /* ax,bx,cx */) {
  REAL t, a, b, c; parabola3(C, it, (REAL)x1, (REAL)x2, (REAL)x3, &t, &a, &b, &c);
  out[0] = a; out[1] = b; out[2] = c;
}
/* fit of the x hits xs[6] (slot order; missing_slot = -1 for six hits) seeded from iteration `it`'s
 * three layers, exactly as O5+O6 do it.  out: ax,bx,cx,chi2 */
void orc_fit_xz(const orc_ctx* C, int it, const double* xs, int missing_slot, double* out) {
  REAL t, ax, bx, cx, r[NX]; int s, nx = 0, pattern = missing_slot < 0 ? 0 : 1 + missing_slot;
  parabola3(C, it, (REAL)xs[C->slot_of_layer[C->l1[it]]], (REAL)xs[C->slot_of_layer[C->l2[it]]],
            (REAL)xs[C->slot_of_layer[C->l3[it]]], &t, &ax, &bx, &cx);
  for (s = 0; s < NX; s++) {
    if (s == missing_slot) { r[s] = 0; continue; }
    r[s] = (REAL)xs[s] - xz_at(C, ax, bx, cx, C->xl[s]); nx++;
  }
  out[3] = fit_xz(C, pattern, r, nx, &ax, &bx, &cx);
  out[0] = ax; out[1] = bx; out[2] = cx;
}
/* y fit of measurement-space residuals m[6] (slot order) for the stereo slots in mask. out: ay,by,chi2 */
void orc_fit_y(const orc_ctx* C, int mask, const double* m, double* out) {
  REAL mm[NX], ay, by; int s, n = 0;
  for (s = 0; s < NX; s++) { mm[s] = (REAL)m[s]; if (mask >> s & 1) n++; }
  out[2] = fit_y(C, mask, mm, n, &ay, &by); out[0] = ay; out[1] = by;
}
uint64_t orc_clone_key(double chi2, double cx, int nx, int it) { return clone_key((REAL)chi2, (REAL)cx, nx, it); }
void orc_clone_kill(int n, const uint64_t* keys, const uint32_t* hits /* [n][6] */, const int32_t* nx,
                    uint32_t nhits, int32_t* keep) {
  cand_t* c = calloc(n ? n : 1, sizeof(cand_t)); int i;
  for (i = 0; i < n; i++) { c[i].key = keys[i]; c[i].nx = nx[i]; memcpy(c[i].hit, hits + NX * i, sizeof(c[i].hit)); }
  clone_kill(c, n, 0, nhits);
  for (i = 0; i < n; i++) keep[i] = c[i].keep;
  free(c);
}
void orc_match_pair(const orc_ctx* C, const double* seed4, const double* velo4, double* out /* dx,dy,dtx,dty,zm,chi2,presel */) {
  REAL sd[4] = { (REAL)seed4[0], (REAL)seed4[1], (REAL)seed4[2], (REAL)seed4[3] };
  pair_t r = match_pair(C, sd, (REAL)velo4[0], (REAL)velo4[1], (REAL)velo4[2], (REAL)velo4[3]);
  out[0] = r.dx; out[1] = r.dy; out[2] = r.dtx; out[3] = r.dty; out[4] = r.zm; out[5] = r.chi2; out[6] = r.presel;
}
double orc_ut_window(const orc_ctx* C, int layer, int tight, double invp_gev) { return ut_window(C, layer, tight, (REAL)invp_gev); }
double orc_gamma(const orc_ctx* C, double q0) { return C->Ag + C->Bg * (REAL)q0; }
/* UT search for one VELO state and kick estimate q0.  out: n, idx[4], gamma, ssq; returns accepted flag */
int orc_ut_search(const orc_ctx* C, const double* velo4, double q0, const uint32_t* ut_off, const REAL* ux,
                  const REAL* uylo, const REAL* uyhi, int32_t* o_n, uint32_t* o_idx, double* o_gamma, double* o_ssq) {
  uthyp_t h; uint64_t cnt[C_N] = { 0 }; int ok, k;
  memset(&h, 0, sizeof(h));
  for (k = 0; k < NUT; k++) h.idx[k] = NO_HIT;
  ok = ut_search(C, (REAL)velo4[0], (REAL)velo4[1], (REAL)velo4[2], (REAL)velo4[3], (REAL)q0, ut_off, ux, uylo, uyhi, &h, cnt);
  *o_n = h.n; memcpy(o_idx, h.idx, sizeof(h.idx)); *o_gamma = h.gamma; *o_ssq = h.ssq;
  return ok;
}
