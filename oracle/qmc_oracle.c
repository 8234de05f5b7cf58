/*
 * qmc_oracle.c -- ORACLE (test infrastructure, not the product; see qmc_oracle.h).
 *
 * Plain fp64 restatement of the crowd move of arXiv:2209.14487:
 *   Alg. 1 lines 4-9 for every walker of a crowd, lock-step in the
 *   electron index k (Alg. 3; Alg. 4).
 * The paper names the steps but prints no formula; BASELINE.json north_star names the
 * arithmetic, and each function below writes out the textbook definition it uses,
 * with the reading label of SURVEY.md 8(c) / DESIGN.md "Readings" (C1..C7, A1..A19).
 *
 * Deliberately naive: the 64-term triple sum for the spline, the full pair loop for
 * the Jastrow factor, LU for every small solve, no blocking, no fusion, no BLAS.
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC
 */
#include "qmc_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------------------------
 * C7. Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11): 10 rounds of
 *   (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)),
 * M0 = 0xD2511F53, M1 = 0xCD9E8D57, key bumped by (0x9E3779B9, 0xBB67AE85) between rounds.
 * Pinned by the Random123 known-answer vectors (tests/golden/philox4x32_10_kat.txt).
 * ---------------------------------------------------------------------------------- */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    if (round > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
    uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
    uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0;
    uint32_t n1 = lo1;
    uint32_t n2 = hi0 ^ c3 ^ k1;
    uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* C7: counter = (global walker id, electron k, sweep s, tag); key = (seed_lo, seed_hi).
 * u_i = (x_i + 0.5) * 2^-32 (exact in fp64, never 0 or 1). */
static double u01(uint32_t x) { return ((double)x + 0.5) * (1.0 / 4294967296.0); }

/* tag 0: three Gaussians by Box-Muller in fp64 (S8c C7):
 *   chi_x = sqrt(-2 ln u0) cos(2 pi u1), chi_y = sqrt(-2 ln u0) sin(2 pi u1),
 *   chi_z = sqrt(-2 ln u2) cos(2 pi u3). */
void oracle_rng_gauss3(uint64_t seed, uint32_t walker, uint32_t k, uint32_t sweep, double chi[3])
{
  const double two_pi = 6.283185307179586476925286766559;
  uint32_t ctr[4] = { walker, k, sweep, 0u };
  uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
  uint32_t x[4];
  oracle_philox4x32_10(ctr, key, x);
  double r0 = sqrt(-2.0 * log(u01(x[0])));
  double r1 = sqrt(-2.0 * log(u01(x[2])));
  chi[0] = r0 * cos(two_pi * u01(x[1]));
  chi[1] = r0 * sin(two_pi * u01(x[1]));
  chi[2] = r1 * cos(two_pi * u01(x[3]));
}

/* tag 1: the uniform of the accept/reject decision, u = (x0 + 0.5) 2^-32. */
double oracle_rng_uniform(uint64_t seed, uint32_t walker, uint32_t k, uint32_t sweep)
{
  uint32_t ctr[4] = { walker, k, sweep, 1u };
  uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
  uint32_t x[4];
  oracle_philox4x32_10(ctr, key, x);
  return u01(x[0]);
}

/* ------------------------------------------------------------------------------------
 * C1. Uniform cubic B-spline basis on [0,1): the four weights of the points i-1..i+2,
 * their first and second derivatives with respect to t (NOT yet divided by h, h^2).
 *   a0 = (1-t)^3/6   a1 = (3t^3-6t^2+4)/6   a2 = (-3t^3+3t^2+3t+1)/6   a3 = t^3/6
 * Pinned by: sum a = 1, sum a' = 0, sum m*a_m = t+1 (tests: partition of unity and
 * the linear-table closed form).
 * ---------------------------------------------------------------------------------- */
void oracle_bspline_weights(double t, double a[4], double da[4], double d2a[4])
{
  double t2 = t * t, t3 = t2 * t, omt = 1.0 - t;
  a[0] = omt * omt * omt / 6.0;
  a[1] = (3.0 * t3 - 6.0 * t2 + 4.0) / 6.0;
  a[2] = (-3.0 * t3 + 3.0 * t2 + 3.0 * t + 1.0) / 6.0;
  a[3] = t3 / 6.0;
  da[0] = -omt * omt / 2.0;
  da[1] = (3.0 * t2 - 4.0 * t) / 2.0;
  da[2] = (-3.0 * t2 + 2.0 * t + 1.0) / 2.0;
  da[3] = t2 / 2.0;
  d2a[0] = omt;
  d2a[1] = 3.0 * t - 2.0;
  d2a[2] = 1.0 - 3.0 * t;
  d2a[3] = t;
}

static double coef_at(const oracle_system* s, int64_t idx)
{
  return s->coef_dtype == 0 ? (double)((const float*)s->coefs)[idx] : ((const double*)s->coefs)[idx];
}

/* C1: phi_j(r) = sum_{a,b,c} A_a(tx) B_b(ty) C_c(tz) P[(ix-1+a) mod Ng][(iy-1+b) mod Ng][(iz-1+c) mod Ng][j]
 * with u = x*(Ng/L), i = floor(u), t = u - i; d/dx uses A'/h, Laplacian = sum of the three
 * pure second derivatives (orthorhombic cell, no mixed terms). Positions are not wrapped;
 * periodicity comes from the mod (A11). The plain 64-term sum, no factoring. */
void oracle_spo_vgl(const oracle_system* s, const double r[3], double* phi, double* dphi, double* d2phi)
{
  const int M = s->n_orb;
  double w[3][4], dw[3][4], d2w[3][4];
  int idx[3][4];
  for (int c = 0; c < 3; ++c) {
    const int Ng = s->grid[c];
    const double inv_h = (double)Ng / s->box[c];
    double u = r[c] * inv_h;
    double fl = floor(u);
    double t = u - fl;
    long long i = (long long)fl;
    oracle_bspline_weights(t, w[c], dw[c], d2w[c]);
    for (int m = 0; m < 4; ++m) {
      dw[c][m] *= inv_h;
      d2w[c][m] *= inv_h * inv_h;
      long long g = (i - 1 + m) % Ng;
      if (g < 0) g += Ng;
      idx[c][m] = (int)g;
    }
  }
  for (int j = 0; j < M; ++j) { phi[j] = 0.0; dphi[j] = 0.0; dphi[M + j] = 0.0; dphi[2 * M + j] = 0.0; d2phi[j] = 0.0; }
  for (int a = 0; a < 4; ++a)
    for (int b = 0; b < 4; ++b)
      for (int c = 0; c < 4; ++c) {
        const int64_t row = (((int64_t)idx[0][a] * s->grid[1] + idx[1][b]) * s->grid[2] + idx[2][c]) * (int64_t)M;
        const double wv = w[0][a] * w[1][b] * w[2][c];
        const double wx = dw[0][a] * w[1][b] * w[2][c];
        const double wy = w[0][a] * dw[1][b] * w[2][c];
        const double wz = w[0][a] * w[1][b] * dw[2][c];
        const double wl = d2w[0][a] * w[1][b] * w[2][c] + w[0][a] * d2w[1][b] * w[2][c] + w[0][a] * w[1][b] * d2w[2][c];
        for (int j = 0; j < M; ++j) {
          const double p = coef_at(s, row + j);
          phi[j] += wv * p;
          dphi[j] += wx * p;
          dphi[M + j] += wy * p;
          dphi[2 * M + j] += wz * p;
          d2phi[j] += wl * p;
        }
      }
}

/* ------------------------------------------------------------------------------------
 * C3. Two-body Jastrow, ln Psi_J = + sum_{i<j} u(r_ij), u(r) = a r/(1 + b r),
 * minimum image per component d_c <- d_c - L rint(d_c/L) (round-half-even), r = |d|.
 * ---------------------------------------------------------------------------------- */
static double min_image_dist(const oracle_system* s, const double a[3], const double b[3], double d[3])
{
  double r2 = 0.0;
  for (int c = 0; c < 3; ++c) {
    double dc = a[c] - b[c];
    dc -= s->box[c] * rint(dc / s->box[c]);
    d[c] = dc;
    r2 += dc * dc;
  }
  return sqrt(r2);
}

double oracle_j2_logpsi(const oracle_system* s, const double* R)
{
  double sum = 0.0, d[3];
  for (int i = 0; i < s->n_elec; ++i)
    for (int j = i + 1; j < s->n_elec; ++j) {
      double r = min_image_dist(s, R + 3 * i, R + 3 * j, d);
      sum += s->j2_a * r / (1.0 + s->j2_b * r);
    }
  return sum;
}

/* For electron k placed at rk (all other electrons at R): usum = sum_{i!=k} u(|rk - r_i|),
 * grad = grad_k ln Psi_J = sum_{i!=k} u'(r_ki) d_ki / r_ki, u'(r) = a/(1 + b r)^2.
 * rho_J of a move is exp(usum(r') - usum(r_k)). */
void oracle_j2_usum_grad(const oracle_system* s, const double* R, int k, const double rk[3],
                         double* usum, double grad[3])
{
  double sum = 0.0, g[3] = { 0.0, 0.0, 0.0 }, d[3];
  for (int i = 0; i < s->n_elec; ++i) {
    if (i == k) continue;
    double r = min_image_dist(s, rk, R + 3 * i, d);
    double den = 1.0 + s->j2_b * r;
    sum += s->j2_a * r / den;
    if (r > 0.0) {
      double du = s->j2_a / (den * den);
      for (int c = 0; c < 3; ++c) g[c] += du * d[c] / r;
    }
  }
  *usum = sum;
  grad[0] = g[0]; grad[1] = g[1]; grad[2] = g[2];
}

/* Kinetic part of the local energy (Alg. 1 line 11), atomic units:
 *   T(R) = -1/2 sum_k lap_k Psi / Psi,      lap_k Psi / Psi = lap_k ln Psi + |grad_k ln Psi|^2,
 * with ln Psi = ln D_up + ln D_dn + ln Psi_J (C4).  For electron k of spin block sigma, row b = B^sigma[k,:] of
 * the transposed inverse (C2) and the orbitals at r_k:
 *   grad_k ln D = sum_j b_j grad phi_j,     lap_k ln D = sum_j b_j lap phi_j - |grad_k ln D|^2,
 *   grad_k ln Psi_J = sum_{i!=k} u'(r) d/r,  lap_k ln Psi_J = sum_{i!=k} [u''(r) + 2 u'(r)/r],
 *   u = a r/(1 + b r), u' = a/(1 + b r)^2, u'' = -2 a b/(1 + b r)^3 (C3).
 * B_up, B_dn: [n][n] transposed inverses at R; e_elec: [N] per-electron terms or NULL.  Returns T. */
double oracle_kinetic_energy(const oracle_system* s, const double* R, const double* B_up, const double* B_dn,
                             double* e_elec)
{
  const int N = s->n_elec, n = N / 2, M = s->n_orb;
  double* phi = (double*)malloc(sizeof(double) * 5 * (size_t)M);
  double* dph = phi + M;
  double* d2ph = phi + 4 * (size_t)M;
  double total = 0.0;
  for (int k = 0; k < N; ++k) {
    const double* b = (k < n ? B_up : B_dn) + (size_t)(k % n) * n;
    oracle_spo_vgl(s, R + 3 * k, phi, dph, d2ph);
    double gd[3] = { 0.0, 0.0, 0.0 }, ld = 0.0;
    for (int j = 0; j < M; ++j) {
      for (int c = 0; c < 3; ++c) gd[c] += b[j] * dph[(size_t)c * M + j];
      ld += b[j] * d2ph[j];
    }
    double lap_ln_d = ld - (gd[0] * gd[0] + gd[1] * gd[1] + gd[2] * gd[2]);
    double gj[3] = { 0.0, 0.0, 0.0 }, lap_ln_j = 0.0, d[3];
    for (int i = 0; i < N; ++i) {
      if (i == k) continue;
      double r = min_image_dist(s, R + 3 * k, R + 3 * i, d);
      if (r > 0.0) {
        double den = 1.0 + s->j2_b * r;
        double du = s->j2_a / (den * den);
        double d2u = -2.0 * s->j2_a * s->j2_b / (den * den * den);
        for (int c = 0; c < 3; ++c) gj[c] += du * d[c] / r;
        lap_ln_j += d2u + 2.0 * du / r;
      }
    }
    double g2 = 0.0;
    for (int c = 0; c < 3; ++c) g2 += (gd[c] + gj[c]) * (gd[c] + gj[c]);
    double ek = -0.5 * (lap_ln_d + lap_ln_j + g2);
    if (e_elec) e_elec[k] = ek;
    total += ek;
  }
  free(phi);
  return total;
}

/* ------------------------------------------------------------------------------------
 * LU with partial pivoting (Doolittle, row swaps), in place on a copy. Returns 0, or 4
 * (= "singular") when a pivot is zero or non-finite (A16).
 * ---------------------------------------------------------------------------------- */
static int lu_factor(int n, double* a, int* piv, int* sign)
{
  *sign = 1;
  for (int c = 0; c < n; ++c) {
    int p = c;
    double best = fabs(a[(size_t)c * n + c]);
    for (int r = c + 1; r < n; ++r) {
      double v = fabs(a[(size_t)r * n + c]);
      if (v > best) { best = v; p = r; }
    }
    piv[c] = p;
    if (!(best > 0.0) || !isfinite(best)) return 4;
    if (p != c) {
      for (int j = 0; j < n; ++j) {
        double tmp = a[(size_t)c * n + j];
        a[(size_t)c * n + j] = a[(size_t)p * n + j];
        a[(size_t)p * n + j] = tmp;
      }
      *sign = -*sign;
    }
    for (int r = c + 1; r < n; ++r) {
      double l = a[(size_t)r * n + c] / a[(size_t)c * n + c];
      a[(size_t)r * n + c] = l;
      for (int j = c + 1; j < n; ++j) a[(size_t)r * n + j] -= l * a[(size_t)c * n + j];
    }
  }
  return 0;
}

static void lu_solve(int n, const double* lu, const int* piv, double* x)
{
  for (int c = 0; c < n; ++c) {
    if (piv[c] != c) { double tmp = x[c]; x[c] = x[piv[c]]; x[piv[c]] = tmp; }
  }
  for (int r = 0; r < n; ++r)
    for (int j = 0; j < r; ++j) x[r] -= lu[(size_t)r * n + j] * x[j];
  for (int r = n - 1; r >= 0; --r) {
    for (int j = r + 1; j < n; ++j) x[r] -= lu[(size_t)r * n + j] * x[j];
    x[r] /= lu[(size_t)r * n + r];
  }
}

/* C2: B = (A^-1)^T, row-major, so that row k of B is "the moved electron's inverse-matrix
 * row" (BJ): row c of B solves A x = e_c. Also ln|det A| and its sign. */
int oracle_lu_inverse_transpose(int n, const double* A, double* B, double* logabsdet, int* sign)
{
  double* lu = (double*)malloc(sizeof(double) * (size_t)n * n);
  int* piv = (int*)malloc(sizeof(int) * (size_t)n);
  memcpy(lu, A, sizeof(double) * (size_t)n * n);
  int sg;
  int st = lu_factor(n, lu, piv, &sg);
  if (st == 0) {
    double la = 0.0;
    for (int i = 0; i < n; ++i) {
      double d = lu[(size_t)i * n + i];
      if (d < 0.0) sg = -sg;
      la += log(fabs(d));
    }
    if (logabsdet) *logabsdet = la;
    if (sign) *sign = sg;
    for (int c = 0; c < n; ++c) {
      double* x = B + (size_t)c * n;
      for (int j = 0; j < n; ++j) x[j] = (j == c) ? 1.0 : 0.0;
      lu_solve(n, lu, piv, x);
    }
  }
  free(lu); free(piv);
  return st;
}

/* C5: Sherman-Morrison in the B = A^-T convention, electron (row of A) k replaced by phi:
 *   b_old = B[k,:]; w_i = B[i,:].phi; B'[i,:] = B[i,:] - ((w_i - delta_ik)/rho_D) b_old,
 * rho_D = B[k,:].phi (matrix-determinant lemma). Pinned by full re-inversion. */
void oracle_sm_update(int n, double* B, int k, const double* phi, double rho_d)
{
  double* b_old = (double*)malloc(sizeof(double) * (size_t)n);
  memcpy(b_old, B + (size_t)k * n, sizeof(double) * (size_t)n);
  for (int i = 0; i < n; ++i) {
    double w = 0.0;
    for (int j = 0; j < n; ++j) w += B[(size_t)i * n + j] * phi[j];
    double f = (w - (i == k ? 1.0 : 0.0)) / rho_d;
    for (int j = 0; j < n; ++j) B[(size_t)i * n + j] -= f * b_old[j];
  }
  free(b_old);
}

/* R6 (mixed precision): the carried inverse is stored in fp32.  Storage only: the value kept is
 * the fp32 number nearest to the fp64 result (ties to even: the C conversion), widened again for every later use. */
void oracle_round_to_fp32(int n, double* B)
{
  for (size_t e = 0; e < (size_t)n * n; ++e) B[e] = (double)(float)B[e];
}

/* C6 (Woodbury): window of m accepted moves since the last flush: rows[l] = electron row
 * replaced by V[l,:] (m x n), C[l,:] = B0[rows[l],:] (m x n), S = V C^T (m x m).
 * Builds S and LU-factors it from scratch (no incremental inverse). */
static int window_factor(int n, int m, const double* V, const double* C, double* S, int* piv)
{
  for (int l = 0; l < m; ++l)
    for (int q = 0; q < m; ++q) {
      double s = 0.0;
      for (int j = 0; j < n; ++j) s += V[(size_t)l * n + j] * C[(size_t)q * n + j];
      S[(size_t)l * m + q] = s;
    }
  int sg;
  return lu_factor(m, S, piv, &sg);
}

/* Current row k of the transposed inverse with the window applied:
 *   p_l = V[l,:].B0[k,:] - [rows[l]==k];  b = B0[k,:] - C^T (S^-1 p). */
int oracle_delayed_row(int n, const double* B0, int m, const int32_t* rows, const double* V,
                       const double* C, int k, double* b)
{
  memcpy(b, B0 + (size_t)k * n, sizeof(double) * (size_t)n);
  if (m == 0) return 0;
  double* S = (double*)malloc(sizeof(double) * (size_t)m * m);
  int* piv = (int*)malloc(sizeof(int) * (size_t)m);
  double* p = (double*)malloc(sizeof(double) * (size_t)m);
  int st = window_factor(n, m, V, C, S, piv);
  if (st == 0) {
    for (int l = 0; l < m; ++l) {
      double s = 0.0;
      for (int j = 0; j < n; ++j) s += V[(size_t)l * n + j] * B0[(size_t)k * n + j];
      p[l] = s - (rows[l] == k ? 1.0 : 0.0);
    }
    lu_solve(m, S, piv, p);
    for (int l = 0; l < m; ++l)
      for (int j = 0; j < n; ++j) b[j] -= p[l] * C[(size_t)l * n + j];
  }
  free(S); free(piv); free(p);
  return st;
}

/* Flush: W = B0 V^T - E (E[rows[l]][l] = 1), T = W S^-T, B <- B0 - T C.  Row-local, so
 * done row by row in place. Pinned by full re-inversion. */
int oracle_delayed_flush(int n, double* B0, int m, const int32_t* rows, const double* V, const double* C)
{
  if (m == 0) return 0;
  double* S = (double*)malloc(sizeof(double) * (size_t)m * m);
  int* piv = (int*)malloc(sizeof(int) * (size_t)m);
  double* w = (double*)malloc(sizeof(double) * (size_t)m);
  int st = window_factor(n, m, V, C, S, piv);
  if (st == 0) {
    for (int i = 0; i < n; ++i) {
      double* bi = B0 + (size_t)i * n;
      for (int l = 0; l < m; ++l) {
        double s = 0.0;
        for (int j = 0; j < n; ++j) s += V[(size_t)l * n + j] * bi[j];
        w[l] = s - (rows[l] == i ? 1.0 : 0.0);
      }
      lu_solve(m, S, piv, w);              /* t_i = S^-1 w_i  <=>  T = W S^-T */
      for (int l = 0; l < m; ++l)
        for (int j = 0; j < n; ++j) bi[j] -= w[l] * C[(size_t)l * n + j];
    }
  }
  free(S); free(piv); free(w);
  return st;
}

/* ------------------------------------------------------------------------------------
 * C4. The move (Alg. 1 L5 and L9; readings A1-A3, A7).
 * Proposal: Delta = fl32(tau G_k(R) + sqrt(tau) chi) per component, r' = r_k + Delta (fp64).
 * ---------------------------------------------------------------------------------- */
void oracle_move_propose(double tau, const double rk[3], const double g_old[3], const double chi[3],
                         double delta[3], double rnew[3], double* disp_margin)
{
  double margin = INFINITY;
  const double sq = sqrt(tau);
  for (int c = 0; c < 3; ++c) {
    double x = tau * g_old[c] + sq * chi[c];
    float f = (float)x;
    delta[c] = (double)f;
    rnew[c] = rk[c] + delta[c];
    if (isfinite(f)) {
      double up = (double)nextafterf(f, INFINITY), dn = (double)nextafterf(f, -INFINITY);
      double ulp = up - (double)f;
      double m1 = 0.5 * ((double)f + up) - x, m2 = x - 0.5 * ((double)f + dn);
      double mm = (m1 < m2 ? m1 : m2) / ulp;
      if (mm < margin) margin = mm;
    }
  }
  if (disp_margin) *disp_margin = margin;
}

/* Acceptance: rho = rho_D rho_J; with the APPLIED Delta,
 *   logGf = -|Delta - tau G(R)|^2/(2 tau), logGb = -|-Delta - tau G(R')|^2/(2 tau),
 *   p = rho^2 exp(logGb - logGf); accept <=> u < p. Non-finite p or rho_D == 0 rejects.
 * VMC: sign changes of rho are allowed (A4). */
int oracle_move_accept(double tau, const double delta[3], const double g_old[3], const double g_new[3],
                       double rho_d, double rho_j, double u, double* p_out)
{
  double f2 = 0.0, b2 = 0.0;
  for (int c = 0; c < 3; ++c) {
    double f = delta[c] - tau * g_old[c];
    double b = -delta[c] - tau * g_new[c];
    f2 += f * f;
    b2 += b * b;
  }
  double log_gf = -f2 / (2.0 * tau), log_gb = -b2 / (2.0 * tau);
  double rho = rho_d * rho_j;
  double p = rho * rho * exp(log_gb - log_gf);
  if (p_out) *p_out = p;
  return (rho_d != 0.0 && isfinite(p) && u < p) ? 1 : 0;
}

/* ------------------------------------------------------------------------------------
 * The crowd. Per walker: positions, transposed inverses of both spins (B0 when a delayed
 * window is open), per-electron caches of grad phi and lap phi at the current position
 * (A12, A13), and the delayed window.
 * ---------------------------------------------------------------------------------- */
struct oracle_crowd {
  oracle_system sys;
  int W, N, n, M, kd;
  int walker_id0;
  uint32_t sweep;
  double* R;      /* [W][N][3]       */
  double* B;      /* [W][2][n][n]    */
  double* dphi;   /* [W][N][3][M]    */
  double* d2phi;  /* [W][N][M]       */
  double* V;      /* [W][kd][n]      */
  double* C;      /* [W][kd][n]      */
  int32_t* rows;  /* [W][kd]         */
  int32_t* m;     /* [W]             */
};

int oracle_num_threads(void)
{
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

void oracle_crowd_destroy(oracle_crowd* c)
{
  if (!c) return;
  free(c->R); free(c->B); free(c->dphi); free(c->d2phi); free(c->V); free(c->C); free(c->rows); free(c->m);
  free(c);
}

/* Builds A^s_ij = phi_j(r_{s n + i}) (C2) for both spins of every walker and inverts by LU. */
oracle_crowd* oracle_crowd_create(const oracle_system* sys, int W, int walker_id0, const double* pos, int* status)
{
  oracle_crowd* c = (oracle_crowd*)calloc(1, sizeof(oracle_crowd));
  c->sys = *sys;
  c->W = W; c->N = sys->n_elec; c->n = sys->n_elec / 2; c->M = sys->n_orb;
  c->kd = sys->delay_rank < 1 ? 1 : sys->delay_rank;
  c->walker_id0 = walker_id0;
  c->sweep = 0;
  const int N = c->N, n = c->n, M = c->M, kd = c->kd;
  int st_all = 0;
  if (M != n || N != 2 * n) { if (status) *status = 1; free(c); return NULL; }
  c->R = (double*)malloc(sizeof(double) * (size_t)W * N * 3);
  c->B = (double*)malloc(sizeof(double) * (size_t)W * 2 * n * n);
  c->dphi = (double*)malloc(sizeof(double) * (size_t)W * N * 3 * M);
  c->d2phi = (double*)malloc(sizeof(double) * (size_t)W * N * M);
  c->V = (double*)calloc((size_t)W * kd * n, sizeof(double));
  c->C = (double*)calloc((size_t)W * kd * n, sizeof(double));
  c->rows = (int32_t*)calloc((size_t)W * kd, sizeof(int32_t));
  c->m = (int32_t*)calloc((size_t)W, sizeof(int32_t));
  memcpy(c->R, pos, sizeof(double) * (size_t)W * N * 3);
#pragma omp parallel for schedule(dynamic) reduction(| : st_all)
  for (int w = 0; w < W; ++w) {
    double* A = (double*)malloc(sizeof(double) * (size_t)n * n);
    for (int s = 0; s < 2; ++s) {
      for (int i = 0; i < n; ++i) {
        int e = s * n + i;
        oracle_spo_vgl(&c->sys, c->R + ((size_t)w * N + e) * 3, A + (size_t)i * n,
                       c->dphi + ((size_t)w * N + e) * 3 * M, c->d2phi + ((size_t)w * N + e) * M);
      }
      st_all |= oracle_lu_inverse_transpose(n, A, c->B + ((size_t)w * 2 + s) * n * n, NULL, NULL);
      if (c->sys.inverse_fp32) oracle_round_to_fp32(n, c->B + ((size_t)w * 2 + s) * n * n);
    }
    free(A);
  }
  if (status) *status = st_all;
  return c;
}

int oracle_crowd_recompute(oracle_crowd* c)
{
  const int W = c->W, N = c->N, n = c->n, M = c->M;
  int st_all = 0;
  for (int w = 0; w < W; ++w)
    if (c->m[w] != 0) return -1;
#pragma omp parallel for schedule(dynamic) reduction(| : st_all)
  for (int w = 0; w < W; ++w) {
    double* A = (double*)malloc(sizeof(double) * (size_t)n * n);
    for (int s = 0; s < 2; ++s) {
      for (int i = 0; i < n; ++i) {
        int e = s * n + i;
        oracle_spo_vgl(&c->sys, c->R + ((size_t)w * N + e) * 3, A + (size_t)i * n,
                       c->dphi + ((size_t)w * N + e) * 3 * M, c->d2phi + ((size_t)w * N + e) * M);
      }
      st_all |= oracle_lu_inverse_transpose(n, A, c->B + ((size_t)w * 2 + s) * n * n, NULL, NULL);
      if (c->sys.inverse_fp32) oracle_round_to_fp32(n, c->B + ((size_t)w * 2 + s) * n * n);
    }
    free(A);
  }
  return st_all;
}

/* One sweep (k = 0..N-1) of one walker: Alg. 1 lines 4-9, steps a0..a5
 * of SURVEY.md 8(a). Walkers never interact, so running them one after the other gives
 * the lock-step result of Alg. 3/4. */
static int64_t walker_sweep(oracle_crowd* c, int w, uint32_t s, oracle_move_log* log)
{
  const oracle_system* sys = &c->sys;
  const int N = c->N, n = c->n, M = c->M, kd = c->kd;
  double* R = c->R + (size_t)w * N * 3;
  double* V = c->V + (size_t)w * kd * n;
  double* C = c->C + (size_t)w * kd * n;
  int32_t* rows = c->rows + (size_t)w * kd;
  int32_t* mw = c->m + w;
  double* b = (double*)malloc(sizeof(double) * (size_t)n);
  double* phi = (double*)malloc(sizeof(double) * (size_t)M * 5);
  double* dph = phi + M;
  double* d2ph = phi + 4 * (size_t)M;
  const uint32_t wid = (uint32_t)(c->walker_id0 + w);
  int64_t n_acc = 0;
  for (int k = 0; k < N; ++k) {
    const int spin = k / n, kk = k % n;
    double* B = c->B + ((size_t)w * 2 + spin) * n * n;
    double* dcache = c->dphi + ((size_t)w * N + k) * 3 * M;
    double* d2cache = c->d2phi + ((size_t)w * N + k) * M;
    oracle_move_log rec;
    memset(&rec, 0, sizeof(rec));
    /* current inverse row (window applied) */
    if (kd > 1) oracle_delayed_row(n, B, *mw, rows, V, C, kk, b);
    else memcpy(b, B + (size_t)kk * n, sizeof(double) * (size_t)n);
    /* a0: G_k(R) = grad_k ln D (cached grad phi at r_k, rho_D = 1) + grad_k ln Psi_J (A13) */
    double usum_old, gj_old[3];
    oracle_j2_usum_grad(sys, R, k, R + 3 * k, &usum_old, gj_old);
    for (int cc = 0; cc < 3; ++cc) {
      double g = 0.0;
      for (int j = 0; j < M; ++j) g += b[j] * dcache[(size_t)cc * M + j];
      rec.g_old[cc] = g + gj_old[cc];
    }
    double chi[3];
    oracle_rng_gauss3(sys->seed, wid, (uint32_t)k, s, chi);
    oracle_move_propose(sys->tau, R + 3 * k, rec.g_old, chi, rec.delta, rec.rnew, &rec.disp_margin);
    /* a1: orbitals at r' */
    oracle_spo_vgl(sys, rec.rnew, phi, dph, d2ph);
    /* a2: rho_D = b.phi', grad = (b.grad phi')/rho_D (C2); Jastrow ratio and gradient (C3) */
    double rho_d = 0.0;
    for (int j = 0; j < M; ++j) rho_d += b[j] * phi[j];
    double usum_new, gj_new[3];
    oracle_j2_usum_grad(sys, R, k, rec.rnew, &usum_new, gj_new);
    for (int cc = 0; cc < 3; ++cc) {
      double g = 0.0;
      for (int j = 0; j < M; ++j) g += b[j] * dph[(size_t)cc * M + j];
      rec.g_new[cc] = g / rho_d + gj_new[cc];
    }
    rec.rho_d = rho_d;
    rec.rho_j = exp(usum_new - usum_old);
    /* a3: Metropolis */
    rec.u = oracle_rng_uniform(sys->seed, wid, (uint32_t)k, s);
    rec.accepted = oracle_move_accept(sys->tau, rec.delta, rec.g_old, rec.g_new, rec.rho_d, rec.rho_j, rec.u, &rec.p);
    if (rec.accepted) {
      ++n_acc;
      for (int cc = 0; cc < 3; ++cc) R[3 * k + cc] = rec.rnew[cc];
      memcpy(dcache, dph, sizeof(double) * 3 * (size_t)M);
      memcpy(d2cache, d2ph, sizeof(double) * (size_t)M);
      if (kd > 1) {           /* a4': append to the window */
        memcpy(V + (size_t)(*mw) * n, phi, sizeof(double) * (size_t)n);
        memcpy(C + (size_t)(*mw) * n, B + (size_t)kk * n, sizeof(double) * (size_t)n);
        rows[*mw] = kk;
        ++*mw;
      } else {                /* a4: rank-1 */
        oracle_sm_update(n, B, kk, phi, rho_d);
        if (sys->inverse_fp32) oracle_round_to_fp32(n, B);   /* R6: stored in fp32 */
      }
    }
    /* a5: flush after every kd PROPOSED moves of a spin block and at its end (C6 schedule) */
    if (kd > 1 && (((kk + 1) % kd) == 0 || kk == n - 1)) {
      oracle_delayed_flush(n, B, *mw, rows, V, C);
      if (sys->inverse_fp32 && *mw > 0) oracle_round_to_fp32(n, B);   /* R6: stored in fp32 */
      *mw = 0;
    }
    if (log) log[k] = rec;
  }
  free(b); free(phi);
  return n_acc;
}

int64_t oracle_crowd_sweep(oracle_crowd* c, int n_sweeps, oracle_move_log* log)
{
  int64_t total = 0;
  for (int it = 0; it < n_sweeps; ++it) {
    const uint32_t s = c->sweep;
#pragma omp parallel for schedule(dynamic) reduction(+ : total)
    for (int w = 0; w < c->W; ++w)
      total += walker_sweep(c, w, s, log ? log + ((size_t)it * c->W + w) * c->N : NULL);
    c->sweep = s + 1;
  }
  return total;
}

void oracle_crowd_set_sweep_index(oracle_crowd* c, uint32_t s) { c->sweep = s; }

/* DMC branching, data movement only (Alg. 1 L13): walker slot w takes over every carried
 * quantity of slot src[w].  Written as the definition: a full copy of the old state, then a gather -- no
 * condition on src beyond its range.  Returns -1 for an entry outside [0, W) or an open delayed window. */
int oracle_crowd_branch(oracle_crowd* c, const int32_t* src)
{
  const size_t W = (size_t)c->W, N = (size_t)c->N, n = (size_t)c->n, M = (size_t)c->M;
  for (size_t w = 0; w < W; ++w)
    if (src[w] < 0 || src[w] >= c->W || c->m[w] != 0) return -1;
  const size_t sR = N * 3, sB = 2 * n * n, sD = N * 3 * M, sL = N * M;
  double* R0 = (double*)malloc(sizeof(double) * W * sR);
  double* B0 = (double*)malloc(sizeof(double) * W * sB);
  double* D0 = (double*)malloc(sizeof(double) * W * sD);
  double* L0 = (double*)malloc(sizeof(double) * W * sL);
  if (!R0 || !B0 || !D0 || !L0) { free(R0); free(B0); free(D0); free(L0); return -2; }
  memcpy(R0, c->R, sizeof(double) * W * sR);
  memcpy(B0, c->B, sizeof(double) * W * sB);
  memcpy(D0, c->dphi, sizeof(double) * W * sD);
  memcpy(L0, c->d2phi, sizeof(double) * W * sL);
  for (size_t w = 0; w < W; ++w) {
    const size_t s = (size_t)src[w];
    memcpy(c->R + w * sR, R0 + s * sR, sizeof(double) * sR);
    memcpy(c->B + w * sB, B0 + s * sB, sizeof(double) * sB);
    memcpy(c->dphi + w * sD, D0 + s * sD, sizeof(double) * sD);
    memcpy(c->d2phi + w * sL, L0 + s * sL, sizeof(double) * sL);
  }
  free(R0); free(B0); free(D0); free(L0);
  return 0;
}

void oracle_crowd_get_positions(const oracle_crowd* c, double* pos)
{
  memcpy(pos, c->R, sizeof(double) * (size_t)c->W * c->N * 3);
}

void oracle_crowd_get_inverse(const oracle_crowd* c, int spin, double* B)
{
  const size_t nn = (size_t)c->n * c->n;
  for (int w = 0; w < c->W; ++w)
    memcpy(B + (size_t)w * nn, c->B + ((size_t)w * 2 + spin) * nn, sizeof(double) * nn);
}
