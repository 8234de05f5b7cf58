// move.cuh -- the per-walker scalar side of a move: inverse row with the delayed window applied,
// drift-diffusion proposal, determinant/Jastrow ratio and gradient, Metropolis decision, window
// append (SURVEY 8(a) steps a0, a2, a3, a4').  One CTA of MOVE_NT threads per walker; all
// length-n / length-N sums are strided over the block and combined by shuffle reductions (BJ).
//
// The window kernel instantiates the shared blocks with NT = 128, 256 or 512 threads per walker (small crowds get
// wider CTAs, window.cuh); the step kernels use MOVE_NT.  Block sums depend on NT at the rounding level only.
//
// The building blocks below (row dots, axpy over window rows, the G_k(R)/proposal tail, ratio, decision)
// are shared by the three step kernels of the C ABI and by the walker-persistent window kernel of
// qmc_sweep (window.cuh), which is what makes the two paths bit-identical: same products, same
// summation trees; only where the operands live (global memory vs shared memory) differs.
#pragma once
#include "common.cuh"
#include "spline.cuh"

namespace qmc {

#ifndef QMC_MOVE_NT
#define QMC_MOVE_NT 128
#endif
constexpr int MOVE_NT = QMC_MOVE_NT;
constexpr int MOVE_NW = MOVE_NT / 32;
constexpr int MOVE_RED = 8 * MOVE_NW < 32 ? 32 : 8 * MOVE_NW;  // doubles of reduction scratch
constexpr int MOVE_MV = 16;                                     // doubles of per-move scalars (MoveScal)

// Per-move scalars of one walker.  The step kernels keep them in global memory (they cross kernel
// boundaries and feed qmc_crowd_get_move); the window kernel keeps them in shared memory.
struct MoveScal {
  double *rn, *delta, *g_old, *g_new;  // [3] each
  double *usum_old, *rho_d, *rho_j;    // [1] each
};
__device__ __forceinline__ MoveScal move_scal_global(const CrowdDev& d, int w)
{
  MoveScal s;
  s.rn = d.rnew + 3 * (size_t)w; s.delta = d.delta + 3 * (size_t)w;
  s.g_old = d.g_old + 3 * (size_t)w; s.g_new = d.g_new + 3 * (size_t)w;
  s.usum_old = d.usum_old + w; s.rho_d = d.rho_d + w; s.rho_j = d.rho_j + w;
  return s;
}
__device__ __forceinline__ MoveScal move_scal_smem(double* mv)
{
  MoveScal s;
  s.rn = mv; s.delta = mv + 3; s.g_old = mv + 6; s.g_new = mv + 9;
  s.usum_old = mv + 12; s.rho_d = mv + 13; s.rho_j = mv + 14;
  return s;
}

// D:C3: one pair term of the two-body Jastrow for electron k placed at rk against electron i.
// u(r) = a r/(1 + b r), u'(r) = a/(1 + b r)^2, minimum image d_c <- d_c - L rint(d_c/L).
__device__ __forceinline__ void j2_pair(const CrowdDev& d, const double (&rk)[3], const double* ri, double& usum,
                                        double (&g)[3])
{
  double dd[3], r2 = 0.0;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    double x = rk[c] - ri[c];
    x -= d.box[c] * rint(x * d.inv_box[c]);
    dd[c] = x;
    r2 = fma(x, x, r2);
  }
  if (r2 > 1e-280) {   // coincident electrons contribute nothing (D:C3); anything else is far inside the normal range
    const double inv_r = rsqrt_pos(r2);
    const double r = r2 * inv_r;
    const double inv_den = rcp_pos(fma(d.j2_b, r, 1.0));
    usum += d.j2_a * r * inv_den;
    const double f = d.j2_a * inv_den * inv_den * inv_r;
#pragma unroll
    for (int c = 0; c < 3; ++c) g[c] = fma(f, dd[c], g[c]);
  }
}

// Thread-strided partial J2 sums of electron k at rk against all other electrons of R [N][3].
template <int NT = MOVE_NT>
__device__ __forceinline__ void j2_partial(const CrowdDev& d, const double* R, int k, const double (&rk)[3], double& usum,
                                           double (&g)[3])
{
  for (int i = threadIdx.x; i < d.N; i += NT)
    if (i != k) j2_pair(d, rk, R + 3 * i, usum, g);
}

// store(l, row(l) . x) for l in [0, nrows) with row(l) != nullptr.  A warp takes RB rows at a time and
// keeps 3 RB 16-byte loads per lane in flight; per row the lane partial runs over the double2 columns
// lane, lane+32, ... in order and the 32 partials are combined by the xor-shuffle tree of warp_sum:
// the result does not depend on RB, on who calls it, or on where the operands live.
// row: int -> const double* (ns doubles, 16-byte aligned) or nullptr; x: int jj -> double2 (columns 2jj, 2jj+1).
template <int RB, typename RowF, typename XF, typename StoreF>
__device__ __forceinline__ void rows_dot(int nrows, int ns, RowF row, XF x, StoreF store)
{
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int l0 = warp * RB; l0 < nrows; l0 += MOVE_NW * RB) {
    const double2* rp[RB];
    double acc[RB];
#pragma unroll
    for (int r = 0; r < RB; ++r) {
      rp[r] = (l0 + r < nrows) ? reinterpret_cast<const double2*>(row(l0 + r)) : nullptr;
      acc[r] = 0.0;
    }
#pragma unroll 3
    for (int jj = lane; jj < ns / 2; jj += 32) {
      const double2 xv = x(jj);
      double2 v[RB];
#pragma unroll
      for (int r = 0; r < RB; ++r) v[r] = rp[r] ? rp[r][jj] : make_double2(0.0, 0.0);
#pragma unroll
      for (int r = 0; r < RB; ++r) acc[r] = fma(v[r].x, xv.x, fma(v[r].y, xv.y, acc[r]));
    }
#pragma unroll
    for (int r = 0; r < RB; ++r) {
      const double t = warp_sum(acc[r]);
      if (lane == 0 && rp[r]) store(l0 + r, t);
    }
  }
}

// b_s[j] -= sum_{l<m} y_s[l] row(l)[j]  (D:C6), a thread owns double2 columns tid, tid+NT, ...; rows in
// order per element, 16 loads in flight.
template <typename RowF>
__device__ __forceinline__ void axpy_rows(double* b_s, int ns, int m, const double* y_s, RowF row)
{
  for (int jj = threadIdx.x; jj < ns / 2; jj += MOVE_NT) {
    double2 acc = make_double2(b_s[2 * jj], b_s[2 * jj + 1]);
#pragma unroll 16
    for (int l = 0; l < m; ++l) {
      const double2 c = reinterpret_cast<const double2*>(row(l))[jj];
      acc.x = fma(-y_s[l], c.x, acc.x);
      acc.y = fma(-y_s[l], c.y, acc.y);
    }
    b_s[2 * jj] = acc.x;
    b_s[2 * jj + 1] = acc.y;
  }
}

// y_s[l] = sum_{q<m} Sinv[l ss + q] p_s[q] for l < m: one thread per l, q in order.
__device__ __forceinline__ void sinv_matvec(const double* Sinv, int ss, int m, const double* p_s, double* y_s)
{
  for (int l = threadIdx.x; l < m; l += MOVE_NT) {
    double y = 0.0;
#pragma unroll 8
    for (int q = 0; q < m; ++q) y = fma(Sinv[(size_t)l * ss + q], p_s[q], y);
    y_s[l] = y;
  }
}

// The five Box-Muller pieces of the Gaussians of move (walker w, electron k, current sweep) (D:C7):
// chi = (g0 g1, g0 g2, g3 g4), g0 = sqrt(-2 ln u0), g1 = cos 2 pi u1, g2 = sin 2 pi u1, g3 = sqrt(-2 ln u2),
// g4 = cos 2 pi u3.  Four lanes (part = 0..3) of one warp: parts 0 / 2 take the two radii, parts 1 / 3 the two angles
// (sincos: one argument reduction for g1 and g2), so the warp runs two code paths instead of five.  The pieces depend
// on nothing but the counter, so the window kernel computes them ahead of time, off the critical path.
// out[0..4] = g0..g4; callers synchronise before reading.
__device__ __forceinline__ void gauss_pieces(const CrowdDev& d, int w, int k, int part, double* out)
{
  unsigned x[4];
  philox4x32_10((unsigned)(d.walker_id0 + w), (unsigned)k, *d.sweep, 0u, d.seed_lo, d.seed_hi, x);
  const double two_pi = 6.283185307179586476925286766559;
  if ((part & 1) == 0) {
    out[part == 0 ? 0 : 3] = sqrt(-2.0 * log(u01(x[part])));
  } else {
    double sn, cs;
    sincos(two_pi * u01(x[part]), &sn, &cs);
    if (part == 1) { out[1] = cs; out[2] = sn; }
    else out[4] = cs;
  }
}

// ---- G_k(R) and the proposal (qmc_spo_vgl step (b)) -------------------------------------------
// G_k(R) = b . grad phi(r_k) [cache] + grad_k ln Psi_J(R)                       (D:C2, C3, A13)
// Delta = fl32(tau G + sqrt(tau) chi), r' = r_k + Delta, chi by Box-Muller      (D:C4, C7)
// b_s: the inverse row of electron k with the window applied (shared memory); cache: [4][ns] of
// electron k; R: positions [N][3] of the walker.  The five transcendental pieces of the Gaussians
// run on five threads (or arrive precomputed in gauss_pre[5]).  Threads 0..2 take one component each, write the
// results to ms and, if sw_out is given, the spline weights of their axis at r'; callers synchronise before reading.
template <typename T, int NT = MOVE_NT>
__device__ __forceinline__ void dev_gold_propose(const CrowdDev& d, int w, int k, const double* b_s, const T* cache,
                                                 const double* R, const double* rnew_given, MoveScal ms, double* red,
                                                 const double* gauss_pre = nullptr, SplineW<T>* sw_out = nullptr)
{
  const int ns = d.ns, tid = threadIdx.x;
  // v[0..2] = b . grad phi(r_k), v[3] = usum_old, v[4..6] = grad_k ln Psi_J(R)
  double v[7] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
  for (int j = tid; j < d.M; j += NT) {
    const double bj = b_s[j];
    v[0] = fma(bj, (double)cache[j], v[0]);
    v[1] = fma(bj, (double)cache[ns + j], v[1]);
    v[2] = fma(bj, (double)cache[2 * ns + j], v[2]);
  }
  const double rk[3] = {R[3 * k], R[3 * k + 1], R[3 * k + 2]};
  {
    double g[3] = {0.0, 0.0, 0.0};
    j2_partial<NT>(d, R, k, rk, v[3], g);
    v[4] = g[0]; v[5] = g[1]; v[6] = g[2];
  }
  block_sum_t0<7, NT>(v, red);
  if (!rnew_given && !gauss_pre) {
    if (tid < 4) gauss_pieces(d, w, k, tid, red);
    __syncthreads();
  }
  const double* gp = gauss_pre ? gauss_pre : red;
  if (tid < 3) {  // one thread per component: G, chi, Delta, r', and (window kernel) the spline weights of that axis
    const int c = tid;
    const double g_old = c == 0 ? v[0] + v[4] : (c == 1 ? v[1] + v[5] : v[2] + v[6]);
    const double rkc = R[3 * k + c];
    double delta, rn;
    if (rnew_given) {
      rn = rnew_given[3 * (size_t)w + c];
      delta = rn - rkc;
    } else {
      const double chi = c == 0 ? gp[0] * gp[1] : (c == 1 ? gp[0] * gp[2] : gp[3] * gp[4]);
      const double xx = __dadd_rn(__dmul_rn(d.tau, g_old), __dmul_rn(d.sqrt_tau, chi));
      delta = (double)__double2float_rn(xx);
      rn = rkc + delta;
    }
    ms.g_old[c] = g_old;
    ms.delta[c] = delta;
    ms.rn[c] = rn;
    if (c == 0) *ms.usum_old = v[3];
    if (sw_out) spline_axis<T>(d, c, rn, *sw_out);
  }
}

// ---- qmc_ratio_grad ------------------------------------------------------------------------
// rho_D = b . phi(r'); grad = (b . grad phi(r'))/rho_D + grad_k ln Psi_J(R'); rho_J (D:C2, C3)
// b: inverse row (window applied); vgl: [5][ns] at r'; R: positions; red: MOVE_RED doubles.
template <typename T, int NT = MOVE_NT>
__device__ __forceinline__ void dev_ratio_grad(const CrowdDev& d, int w, int k, const double* b, const T* vgl,
                                               const double* R, MoveScal ms, double* ratio_out, double* grad_out,
                                               double* red)
{
  const int ns = d.ns, tid = threadIdx.x;
  double v[8] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
  for (int j = tid; j < d.M; j += NT) {
    const double bj = b[j];
    v[0] = fma(bj, (double)vgl[j], v[0]);
    v[1] = fma(bj, (double)vgl[ns + j], v[1]);
    v[2] = fma(bj, (double)vgl[2 * ns + j], v[2]);
    v[3] = fma(bj, (double)vgl[3 * ns + j], v[3]);
  }
  const double rn[3] = {ms.rn[0], ms.rn[1], ms.rn[2]};
  {
    double g[3] = {0.0, 0.0, 0.0};
    j2_partial<NT>(d, R, k, rn, v[4], g);
    v[5] = g[0]; v[6] = g[1]; v[7] = g[2];
  }
  block_sum_t0<8, NT>(v, red);
  if (tid == 0) {
    const double rho_d = v[0];
    const double rho_j = exp(v[4] - *ms.usum_old);
    *ms.rho_d = rho_d;
    *ms.rho_j = rho_j;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const double g = v[1 + c] / rho_d + v[5 + c];
      ms.g_new[c] = g;
      if (grad_out) grad_out[3 * (size_t)w + c] = g;
    }
    if (ratio_out) ratio_out[w] = rho_d * rho_j;
  }
}

// ---- Metropolis decision (D:C4) -------------------------------------------------------------------
// p = rho^2 exp(logGb - logGf), logGf = -|Delta - tau G(R)|^2/2tau, logGb = -|-Delta - tau G(R')|^2/2tau;
// accept <=> u < p.  Thread 0 decides; every thread gets the flag (contains one __syncthreads).
__device__ __forceinline__ int dev_decide(const CrowdDev& d, int w, int k, MoveScal ms, unsigned char* acc_out)
{
  __shared__ int s_acc;
  if (threadIdx.x == 0) {
    const double tau = d.tau;
    double f2 = 0.0, b2 = 0.0;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const double dl = ms.delta[c];
      const double f = dl - tau * ms.g_old[c];
      const double b = -dl - tau * ms.g_new[c];
      f2 += f * f;
      b2 += b * b;
    }
    const double log_gf = -f2 / (2.0 * tau), log_gb = -b2 / (2.0 * tau);
    const double rho_d = *ms.rho_d;
    const double rho = rho_d * *ms.rho_j;
    const double p = rho * rho * exp(log_gb - log_gf);
    unsigned x[4];
    philox4x32_10((unsigned)(d.walker_id0 + w), (unsigned)k, *d.sweep, 1u, d.seed_lo, d.seed_hi, x);
    const double u = u01(x[0]);
    const int acc = (rho_d != 0.0 && isfinite(p) && u < p) ? 1 : 0;
    d.p[w] = p;
    d.u[w] = u;
    d.accepted[w] = (unsigned char)acc;
    if (acc_out) acc_out[w] = (unsigned char)acc;
    if (acc) atomicAdd(d.counters, 1ull);
    s_acc = acc;
  }
  __syncthreads();
  return s_acc;
}

// ---- bordering of S^-1 by one accepted move (D:C6, R2) ------------------------------------------------
// Given q_s[l] = C[l,:].phi' (l < m), the corner B0[k,:].phi', y_s = Sinv p (from the row step) and
// z = q^T Sinv:  sigma = corner - q.y (= rho_D up to rounding); Sinv <- [[Sinv + y z^T/sigma, -y/sigma],
// [-z^T/sigma, 1/sigma]].  Sinv has row stride ss; contains two __syncthreads.
__device__ __forceinline__ void sinv_border(double* Sinv, int ss, int m, const double* q_s, const double* y_s,
                                            double* z_s, double* misc)
{
  const int tid = threadIdx.x;
  for (int l = tid; l < m; l += MOVE_NT) {
    double z = 0.0;
#pragma unroll 8
    for (int q = 0; q < m; ++q) z = fma(q_s[q], Sinv[(size_t)q * ss + l], z);
    z_s[l] = z;
  }
  if (tid == 0) {
    double s = misc[0];
    for (int l = 0; l < m; ++l) s = fma(-q_s[l], y_s[l], s);
    misc[1] = 1.0 / s;
  }
  __syncthreads();
  const double inv_sigma = misc[1];
  for (int e = tid; e < m * m; e += MOVE_NT) {
    const int a = e / m, b = e - a * m;
    Sinv[(size_t)a * ss + b] = fma(y_s[a] * inv_sigma, z_s[b], Sinv[(size_t)a * ss + b]);
  }
  for (int l = tid; l < m; l += MOVE_NT) {
    Sinv[(size_t)l * ss + m] = -y_s[l] * inv_sigma;
    Sinv[(size_t)m * ss + l] = -z_s[l] * inv_sigma;
  }
  if (tid == 0) Sinv[(size_t)m * ss + m] = inv_sigma;
  __syncthreads();
}

// ---- step path: operands in global memory (the C-ABI step calls, any electron order) -------------------
// (a) b = B0[k,:] - C^T (Sinv p), p_l = V[l,:].B0[k,:] - [rows[l]==k]   (D:C6), then G_k(R) and the proposal.
// sm: (ns + 2 kdp + MOVE_RED) doubles
template <typename T>
__device__ __forceinline__ void dev_row_propose(const CrowdDev& d, int w, int k, const double* rnew_given, double* sm)
{
  const int ns = d.ns, kdp = d.kdp, tid = threadIdx.x;
  double* b_s = sm;
  double* p_s = b_s + ns;
  double* y_s = p_s + kdp;
  double* red = y_s + kdp;
  const int spin = k / d.n, kk = k - spin * d.n;
  const size_t B0 = ((size_t)w * 2 + spin) * ns * ns;   // index of the matrix in the carried inverses (fp64 or fp32 storage)
  const int m = d.kd > 1 ? d.mwin[w] : 0;

  for (int j = tid; j < ns; j += MOVE_NT) b_s[j] = ld_binv(d, B0 + (size_t)kk * ns + j);
  __syncthreads();
  if (m > 0) {
    const double* V = d.V + (size_t)w * kdp * ns;
    const double* C = d.C + (size_t)w * kdp * ns;
    const int* rows = d.rows + (size_t)w * kdp;
    double* pvec = d.pvec + (size_t)w * kdp;
    rows_dot<4>(m, ns, [&](int l) { return V + (size_t)l * ns; },
                [&](int jj) { return make_double2(b_s[2 * jj], b_s[2 * jj + 1]); },
                [&](int l, double acc) {
                  const double pl = acc - (rows[l] == kk ? 1.0 : 0.0);
                  p_s[l] = pl;
                  pvec[l] = pl;
                });
    __syncthreads();
    sinv_matvec(d.Sinv + (size_t)w * kdp * kdp, kdp, m, p_s, y_s);
    __syncthreads();
    for (int l = tid; l < m; l += MOVE_NT) d.yvec[(size_t)w * kdp + l] = y_s[l];
    axpy_rows(b_s, ns, m, y_s, [&](int l) { return C + (size_t)l * ns; });
    __syncthreads();
  }
  double* brow = d.brow + (size_t)w * ns;
  for (int j = tid; j < ns; j += MOVE_NT) brow[j] = b_s[j];
  const T* cache = static_cast<const T*>(d.cache) + ((size_t)w * d.N + k) * 4 * ns;
  dev_gold_propose<T>(d, w, k, b_s, cache, d.R + (size_t)w * d.N * 3, rnew_given, move_scal_global(d, w), red);
}

// Accepted move: r_k <- r', caches, and with a delayed window (D:C6) V[m] = phi', C[m] = B0[k,:], S^-1 bordered.
// sm: (ns + 3 kdp + 16) doubles
template <typename T>
__device__ __forceinline__ void dev_accept_update(const CrowdDev& d, int w, int k, double* sm)
{
  const int ns = d.ns, kdp = d.kdp, tid = threadIdx.x;
  const T* vgl = static_cast<const T*>(d.vgl) + (size_t)w * 5 * ns;
  T* cache = static_cast<T*>(d.cache) + ((size_t)w * d.N + k) * 4 * ns;
  for (int j = tid; j < 4 * ns; j += MOVE_NT) cache[j] = vgl[ns + j];
  if (tid < 3) d.R[((size_t)w * d.N + k) * 3 + tid] = d.rnew[3 * (size_t)w + tid];
  if (d.kd == 1) return;

  const int spin = k / d.n, kk = k - spin * d.n;
  const int m = d.mwin[w];
  double* V = d.V + (size_t)w * kdp * ns;
  double* C = d.C + (size_t)w * kdp * ns;
  const size_t B0k = (((size_t)w * 2 + spin) * ns + kk) * ns;
  double* q_s = sm;            // [kdp]  q_l = C[l,:].phi'
  double* z_s = q_s + kdp;     // [kdp]  z = q^T Sinv
  double* y_s = z_s + kdp;     // [kdp]  y = Sinv p
  double* misc = y_s + kdp;    // corner, 1/sigma
  double* phi_s = misc + 16;   // [ns]   phi' widened to fp64 (padding columns are zero)
  for (int j = tid; j < ns; j += MOVE_NT) {
    const double ph = (double)vgl[j];
    phi_s[j] = ph;
    V[(size_t)m * ns + j] = ph;
    C[(size_t)m * ns + j] = ld_binv(d, B0k + j);
  }
  for (int l = tid; l < m; l += MOVE_NT) y_s[l] = d.yvec[(size_t)w * kdp + l];
  __syncthreads();
  // q_l = C[l,:].phi' for l < m, and the corner B0[k,:].phi' (= row m of C, just written)
  rows_dot<4>(m + 1, ns, [&](int l) { return C + (size_t)l * ns; },
              [&](int jj) { return make_double2(phi_s[2 * jj], phi_s[2 * jj + 1]); },
              [&](int l, double acc) { if (l < m) q_s[l] = acc; else misc[0] = acc; });
  __syncthreads();
  sinv_border(d.Sinv + (size_t)w * kdp * kdp, kdp, m, q_s, y_s, z_s, misc);
  if (tid == 0) {
    d.rows[(size_t)w * kdp + m] = kk;
    d.mwin[w] = m + 1;
  }
}

// ---- the three step kernels.  dynamic smem of all of them: move_smem(d) -----------------------------
template <typename T>
__global__ void __launch_bounds__(MOVE_NT) row_propose_kernel(CrowdDev d, int k, const double* __restrict__ rnew_given)
{
  extern __shared__ double sm[];
  dev_row_propose<T>(d, blockIdx.x, k, rnew_given, sm);
}
template <typename T>
__global__ void __launch_bounds__(MOVE_NT) ratio_grad_kernel(CrowdDev d, int k, double* ratio_out, double* grad_out)
{
  extern __shared__ double sm[];
  const int w = blockIdx.x;
  dev_ratio_grad<T>(d, w, k, d.brow + (size_t)w * d.ns, static_cast<const T*>(d.vgl) + (size_t)w * 5 * d.ns,
                    d.R + (size_t)w * d.N * 3, move_scal_global(d, w), ratio_out, grad_out, sm);
}
template <typename T>
__global__ void __launch_bounds__(MOVE_NT) accept_kernel(CrowdDev d, int k, unsigned char* acc_out)
{
  extern __shared__ double sm[];
  const int w = blockIdx.x;
  if (dev_decide(d, w, k, move_scal_global(d, w), acc_out)) dev_accept_update<T>(d, w, k, sm);
}
// qmc_sweep with delay_rank = 1: ratio(k) + decision + state update in one launch (rank-1 kernel follows)
template <typename T>
__global__ void __launch_bounds__(MOVE_NT) ratio_accept_kernel(CrowdDev d, int k)
{
  extern __shared__ double sm[];
  const int w = blockIdx.x;
  const MoveScal ms = move_scal_global(d, w);
  dev_ratio_grad<T>(d, w, k, d.brow + (size_t)w * d.ns, static_cast<const T*>(d.vgl) + (size_t)w * 5 * d.ns,
                    d.R + (size_t)w * d.N * 3, ms, nullptr, nullptr, sm);
  __syncthreads();
  if (dev_decide(d, w, k, ms, nullptr)) dev_accept_update<T>(d, w, k, sm);
}

__global__ void bump_sweep_kernel(unsigned* sweep) { *sweep += 1u; }
__global__ void set_u32_kernel(unsigned* p, unsigned v) { *p = v; }

}  // namespace qmc
