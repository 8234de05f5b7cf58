// move.cuh -- the per-walker scalar side of a move: inverse row with the delayed window applied,
// drift-diffusion proposal, determinant/Jastrow ratio and gradient, Metropolis decision, window
// append (SURVEY 8(a) steps a0, a2, a3, a4').  One CTA of MOVE_NT threads per walker; all
// length-n / length-N sums are strided over the block and combined by shuffle reductions (BJ).
#pragma once
#include "common.cuh"
#include "spline.cuh"

namespace qmc {

#ifndef QMC_MOVE_NT
#define QMC_MOVE_NT 128
#endif
#ifndef QMC_MOVE_DOT_ROWS
#define QMC_MOVE_DOT_ROWS 2
#endif
constexpr int MOVE_NT = QMC_MOVE_NT;
constexpr int MOVE_RED = 8 * (MOVE_NT / 32) < 32 ? 32 : 8 * (MOVE_NT / 32);  // doubles of reduction scratch

// D:C3: one pair term of the two-body Jastrow for electron k placed at rk against electron i.
// u(r) = a r/(1 + b r), u'(r) = a/(1 + b r)^2, minimum image d_c <- d_c - L rint(d_c/L).
__device__ __forceinline__ void j2_pair(const CrowdDev& d, const double (&rk)[3], const double* ri,
                                        double& usum, double (&g)[3])
{
  double dd[3], r2 = 0.0;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    double x = rk[c] - ri[c];
    x -= d.box[c] * rint(x * d.inv_box[c]);
    dd[c] = x;
    r2 = fma(x, x, r2);
  }
  if (r2 > 0.0) {
    const double inv_r = rsqrt(r2);
    const double r = r2 * inv_r;
    const double inv_den = 1.0 / fma(d.j2_b, r, 1.0);
    usum += d.j2_a * r * inv_den;
    const double f = d.j2_a * inv_den * inv_den * inv_r;
#pragma unroll
    for (int c = 0; c < 3; ++c) g[c] = fma(f, dd[c], g[c]);
  }
}

// out[l] = mat[l,:] . x for l in [0, nrows), mat row-major with stride ns (ns % 2 == 0), x in shared
// memory.  A warp takes MOVE_DOT_ROWS rows at a time and keeps their loads in flight together
// (one DRAM round trip per group instead of one per row); then shuffle-reduces each row.
constexpr int MOVE_DOT_ROWS = QMC_MOVE_DOT_ROWS;
template <typename F>
__device__ __forceinline__ void rows_dot(const double* mat, int ns, int nrows, const double* x_s, F&& store)
{
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int l0 = warp * MOVE_DOT_ROWS; l0 < nrows; l0 += (MOVE_NT / 32) * MOVE_DOT_ROWS) {
    double acc[MOVE_DOT_ROWS];
#pragma unroll
    for (int r = 0; r < MOVE_DOT_ROWS; ++r) acc[r] = 0.0;
#pragma unroll 2
    for (int jj = lane; jj < ns / 2; jj += 32) {
      const double x0 = x_s[2 * jj], x1 = x_s[2 * jj + 1];
      double2 v[MOVE_DOT_ROWS];
#pragma unroll
      for (int r = 0; r < MOVE_DOT_ROWS; ++r)
        v[r] = (l0 + r < nrows) ? reinterpret_cast<const double2*>(mat + (size_t)(l0 + r) * ns)[jj] : make_double2(0.0, 0.0);
#pragma unroll
      for (int r = 0; r < MOVE_DOT_ROWS; ++r) acc[r] = fma(v[r].x, x0, fma(v[r].y, x1, acc[r]));
    }
#pragma unroll
    for (int r = 0; r < MOVE_DOT_ROWS; ++r) {
      const double t = warp_sum(acc[r]);
      if (lane == 0 && l0 + r < nrows) store(l0 + r, t);
    }
  }
}

// ---- qmc_spo_vgl steps (a)+(b) -----------------------------------------------------------
// (a) b = B0[k,:] - C^T (Sinv p), p_l = V[l,:].B0[k,:] - [rows[l]==k]   (D:C6)
//     G_k(R) = b . grad phi(r_k) [cache] + grad_k ln Psi_J(R)             (D:C2, C3, A13)
// (b) Delta = fl32(tau G + sqrt(tau) chi), r' = r_k + Delta               (D:C4, C7)
// sm: (ns + 2 kdp + MOVE_RED) doubles
template <typename T>
__device__ __forceinline__ void dev_row_propose(const CrowdDev& d, int w, int k, const double* __restrict__ rnew_given,
                                                double* sm)
{
  const int ns = d.ns, kdp = d.kdp, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  double* b_s = sm;
  double* p_s = b_s + ns;
  double* y_s = p_s + kdp;
  double* red = y_s + kdp;
  const int spin = k / d.n, kk = k - spin * d.n;
  const double* B0 = d.Binv + ((size_t)w * 2 + spin) * ns * ns;
  const int m = d.kd > 1 ? d.mwin[w] : 0;

  for (int j = tid; j < ns; j += MOVE_NT) b_s[j] = B0[(size_t)kk * ns + j];
  __syncthreads();
  if (m > 0) {
    const double* V = d.V + (size_t)w * kdp * ns;
    const double* C = d.C + (size_t)w * kdp * ns;
    const double* Sinv = d.Sinv + (size_t)w * kdp * kdp;
    const int* rows = d.rows + (size_t)w * kdp;
    double* pvec = d.pvec + (size_t)w * kdp;
    rows_dot(V, ns, m, b_s, [&](int l, double acc) {
      const double pl = acc - (rows[l] == kk ? 1.0 : 0.0);
      p_s[l] = pl;
      pvec[l] = pl;
    });
    __syncthreads();
    for (int l = tid; l < m; l += MOVE_NT) {
      double y = 0.0;
#pragma unroll 8
      for (int q = 0; q < m; ++q) y = fma(Sinv[(size_t)l * kdp + q], p_s[q], y);
      y_s[l] = y;
      d.yvec[(size_t)w * kdp + l] = y;
    }
    __syncthreads();
    for (int jj = tid; jj < ns / 2; jj += MOVE_NT) {
      double2 acc = make_double2(b_s[2 * jj], b_s[2 * jj + 1]);
#pragma unroll 8
      for (int l = 0; l < m; ++l) {
        const double2 c = reinterpret_cast<const double2*>(C + (size_t)l * ns)[jj];
        acc.x = fma(-y_s[l], c.x, acc.x);
        acc.y = fma(-y_s[l], c.y, acc.y);
      }
      b_s[2 * jj] = acc.x;
      b_s[2 * jj + 1] = acc.y;
    }
    __syncthreads();
  }
  double* brow = d.brow + (size_t)w * ns;
  for (int j = tid; j < ns; j += MOVE_NT) brow[j] = b_s[j];

  // v[0..2] = b . grad phi(r_k), v[3] = usum_old, v[4..6] = grad_k ln Psi_J(R)
  double v[7] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
  const T* cache = static_cast<const T*>(d.cache) + ((size_t)w * d.N + k) * 4 * ns;
  for (int j = tid; j < d.M; j += MOVE_NT) {
    const double bj = b_s[j];
    v[0] = fma(bj, (double)cache[j], v[0]);
    v[1] = fma(bj, (double)cache[ns + j], v[1]);
    v[2] = fma(bj, (double)cache[2 * ns + j], v[2]);
  }
  const double* R = d.R + (size_t)w * d.N * 3;
  double rk[3] = {R[3 * k], R[3 * k + 1], R[3 * k + 2]};
  {
    double g[3] = {0.0, 0.0, 0.0};
    for (int i = tid; i < d.N; i += MOVE_NT)
      if (i != k) j2_pair(d, rk, R + 3 * i, v[3], g);
    v[4] = g[0]; v[5] = g[1]; v[6] = g[2];
  }
  block_sum<7, MOVE_NT>(v, red);
  if (tid == 0) {
    double g_old[3] = {v[0] + v[4], v[1] + v[5], v[2] + v[6]};
    double delta[3], rn[3];
    if (rnew_given) {
#pragma unroll
      for (int c = 0; c < 3; ++c) { rn[c] = rnew_given[3 * (size_t)w + c]; delta[c] = rn[c] - rk[c]; }
    } else {
      unsigned x[4];
      philox4x32_10((unsigned)(d.walker_id0 + w), (unsigned)k, *d.sweep, 0u, d.seed_lo, d.seed_hi, x);
      const double two_pi = 6.283185307179586476925286766559;
      const double r0 = sqrt(-2.0 * log(u01(x[0])));
      const double r1 = sqrt(-2.0 * log(u01(x[2])));
      const double chi[3] = {r0 * cos(two_pi * u01(x[1])), r0 * sin(two_pi * u01(x[1])), r1 * cos(two_pi * u01(x[3]))};
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const double xx = __dadd_rn(__dmul_rn(d.tau, g_old[c]), __dmul_rn(d.sqrt_tau, chi[c]));
        delta[c] = (double)__double2float_rn(xx);
        rn[c] = rk[c] + delta[c];
      }
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      d.g_old[3 * (size_t)w + c] = g_old[c];
      d.delta[3 * (size_t)w + c] = delta[c];
      d.rnew[3 * (size_t)w + c] = rn[c];
    }
    d.usum_old[w] = v[3];
  }
}

// ---- qmc_ratio_grad ------------------------------------------------------------------------
// rho_D = b . phi(r'); grad = (b . grad phi(r'))/rho_D + grad_k ln Psi_J(R'); rho_J (D:C2, C3)
// sm: MOVE_RED doubles
template <typename T>
__device__ __forceinline__ void dev_ratio_grad(const CrowdDev& d, int w, int k, double* __restrict__ ratio_out,
                                               double* __restrict__ grad_out, double* red)
{
  const int ns = d.ns, tid = threadIdx.x;
  const double* b = d.brow + (size_t)w * ns;
  const T* vgl = static_cast<const T*>(d.vgl) + (size_t)w * 5 * ns;
  double v[8] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
  for (int j = tid; j < d.M; j += MOVE_NT) {
    const double bj = b[j];
    v[0] = fma(bj, (double)vgl[j], v[0]);
    v[1] = fma(bj, (double)vgl[ns + j], v[1]);
    v[2] = fma(bj, (double)vgl[2 * ns + j], v[2]);
    v[3] = fma(bj, (double)vgl[3 * ns + j], v[3]);
  }
  const double* R = d.R + (size_t)w * d.N * 3;
  const double rn[3] = {d.rnew[3 * (size_t)w], d.rnew[3 * (size_t)w + 1], d.rnew[3 * (size_t)w + 2]};
  {
    double g[3] = {0.0, 0.0, 0.0};
    for (int i = tid; i < d.N; i += MOVE_NT)
      if (i != k) j2_pair(d, rn, R + 3 * i, v[4], g);
    v[5] = g[0]; v[6] = g[1]; v[7] = g[2];
  }
  block_sum<8, MOVE_NT>(v, red);
  if (tid == 0) {
    const double rho_d = v[0];
    const double rho_j = exp(v[4] - d.usum_old[w]);
    d.rho_d[w] = rho_d;
    d.rho_j[w] = rho_j;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const double g = v[1 + c] / rho_d + v[5 + c];
      d.g_new[3 * (size_t)w + c] = g;
      if (grad_out) grad_out[3 * (size_t)w + c] = g;
    }
    if (ratio_out) ratio_out[w] = rho_d * rho_j;
  }
}

// ---- qmc_accept_reject: decision, state update, window append --------------------------------
// p = rho^2 exp(logGb - logGf), logGf = -|Delta - tau G(R)|^2/2tau, logGb = -|-Delta - tau G(R')|^2/2tau
// (D:C4); accept <=> u < p.  On accept with a delayed window (D:C6): V[m] = phi', C[m] = B0[k,:],
// S^-1 bordered with column p (kept by row_propose), row q_l = C[l,:].phi' and Schur complement
// sigma = B0[k,:].phi' - q.(Sinv p) (= rho_D up to rounding).
// sm: (ns + 3 kdp + 16) doubles
template <typename T>
__device__ __forceinline__ void dev_accept(const CrowdDev& d, int w, int k, unsigned char* __restrict__ acc_out,
                                           double* sm)
{
  __shared__ int s_acc;
  const int ns = d.ns, kdp = d.kdp, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) {
    const double tau = d.tau;
    double f2 = 0.0, b2 = 0.0;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const double dl = d.delta[3 * (size_t)w + c];
      const double f = dl - tau * d.g_old[3 * (size_t)w + c];
      const double b = -dl - tau * d.g_new[3 * (size_t)w + c];
      f2 += f * f;
      b2 += b * b;
    }
    const double log_gf = -f2 / (2.0 * tau), log_gb = -b2 / (2.0 * tau);
    const double rho_d = d.rho_d[w];
    const double rho = rho_d * d.rho_j[w];
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
  if (!s_acc) return;

  const T* vgl = static_cast<const T*>(d.vgl) + (size_t)w * 5 * ns;
  T* cache = static_cast<T*>(d.cache) + ((size_t)w * d.N + k) * 4 * ns;
  for (int j = tid; j < 4 * ns; j += MOVE_NT) cache[j] = vgl[ns + j];
  if (tid < 3) d.R[((size_t)w * d.N + k) * 3 + tid] = d.rnew[3 * (size_t)w + tid];
  if (d.kd == 1) return;

  const int spin = k / d.n, kk = k - spin * d.n;
  const int m = d.mwin[w];
  double* V = d.V + (size_t)w * kdp * ns;
  double* C = d.C + (size_t)w * kdp * ns;
  double* Sinv = d.Sinv + (size_t)w * kdp * kdp;
  const double* B0k = d.Binv + (((size_t)w * 2 + spin) * ns + kk) * ns;
  double* q_s = sm;            // [kdp]  q_l = C[l,:].phi'
  double* z_s = q_s + kdp;     // [kdp]  z = q^T Sinv
  double* y_s = z_s + kdp;     // [kdp]  y = Sinv p
  double* misc = y_s + kdp;    // corner, sigma
  double* phi_s = misc + 16;   // [ns]   phi' widened to fp64 (padding columns are zero)
  for (int j = tid; j < ns; j += MOVE_NT) {
    const double ph = (double)vgl[j];
    phi_s[j] = ph;
    V[(size_t)m * ns + j] = ph;
    C[(size_t)m * ns + j] = B0k[j];
  }
  __syncthreads();
  // q_l = C[l,:].phi' for l < m, and the corner B0[k,:].phi' (= row m of C, just written)
  rows_dot(C, ns, m + 1, phi_s, [&](int l, double acc) { if (l < m) q_s[l] = acc; else misc[0] = acc; });
  for (int l = tid; l < m; l += MOVE_NT) y_s[l] = d.yvec[(size_t)w * kdp + l];
  __syncthreads();
  for (int l = tid; l < m; l += MOVE_NT) {
    double z = 0.0;
#pragma unroll 8
    for (int q = 0; q < m; ++q) z = fma(q_s[q], Sinv[(size_t)q * kdp + l], z);
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
    Sinv[(size_t)a * kdp + b] = fma(y_s[a] * inv_sigma, z_s[b], Sinv[(size_t)a * kdp + b]);
  }
  for (int l = tid; l < m; l += MOVE_NT) {
    Sinv[(size_t)l * kdp + m] = -y_s[l] * inv_sigma;
    Sinv[(size_t)m * kdp + l] = -z_s[l] * inv_sigma;
  }
  if (tid == 0) {
    Sinv[(size_t)m * kdp + m] = inv_sigma;
    d.rows[(size_t)w * kdp + m] = kk;
    d.mwin[w] = m + 1;
  }
}

// ---- kernels: the three step calls, and their fusions used by qmc_sweep ------------------------
// Walkers never interact, so nothing forces a kernel boundary between accept(k) and the row/proposal
// of electron k+1 of the same walker: move_fused_kernel does ratio(k), accept(k), row_propose(k+1) in
// one CTA, so the window rows C (read for the append and again for the next row), V and the positions
// come from DRAM once.  The device functions are the ones the step kernels run.
// dynamic smem of all of them: move_smem_doubles(d) doubles
template <typename T>
__global__ void __launch_bounds__(MOVE_NT) row_propose_kernel(CrowdDev d, int k, const double* __restrict__ rnew_given)
{
  extern __shared__ double sm[];
  dev_row_propose<T>(d, blockIdx.x, k, rnew_given, sm);
}
template <typename T>
__global__ void __launch_bounds__(MOVE_NT) ratio_grad_kernel(CrowdDev d, int k, double* __restrict__ ratio_out,
                                                             double* __restrict__ grad_out)
{
  extern __shared__ double sm[];
  dev_ratio_grad<T>(d, blockIdx.x, k, ratio_out, grad_out, sm);
}
template <typename T>
__global__ void __launch_bounds__(MOVE_NT) accept_kernel(CrowdDev d, int k, unsigned char* __restrict__ acc_out)
{
  extern __shared__ double sm[];
  dev_accept<T>(d, blockIdx.x, k, acc_out, sm);
}
// ratio(k) + accept(k); with NEXT also row_propose(k + 1) (same spin block, no flush in between)
template <typename T, bool NEXT>
__global__ void __launch_bounds__(MOVE_NT) move_fused_kernel(CrowdDev d, int k)
{
  extern __shared__ double sm[];
  const int w = blockIdx.x;
  dev_ratio_grad<T>(d, w, k, nullptr, nullptr, sm);
  __syncthreads();
  dev_accept<T>(d, w, k, nullptr, sm);
  if (NEXT) {
    __syncthreads();
    dev_row_propose<T>(d, w, k + 1, nullptr, sm);
  }
}

// ---- qmc_sweep, delayed update: one launch per delay window ---------------------------------------
// The crowd advances in lock-step per *window*: a CTA owns one walker for the cnt <= delay_rank
// moves k0 .. k0+cnt-1 of the window (row/proposal, spline, ratio, accept, append for each), then the
// whole crowd flushes.  Walkers never interact inside a window, so nothing needs a kernel boundary
// between moves: the SM overlaps the DRAM-bound gather of one walker with the fp64 work of the others,
// the window rows V, C a walker appends stay in L2 for its next moves, and the launch tail is paid
// once per window instead of twice per move.  Same device functions as the step kernels.
// dynamic smem: move_smem_doubles(d) doubles
template <typename T>
__global__ void __launch_bounds__(MOVE_NT, 4) window_kernel(CrowdDev d, int k0, int cnt)
{
  extern __shared__ double sm[];
  __shared__ SplineW<T> sw;
  const int w = blockIdx.x, ns = d.ns;
  T* vgl = static_cast<T*>(d.vgl) + (size_t)w * 5 * ns;
  const int spin = k0 / d.n;
  for (int k = k0; k < k0 + cnt; ++k) {
    if (k + 1 < k0 + cnt) {
      // next move's inverse row and gradient cache are first-touch DRAM lines: pull them into L2 now
      const int kk1 = k + 1 - spin * d.n;
      const char* brow_n = reinterpret_cast<const char*>(d.Binv + (((size_t)w * 2 + spin) * ns + kk1) * ns);
      const char* cache_n = reinterpret_cast<const char*>(static_cast<const T*>(d.cache) + ((size_t)w * d.N + k + 1) * 4 * ns);
      const int lb = ns * 8 / 128, lc = 3 * ns * (int)sizeof(T) / 128;
      for (int i = threadIdx.x; i < lb + lc; i += MOVE_NT) {
        const char* p = i < lb ? brow_n + (size_t)i * 128 : cache_n + (size_t)(i - lb) * 128;
        asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
      }
    }
    dev_row_propose<T>(d, w, k, nullptr, sm);
    spline_cta<T, MOVE_NT>(d, d.rnew + 3 * (size_t)w, sw, vgl);
    __syncthreads();
    dev_ratio_grad<T>(d, w, k, nullptr, nullptr, sm);
    __syncthreads();
    dev_accept<T>(d, w, k, nullptr, sm);
    __syncthreads();
  }
}

__global__ void bump_sweep_kernel(unsigned* sweep) { *sweep += 1u; }
__global__ void set_u32_kernel(unsigned* p, unsigned v) { *p = v; }

}  // namespace qmc
