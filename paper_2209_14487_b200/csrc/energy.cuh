// energy.cuh -- kinetic part of the local energy, T = -1/2 sum_k lap_k Psi / Psi (Alg. 1 line 11,
// PAPER.md:59), from what the move path already carries: the transposed
// inverses (row k = electron k, D:C2), the per-electron caches of grad phi and lap phi at the current
// positions (D:A12: "computed and cached, not consumed" by the move -- consumed here) and the positions.
//   lap_k Psi / Psi = lap_k ln Psi + |grad_k ln Psi|^2
//                   = b.lap phi + lap_k J + 2 (b.grad phi).(grad_k J) + |grad_k J|^2,
//   grad_k J = sum_i u'(r) d/r,  lap_k J = sum_i [u''(r) + 2 u'(r)/r],  u = a r/(1 + b r)      (D:C3)
// (the |b.grad phi|^2 of lap ln D cancels against the one in |grad ln Psi|^2).
// One CTA per (walker, group of EKIN_EPB electrons), one warp per electron at a time: 4 dots of length M and N pair
// terms strided over the lanes, one warp butterfly -- no block barrier after the positions are staged (the first
// version reduced every electron over the whole CTA: six pair terms per thread between two barriers, 10.9 ms per
// call at cfg 5, W = 4096).
#pragma once
#include "common.cuh"

namespace qmc {

constexpr int EKIN_NT = 128;
constexpr int EKIN_EPB = 8;

// dynamic smem: 3 N doubles.  e_elec: [W][N] per-electron terms.
template <typename T>
__global__ void __launch_bounds__(EKIN_NT) kinetic_kernel(CrowdDev d, double* __restrict__ e_elec)
{
  extern __shared__ double sm_e[];
  double* R_s = sm_e;
  const int w = blockIdx.y, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, ns = d.ns;
  const double* Rg = d.R + (size_t)w * d.N * 3;
  for (int j = tid; j < 3 * d.N; j += EKIN_NT) R_s[j] = Rg[j];
  __syncthreads();
  const int k_end = min((int)(blockIdx.x + 1) * EKIN_EPB, d.N);
  for (int k = blockIdx.x * EKIN_EPB + warp; k < k_end; k += EKIN_NT / 32) {
    const int spin = k / d.n, kk = k - spin * d.n;
    const size_t b = (((size_t)w * 2 + spin) * ns + kk) * ns;   // the electron's inverse row, fp64 or fp32 storage
    const T* cache = static_cast<const T*>(d.cache) + ((size_t)w * d.N + k) * 4 * ns;
    // v[0..2] = b.grad phi, v[3] = b.lap phi, v[4..6] = grad_k J, v[7] = lap_k J
    double v[8] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
#pragma unroll 4   // 20 independent loads in flight per lane (the loop is otherwise one L2 round trip per iteration)
    for (int j = lane; j < d.M; j += 32) {
      const double bj = ld_binv(d, b + j);
      v[0] = fma(bj, (double)cache[j], v[0]);
      v[1] = fma(bj, (double)cache[ns + j], v[1]);
      v[2] = fma(bj, (double)cache[2 * ns + j], v[2]);
      v[3] = fma(bj, (double)cache[3 * ns + j], v[3]);
    }
    const double rk[3] = {R_s[3 * k], R_s[3 * k + 1], R_s[3 * k + 2]};
#pragma unroll 2
    for (int i = lane; i < d.N; i += 32) {
      if (i == k) continue;
      double dd[3], r2 = 0.0;
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        double x = rk[c] - R_s[3 * i + c];
        x -= d.box[c] * rint(x * d.inv_box[c]);
        dd[c] = x;
        r2 = fma(x, x, r2);
      }
      if (r2 > 1e-280) {   // as j2_pair (move.cuh)
        const double inv_r = rsqrt_pos(r2);
        const double r = r2 * inv_r;
        const double inv_den = rcp_pos(fma(d.j2_b, r, 1.0));
        const double du = d.j2_a * inv_den * inv_den;
        const double f = du * inv_r;
#pragma unroll
        for (int c = 0; c < 3; ++c) v[4 + c] = fma(f, dd[c], v[4 + c]);
        v[7] += fma(-2.0 * d.j2_b * du, inv_den, 2.0 * f);
      }
    }
    warp_sum8(v);
    if (lane == 0) {
      const double cross = v[0] * v[4] + v[1] * v[5] + v[2] * v[6];
      const double gj2 = v[4] * v[4] + v[5] * v[5] + v[6] * v[6];
      e_elec[(size_t)w * d.N + k] = -0.5 * (v[3] + v[7] + 2.0 * cross + gj2);
    }
  }
}

// ekin[w] = sum_k e_elec[w][k]: one warp per walker, lane-strided partial sums, shuffle tree (fixed order).
__global__ void __launch_bounds__(128) kinetic_sum_kernel(int W, int N, const double* __restrict__ e_elec,
                                                         double* __restrict__ ekin)
{
  const int w = blockIdx.x * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (w >= W) return;
  double s = 0.0;
  for (int k = lane; k < N; k += 32) s += e_elec[(size_t)w * N + k];
  s = warp_sum(s);
  if (lane == 0) ekin[w] = s;
}

}  // namespace qmc
