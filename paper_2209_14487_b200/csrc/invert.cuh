// invert.cuh -- qmc_crowd_create / set_positions: X = A^T (filled by spline_build_kernel) is
// inverted in place, giving B = (A^T)^-1 = (A^-1)^T (D:C2).  In-place Gauss-Jordan with partial
// pivoting (row swaps, undone as column swaps at the end), one CTA per (walker, spin).  Not on the
// timed path.  A zero or non-finite pivot sets *d.status (D:A16).
// Also the small gather/scatter kernels behind the state getters.
#pragma once
#include "common.cuh"

namespace qmc {

constexpr int INV_NT = 512;

// dynamic smem: 2 ns doubles + ns ints + 2*INV_NT/32 (double + int) reduction slots
__global__ void __launch_bounds__(INV_NT) invert_kernel(CrowdDev d)
{
  extern __shared__ double sm[];
  const int ns = d.ns, n = d.n, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  double* colf = sm;
  double* rowc = colf + ns;
  double* redv = rowc + ns;
  int* redi = reinterpret_cast<int*>(redv + INV_NT / 32);
  int* piv = redi + INV_NT / 32;
  __shared__ int s_p;
  __shared__ int s_bad;
  double* X = d.Binv + (size_t)blockIdx.x * ns * ns;
  if (tid == 0) s_bad = 0;
  __syncthreads();
  for (int c = 0; c < n; ++c) {
    // pivot: first row r >= c with the largest |X[r][c]|
    // (a NaN entry counts as +inf so that the singular check below fires)
    double best = -1.0;
    int bi = c;
    for (int r = c + tid; r < n; r += INV_NT) {
      double v = fabs(X[(size_t)r * ns + c]);
      if (!(v == v)) v = INFINITY;
      if (v > best) { best = v; bi = r; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const double ov = __shfl_xor_sync(0xffffffffu, best, o);
      const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
      if (ov > best || (ov == best && oi < bi)) { best = ov; bi = oi; }
    }
    if (lane == 0) { redv[warp] = best; redi[warp] = bi; }
    __syncthreads();
    if (tid == 0) {
      double bv = redv[0];
      int bj = redi[0];
      for (int q = 1; q < INV_NT / 32; ++q) {
        const double ov = redv[q];
        const int oi = redi[q];
        const bool take = ov > bv || (ov == bv && oi < bj);
        if (take) { bv = ov; bj = oi; }
      }
      s_p = bj;
      piv[c] = bj;
      if (!(bv > 0.0) || !isfinite(bv)) s_bad = 1;
    }
    __syncthreads();
    if (s_bad) break;
    const int p = s_p;
    if (p != c) {
      for (int j = tid; j < n; j += INV_NT) {
        const double a = X[(size_t)c * ns + j], b = X[(size_t)p * ns + j];
        X[(size_t)c * ns + j] = b;
        X[(size_t)p * ns + j] = a;
      }
      __syncthreads();
    }
    // true divisions (not a reciprocal multiply): a duplicated column then cancels exactly and the
    // next pivot search sees an exact zero, as the oracle's LU does
    const double pv = X[(size_t)c * ns + c];
    for (int j = tid; j < n; j += INV_NT) {
      colf[j] = X[(size_t)j * ns + c];
      rowc[j] = (j == c) ? 1.0 / pv : X[(size_t)c * ns + j] / pv;
    }
    __syncthreads();
    for (int e = tid; e < n * n; e += INV_NT) {
      const int r = e / n, j = e - r * n;
      double v;
      if (r == c) v = rowc[j];
      else v = fma(-colf[r], rowc[j], (j == c) ? 0.0 : X[(size_t)r * ns + j]);
      X[(size_t)r * ns + j] = v;
    }
    __syncthreads();
  }
  if (s_bad) {
    if (tid == 0) atomicExch(d.status, 4);
    return;
  }
  for (int c = n - 1; c >= 0; --c) {
    const int p = piv[c];
    if (p != c) {
      for (int r = tid; r < n; r += INV_NT) {
        const double a = X[(size_t)r * ns + c], b = X[(size_t)r * ns + p];
        X[(size_t)r * ns + c] = b;
        X[(size_t)r * ns + p] = a;
      }
      __syncthreads();
    }
  }
}

// dst[(b * rows + r) * cols + c] = src[b * sb + r * sr + c]   (gather = pack; scatter = unpack)
template <typename TD, typename TS>
__global__ void pack_kernel(TD* __restrict__ dst, const TS* __restrict__ src, size_t nb, int rows, int cols, size_t sb,
                            size_t sr, int scatter)
{
  const size_t total = nb * (size_t)rows * cols;
  for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (size_t)gridDim.x * blockDim.x) {
    const size_t b = e / ((size_t)rows * cols);
    const size_t rem = e - b * (size_t)rows * cols;
    const size_t r = rem / cols, c = rem - r * cols;
    if (scatter) dst[b * sb + r * sr + c] = (TD)src[e];
    else dst[e] = (TD)src[b * sb + r * sr + c];
  }
}

}  // namespace qmc
