// update.cuh -- the inverse update.
//
// rank1_kernel: Sherman-Morrison in the B = A^-T convention (D:C5),
//   B'[i,:] = B[i,:] - ((B[i,:].phi' - delta_ik)/rho_D) b_old,
// row-local: a warp keeps one row in registers, shuffle-reduces the dot, rewrites the row, so B is
// read once and written once (16 n^2 bytes per accepted walker-move; HBM-bound, 0.25 flop/B).
//
// flush_kernel: delayed rank-k flush (D:C6), B <- B0 - (B0 V^T - E) S^-T C, as three chained FP64
// tensor-core GEMMs (mma.sync m8n8k4 -> DMMA.8x8x4) per 16-row strip of B0, all operands taken
// straight from global/L1 as 32- or 16-byte vectors.  The contraction index of an MMA may be
// permuted freely as long as A and B use the same permutation, and so may the column index of the
// result; both freedoms are used so that
//   - the A fragment of GEMM 1 (B0 strip) and the B fragment (V rows) are each one 32-byte load
//     per lane covering four k-steps,
//   - the accumulator tile of GEMM 1 is directly the A fragment of GEMM 2, and that of GEMM 2 the
//     A fragment of GEMM 3 (no shuffle, no shared memory),
//   - two GEMM-3 accumulator tiles interleave into four consecutive columns per lane, i.e. one
//     32-byte load of B0 and one 32-byte store of B.
#pragma once
#include "common.cuh"

namespace qmc {

constexpr int RANK1_NT = 256;
constexpr int RANK1_ROWS_PER_WARP = 4;

// NV = double2 vectors per lane (row length <= 64 NV). grid = (ceil(n / (8*ROWS_PER_WARP)), W).
template <typename T, int NV>
__global__ void __launch_bounds__(RANK1_NT) rank1_kernel(CrowdDev d, int k)
{
  const int w = blockIdx.y;
  if (!d.accepted[w]) return;
  const int ns = d.ns, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int spin = k / d.n, kk = k - spin * d.n;
  double* B = d.Binv + ((size_t)w * 2 + spin) * ns * ns;
  const double* bo = d.brow + (size_t)w * ns;
  const T* phi = static_cast<const T*>(d.vgl) + (size_t)w * 5 * ns;
  const double inv_rho = 1.0 / d.rho_d[w];
  double2 ph[NV], bold[NV];
#pragma unroll
  for (int v = 0; v < NV; ++v) {
    const int j = 2 * (lane + 32 * v);
    if (j < ns) {
      ph[v] = make_double2((double)phi[j], (double)phi[j + 1]);
      bold[v] = *reinterpret_cast<const double2*>(bo + j);
    } else {
      ph[v] = make_double2(0.0, 0.0);
      bold[v] = make_double2(0.0, 0.0);
    }
  }
  const int row0 = (blockIdx.x * (RANK1_NT / 32) + warp) * RANK1_ROWS_PER_WARP;
#pragma unroll
  for (int rr = 0; rr < RANK1_ROWS_PER_WARP; ++rr) {
    const int i = row0 + rr;
    if (i >= d.n) break;
    double2* row = reinterpret_cast<double2*>(B + (size_t)i * ns);
    double2 x[NV];
    double acc = 0.0;
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      const int jj = lane + 32 * v;
      x[v] = (2 * jj < ns) ? row[jj] : make_double2(0.0, 0.0);
      acc = fma(x[v].x, ph[v].x, acc);
      acc = fma(x[v].y, ph[v].y, acc);
    }
    acc = warp_sum(acc);
    const double f = (acc - (i == kk ? 1.0 : 0.0)) * inv_rho;
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      const int jj = lane + 32 * v;
      if (2 * jj < ns) {
        x[v].x = fma(-f, bold[v].x, x[v].x);
        x[v].y = fma(-f, bold[v].y, x[v].y);
        row[jj] = x[v];
      }
    }
  }
}

// Generic row length: two passes over the row (second one hits L1).
template <typename T>
__global__ void __launch_bounds__(RANK1_NT) rank1_generic_kernel(CrowdDev d, int k)
{
  const int w = blockIdx.y;
  if (!d.accepted[w]) return;
  const int ns = d.ns, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int spin = k / d.n, kk = k - spin * d.n;
  double* B = d.Binv + ((size_t)w * 2 + spin) * ns * ns;
  const double* bo = d.brow + (size_t)w * ns;
  const T* phi = static_cast<const T*>(d.vgl) + (size_t)w * 5 * ns;
  const double inv_rho = 1.0 / d.rho_d[w];
  const int row0 = (blockIdx.x * (RANK1_NT / 32) + warp) * RANK1_ROWS_PER_WARP;
  for (int rr = 0; rr < RANK1_ROWS_PER_WARP; ++rr) {
    const int i = row0 + rr;
    if (i >= d.n) break;
    double* row = B + (size_t)i * ns;
    double acc = 0.0;
    for (int j = lane; j < ns; j += 32) acc = fma(row[j], (double)phi[j], acc);
    acc = warp_sum(acc);
    const double f = (acc - (i == kk ? 1.0 : 0.0)) * inv_rho;
    for (int j = lane; j < ns; j += 32) row[j] = fma(-f, bo[j], row[j]);
  }
}

constexpr int FLUSH_NT = 128;          // 4 warps
constexpr int FLUSH_ROWS_PER_WARP = 16;  // two 8-row MMA blocks

__device__ __forceinline__ void ld32(const double* p, double (&v)[4])
{
  const double2 a = *reinterpret_cast<const double2*>(p);
  const double2 b = *reinterpret_cast<const double2*>(p + 2);
  v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
}

// KB = kdp / 8. grid = (ceil(ns / 64), W).
template <int KB>
__global__ void __launch_bounds__(FLUSH_NT) flush_kernel(CrowdDev d, int spin)
{
  const int w = blockIdx.y;
  const int m = d.mwin[w];
  if (m == 0) return;
  const int ns = d.ns, kdp = d.kdp;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const int row0 = (blockIdx.x * (FLUSH_NT / 32) + warp) * FLUSH_ROWS_PER_WARP;
  if (row0 >= ns) return;
  double* B = d.Binv + ((size_t)w * 2 + spin) * ns * ns;
  const double* V = d.V + (size_t)w * kdp * ns;
  const double* C = d.C + (size_t)w * kdp * ns;
  const double* Sinv = d.Sinv + (size_t)w * kdp * kdp;
  const int* rows = d.rows + (size_t)w * kdp;
  const int mb = (m + 7) >> 3;  // 8-wide blocks of the window that hold accepted moves

  // GEMM 1: Wm = B0_strip V^T. acc[i][b] = tile (rows row0+8i.., window columns 8b..8b+7);
  // lane holds (row g, columns 8b+2t, 8b+2t+1).
  double acc[2][KB][2];
#pragma unroll
  for (int i = 0; i < 2; ++i)
#pragma unroll
    for (int b = 0; b < KB; ++b) acc[i][b][0] = acc[i][b][1] = 0.0;
  const double* a0p = B + (size_t)(row0 + g) * ns + 4 * t;
  const double* a1p = a0p + (size_t)8 * ns;
  for (int s = 0; s < ns; s += 16) {
    double a0[4], a1[4];
    ld32(a0p + s, a0);
    ld32(a1p + s, a1);
#pragma unroll
    for (int b = 0; b < KB; ++b) {
      if (b < mb) {
        const int l = 8 * b + g;
        double v[4] = {0.0, 0.0, 0.0, 0.0};
        if (l < m) ld32(V + (size_t)l * ns + s + 4 * t, v);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          dmma884(acc[0][b], a0[q], v[q]);
          dmma884(acc[1][b], a1[q], v[q]);
        }
      }
    }
  }
  // minus E: E[rows[l]][l] = 1
#pragma unroll
  for (int b = 0; b < KB; ++b) {
    if (b < mb) {
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int l = 8 * b + 2 * t + e;
        const int rl = (l < m) ? rows[l] : -1;
        if (rl == row0 + g) acc[0][b][e] -= 1.0;
        if (rl == row0 + 8 + g) acc[1][b][e] -= 1.0;
      }
    }
  }
  // GEMM 2: Tm = Wm S^-T, Tm[r][c] = sum_l Wm[r][l] Sinv[c][l]. nt = -Tm.
  double nt[2][KB][2];
#pragma unroll
  for (int i = 0; i < 2; ++i)
#pragma unroll
    for (int b = 0; b < KB; ++b) nt[i][b][0] = nt[i][b][1] = 0.0;
#pragma unroll
  for (int bc = 0; bc < KB; ++bc) {
    if (bc < mb) {
      const int c = 8 * bc + g;
#pragma unroll
      for (int b = 0; b < KB; ++b) {
        if (b < mb) {
          const int l = 8 * b + 2 * t;
          double2 sv = make_double2(0.0, 0.0);
          if (c < m) sv = *reinterpret_cast<const double2*>(Sinv + (size_t)c * kdp + l);
          if (l >= m) sv.x = 0.0;
          if (l + 1 >= m) sv.y = 0.0;
          dmma884(nt[0][bc], acc[0][b][0], sv.x);
          dmma884(nt[0][bc], acc[0][b][1], sv.y);
          dmma884(nt[1][bc], acc[1][b][0], sv.x);
          dmma884(nt[1][bc], acc[1][b][1], sv.y);
        }
      }
    }
  }
#pragma unroll
  for (int i = 0; i < 2; ++i)
#pragma unroll
    for (int b = 0; b < KB; ++b) { nt[i][b][0] = -nt[i][b][0]; nt[i][b][1] = -nt[i][b][1]; }
  // GEMM 3: B_strip = B0_strip + nt C, 16 columns at a time; tile pair (even, odd columns).
  for (int j0 = 0; j0 < ns; j0 += 16) {
    double x0[4], x1[4];
    ld32(a0p + j0, x0);
    ld32(a1p + j0, x1);
    double de0[2] = {x0[0], x0[2]}, do0[2] = {x0[1], x0[3]};
    double de1[2] = {x1[0], x1[2]}, do1[2] = {x1[1], x1[3]};
#pragma unroll
    for (int b = 0; b < KB; ++b) {
      if (b < mb) {
#pragma unroll
        for (int q = 0; q < 2; ++q) {
          const int l = 8 * b + 2 * t + q;
          double2 cv = make_double2(0.0, 0.0);
          if (l < m) cv = *reinterpret_cast<const double2*>(C + (size_t)l * ns + j0 + 2 * g);
          dmma884(de0, nt[0][b][q], cv.x);
          dmma884(do0, nt[0][b][q], cv.y);
          dmma884(de1, nt[1][b][q], cv.x);
          dmma884(do1, nt[1][b][q], cv.y);
        }
      }
    }
    double* o0 = B + (size_t)(row0 + g) * ns + j0 + 4 * t;
    double* o1 = o0 + (size_t)8 * ns;
    *reinterpret_cast<double2*>(o0) = make_double2(de0[0], do0[0]);
    *reinterpret_cast<double2*>(o0 + 2) = make_double2(de0[1], do0[1]);
    *reinterpret_cast<double2*>(o1) = make_double2(de1[0], do1[0]);
    *reinterpret_cast<double2*>(o1 + 2) = make_double2(de1[1], do1[1]);
  }
}

}  // namespace qmc
