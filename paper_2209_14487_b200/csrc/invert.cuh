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

// ---- blocked variant (the one qmc_crowd_create uses when its shared memory fits) -----------------
// Same elimination, same pivot choices as invert_kernel, but right-looking in panels of INVB_NB columns so that the
// matrix is swept 2 n / NB times instead of 2 n times (the unblocked kernel is bound by that traffic: 3.7 TB at
// cfg 5 / W = 4096):
//   (a) the panel (n x NB) is loaded into shared memory and eliminated there in place (in sub-panels of INVB_SB
//       columns): afterwards it holds the NB columns X_G of the composite Gauss-Jordan operator G of the panel;
//   (b) the panel's row swaps are applied to all other columns (column-local, no barrier);
//   (c) every other column block is updated with one FP64 tensor-core GEMM,
//       A[:, o] <- A[:, o] + (X_G - E_K) A_K[:, o]   (rows of K: A[K, o] <- X_G[K, :] A_K[:, o]);
//   (d) at the end the row swaps are undone as column swaps, last first: the kernel inverts P A, and
//       (P A)^-1 = A^-1 P^T.
// Two CTAs of 256 threads per SM: the pivot rows A_K are not staged in shared memory (a warp owns a 16-column block of
// the trailing update, keeps its A_K fragments in registers for all row tiles and finishes with the rows of K of that
// block, which nobody else reads), the panel uses a row stride of 34 doubles, and the dependent chain of pivot steps of
// one matrix runs under the memory-bound trailing update of the other.  (A first version with one CTA of 512 threads per
// SM and A_K staged in shared memory was 22 % slower and is gone: DESIGN.md section 8.)
constexpr int INVB_NB = 32;
constexpr int INVB_SB = 8;            // sub-panel width inside the shared-memory panel
constexpr int INVB2_NT = 256;
constexpr int INVB2_XS = INVB_NB + 2;   // 2 g + t: every double-bank hit twice by the DMMA fragment loads

inline __host__ __device__ size_t invert_blocked2_smem(int ns)
{
  return ((size_t)ns * INVB2_XS + INVB_SB * INVB_NB + ns + 2 * (INVB2_NT / 32)) * 8 + (size_t)ns * 4 + 64;
}

__global__ void __launch_bounds__(INVB2_NT, 2) invert_blocked2_kernel(CrowdDev d)
{
  extern __shared__ double sm[];
  const int ns = d.ns, n = d.n, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  double* XG = sm;                                  // [ns][INVB2_XS]
  double* AKs = XG + (size_t)ns * INVB2_XS;         // [SB][NB] pivot rows of a sub-panel
  double* colf = AKs + INVB_SB * INVB_NB;           // [ns] (the column relabelling at the end)
  double* redv = colf + ns;
  int* redi = reinterpret_cast<int*>(redv + INVB2_NT / 32);
  int* piv = redi + INVB2_NT / 32;
  __shared__ int s_bad;
  double* X = d.Binv + (size_t)blockIdx.x * ns * ns;
  if (tid == 0) s_bad = 0;
  __syncthreads();
  for (int c0 = 0; c0 < n; c0 += INVB_NB) {
    const int nb = min(INVB_NB, n - c0);
    // (a) panel into shared memory (zero padded), eliminated there in place
    for (int e = tid; e < ns * INVB_NB; e += INVB2_NT) {
      const int r = e / INVB_NB, j = e - r * INVB_NB;
      XG[r * INVB2_XS + j] = (r < n && j < nb) ? X[(size_t)r * ns + c0 + j] : 0.0;
    }
    __syncthreads();
    // The panel itself is eliminated in sub-panels of INVB_SB columns, the same right-looking scheme one level down:
    // a pivot step touches n x SB elements (a warp takes four rows at a time, lane = (row, sub-panel column), the
    // multiplier of a row is a shuffle, the row interchange is done on register copies of rows c and p, the search
    // for the next pivot rides on the update), and after each sub-panel the other 32 - SB panel columns get its row
    // swaps and one rank-SB update.  (Eliminating all 32 columns at every pivot step cost 67 of the kernel's 139 ms at
    // cfg 5, W = 4096.)
    constexpr int NW = INVB2_NT / 32, SB = INVB_SB, RPW = 32 / SB;   // RPW rows per warp pass
    static_assert(INVB_NB == 32 && SB == 8, "lane = panel column; four rows x eight columns per warp pass");
    const int rsub = lane / SB, col = lane % SB, lbase = lane - col;
    bool bad = false;
    for (int s0 = 0; s0 < nb && !bad; s0 += SB) {
      const int sb = min(SB, nb - s0);
      {  // pivot candidates of the sub-panel's first column
        double best = -1.0;
        int bi = c0 + s0;
        for (int r = c0 + s0 + tid; r < n; r += INVB2_NT) {
          double v = fabs(XG[r * INVB2_XS + s0]);
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
      }
      for (int jl = 0; jl < sb; ++jl) {
        const int c = c0 + s0 + jl;
        __syncthreads();   // the partial maxima of this column (and the previous step's update) are complete
        // every warp reduces the NW partial maxima itself: one shared-memory read per lane and a shuffle tree
        double bv = redv[lane & (NW - 1)];
        int p = redi[lane & (NW - 1)];
#pragma unroll
        for (int o = NW / 2; o > 0; o >>= 1) {
          const double ov = __shfl_xor_sync(0xffffffffu, bv, o);
          const int oi = __shfl_xor_sync(0xffffffffu, p, o);
          if (ov > bv || (ov == bv && oi < p)) { bv = ov; p = oi; }
        }
        if (tid == 0) piv[c] = p;
        if (!(bv > 0.0) || !isfinite(bv)) { bad = true; break; }   // uniform over the CTA
        const double prow = XG[p * INVB2_XS + s0 + col], crow = XG[c * INVB2_XS + s0 + col];
        const double pv = __shfl_sync(0xffffffffu, prow, lbase + jl);
        const double rc = ((col == jl) ? 1.0 : prow) / pv;   // a true division (see above), one per lane
        __syncthreads();   // rows c and p are in registers everywhere; the partial maxima have been read
        double best = -1.0;
        int bi = c + 1;
        for (int rb = warp * RPW; rb < n; rb += 4 * RPW * NW) {   // warp-uniform trip count; four independent row groups
          const int r0 = rb + rsub;
          double v[4];
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const int r = r0 + i * RPW * NW;
            v[i] = (r < n) ? XG[r * INVB2_XS + s0 + col] : 0.0;
            v[i] = (r == p) ? crow : v[i];   // row p receives the old row c
          }
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const int r = r0 + i * RPW * NW;
            const double cf = __shfl_sync(0xffffffffu, v[i], lbase + jl);
            double nv = fma(-cf, rc, (col == jl) ? 0.0 : v[i]);
            nv = (r == c) ? rc : nv;
            if (r < n) XG[r * INVB2_XS + s0 + col] = nv;
            double a = fabs(nv);
            a = (a == a) ? a : INFINITY;
            const bool take = r > c && r < n && (a > best || (a == best && r < bi));
            best = take ? a : best;
            bi = take ? r : bi;
          }
        }
        if (jl + 1 < sb) {   // column jl + 1 lives in the lanes col == jl + 1 of the RPW row groups
          double bj = __shfl_sync(0xffffffffu, best, lbase + jl + 1);
          int ij = __shfl_sync(0xffffffffu, bi, lbase + jl + 1);
#pragma unroll
          for (int o = SB; o < 32; o <<= 1) {
            const double ov = __shfl_xor_sync(0xffffffffu, bj, o);
            const int oi = __shfl_xor_sync(0xffffffffu, ij, o);
            if (ov > bj || (ov == bj && oi < ij)) { bj = ov; ij = oi; }
          }
          if (lane == 0) { redv[warp] = bj; redi[warp] = ij; }
        }
      }
      if (bad) break;
      __syncthreads();   // the sub-panel holds its Gauss-Jordan operator; piv[] of its columns is visible
      if (nb > sb) {
        // the sub-panel's row swaps on the other panel columns (a thread owns a column: no barrier), then its pivot
        // rows, then the rank-sb update X[:, o] <- X[:, o] + (G - E_K) A_K[:, o]  (rows of K: G[K, :] A_K[:, o])
        if (tid < INVB_NB && (tid < s0 || tid >= s0 + sb)) {
          for (int q = 0; q < sb; ++q) {
            const int c = c0 + s0 + q, p = piv[c];
            if (p != c) {
              const double x = XG[c * INVB2_XS + tid], y = XG[p * INVB2_XS + tid];
              XG[c * INVB2_XS + tid] = y;
              XG[p * INVB2_XS + tid] = x;
            }
          }
          for (int q = 0; q < sb; ++q) AKs[q * INVB_NB + tid] = XG[(c0 + s0 + q) * INVB2_XS + tid];
        }
        __syncthreads();
        const bool other = lane < s0 || lane >= s0 + sb;   // lane = panel column again, a warp owns whole rows
        double ak[SB];
#pragma unroll
        for (int q = 0; q < SB; ++q) ak[q] = (q < sb && other) ? AKs[q * INVB_NB + lane] : 0.0;
#pragma unroll 2
        for (int r = warp; r < n; r += NW) {
          const double x = XG[r * INVB2_XS + lane];
          const bool in_k = r >= c0 + s0 && r < c0 + s0 + sb;
          double acc = in_k ? 0.0 : x;
#pragma unroll
          for (int q = 0; q < SB; ++q) acc = fma(__shfl_sync(0xffffffffu, x, s0 + q), ak[q], acc);
          if (other) XG[r * INVB2_XS + lane] = acc;
        }
        __syncthreads();
      }
    }
    if (bad && tid == 0) s_bad = 1;
    __syncthreads();
    if (s_bad) break;
    // (b) the panel's row swaps on every other column (a thread owns whole columns: no barrier needed)
    for (int o = tid; o < n; o += INVB2_NT) {
      if (o >= c0 && o < c0 + nb) continue;
      for (int j = 0; j < nb; ++j) {
        const int c = c0 + j, p = piv[c];
        if (p != c) {
          const double a = X[(size_t)c * ns + o], b = X[(size_t)p * ns + o];
          X[(size_t)c * ns + o] = b;
          X[(size_t)p * ns + o] = a;
        }
      }
    }
    __syncthreads();
    // (d) trailing update by 16-column blocks: A[:, o] <- A[:, o] + (X_G - E_K) A_K[:, o], rows of K last
    {
      const int g = lane >> 2, t = lane & 3;
      const int ncb = (n + 15) / 16, nrt = (n + 31) / 32;
      for (int cb = warp; cb < ncb; cb += INVB2_NT / 32) {
        const int o0 = cb * 16;
        if (o0 >= c0 && o0 < c0 + INVB_NB) continue;   // the panel's own columns come from XG
        double bb[INVB_NB / 4][2];
#pragma unroll
        for (int q = 0; q < INVB_NB / 4; ++q)
#pragma unroll
          for (int b = 0; b < 2; ++b) {
            const int j = 4 * q + t, o = o0 + 8 * b + g;
            bb[q][b] = (j < nb && o < n) ? X[(size_t)(c0 + j) * ns + o] : 0.0;
          }
        for (int rt = 0; rt <= nrt; ++rt) {
          // row tiles in order with the tile of K skipped, then the tile of K
          const bool in_k = rt == nrt;
          const int r0 = in_k ? c0 : rt * 32;
          if (!in_k && r0 == c0) continue;
          double acc[4][2][2];
#pragma unroll
          for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int b = 0; b < 2; ++b) {
              const int r = r0 + 8 * i + g, o = o0 + 8 * b + 2 * t;
              double2 x = make_double2(0.0, 0.0);
              if (!in_k && r < n && o < ns) x = *reinterpret_cast<const double2*>(X + (size_t)r * ns + o);
              acc[i][b][0] = x.x;
              acc[i][b][1] = x.y;
            }
#pragma unroll
          for (int q = 0; q < INVB_NB / 4; ++q) {
            double a[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) a[i] = (r0 + 8 * i + g < ns) ? XG[(r0 + 8 * i + g) * INVB2_XS + 4 * q + t] : 0.0;
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
              for (int b = 0; b < 2; ++b) dmma884(acc[i][b], a[i], bb[q][b]);
          }
#pragma unroll
          for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int b = 0; b < 2; ++b) {
              const int r = r0 + 8 * i + g, o = o0 + 8 * b + 2 * t;
              if (r < n) {
                if (o < n) X[(size_t)r * ns + o] = acc[i][b][0];
                if (o + 1 < n) X[(size_t)r * ns + o + 1] = acc[i][b][1];
              }
            }
        }
      }
    }
    // the panel's own columns
    for (int e = tid; e < n * nb; e += INVB2_NT) {
      const int r = e / nb, j = e - r * nb;
      X[(size_t)r * ns + c0 + j] = XG[r * INVB2_XS + j];
    }
    __syncthreads();
  }
  if (s_bad) {
    if (tid == 0) atomicExch(d.status, 4);
    return;
  }
  // undo the row swaps as column swaps, last first
  int* src = reinterpret_cast<int*>(colf);     // [n] final column j <- current column src[j]
  for (int j = tid; j < n; j += INVB2_NT) src[j] = j;
  __syncthreads();
  if (tid == 0)
    for (int c = n - 1; c >= 0; --c) {
      const int p = piv[c];
      const int a = src[c];
      src[c] = src[p];
      src[p] = a;
    }
  __syncthreads();
  double* rowbuf = XG + (size_t)warp * ns;     // one row per warp (the panel is dead)
  for (int r = warp; r < n; r += INVB2_NT / 32) {
    for (int j = lane; j < n; j += 32) rowbuf[j] = X[(size_t)r * ns + j];
    __syncwarp();
    for (int j = lane; j < n; j += 32) X[(size_t)r * ns + j] = rowbuf[src[j]];
    __syncwarp();
  }
}

// D:R6: dst = fl32(src), four elements per thread (total % 4 == 0: ns is a multiple of 16)
__global__ void __launch_bounds__(256) narrow_kernel(float* __restrict__ dst, const double* __restrict__ src, size_t total)
{
  for (size_t e = ((size_t)blockIdx.x * 256 + threadIdx.x) * 4; e < total; e += (size_t)gridDim.x * 256 * 4) {
    const double2 a = *reinterpret_cast<const double2*>(src + e), b = *reinterpret_cast<const double2*>(src + e + 2);
    *reinterpret_cast<float4*>(dst + e) = make_float4((float)a.x, (float)a.y, (float)b.x, (float)b.y);
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
