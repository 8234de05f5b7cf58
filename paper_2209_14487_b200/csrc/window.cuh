// window.cuh -- qmc_sweep with a delayed update: one launch per delay window, one CTA per walker.
//
// The crowd advances in lock-step per *window* (D:C6 schedule): a CTA owns one walker for the
// cnt <= delay_rank consecutive moves k0 .. k0+cnt-1 (row/proposal, spline, ratio, decision, append
// for each), then the whole crowd flushes (update.cuh).  Walkers never interact inside a window, so
// no kernel boundary is needed between moves: an SM overlaps the DRAM-bound spline gather of one
// walker with the fp64 work of its other resident walkers, the per-walker state (positions, inverse
// row, orbitals at r', S^-1, the table T) lives in shared memory for the whole window, and the launch
// tail is paid once per window instead of twice per move.
//
// Because the electrons of a window are consecutive, the rows B0[k0 .. k0+cnt) the window will ever
// need (as proposal rows and, once accepted, as rows of C) form one contiguous block `blk` of the
// transposed inverse that nobody writes before the flush.  On an accepted move l (orbital vector
// V[l] = phi') the kernel takes ONE pass over that block, T[l][i] = blk[i] . V[l], which yields
//   - p_l = V[l] . B0[k] for every later move k = k0 + i of the window     (column i of T),
//   - q_j = C[j] . phi' = blk[i_j] . V[l] for the earlier accepted rows     (entries T[l][i_j]),
//   - the corner B0[k] . phi'                                                (entry T[l][i]).
// So V is only written (for the flush GEMM), C is never materialised (C[l] = blk[i_l]), and a move
// reads the block twice (axpy for the row, T pass on accept) instead of V + C + C.
// The dots use the same lane/shuffle summation trees as the step kernels (move.cuh), so qmc_sweep and
// the three step calls give bit-identical trajectories.
#pragma once
#include "move.cuh"

namespace qmc {

#ifndef QMC_WIN_MIN_CTAS
#define QMC_WIN_MIN_CTAS (512 / QMC_MOVE_NT)
#endif

// Shared-memory layout of the window kernel, offsets in doubles.
struct WinLayout {
  int R, b, Sinv, Tm, p, y, q, z, red, mv, misc, rows, vgl, total;
};
__host__ __device__ inline WinLayout win_layout(int N, int ns, int kdp, int elem)
{
  WinLayout L;
  int o = 0;
  L.R = o; o += 3 * N;               // positions of the walker
  L.b = o; o += ns;                  // inverse row of the move, window applied
  L.Sinv = o; o += kdp * (kdp + 1);  // S^-1, row stride kdp + 1 (bank spread)
  L.Tm = o; o += kdp * kdp;          // T[l][i] = blk[i] . V[l]
  L.p = o; o += kdp;
  L.y = o; o += kdp;
  L.q = o; o += kdp;
  L.z = o; o += kdp;
  L.red = o; o += MOVE_RED;
  L.mv = o; o += MOVE_MV;
  L.misc = o; o += 16;
  L.rows = o; o += kdp / 2;          // int[kdp]: window-local index of accepted move l
  o = (o + 1) & ~1;
  L.vgl = o; o += (5 * ns * elem + 7) / 8;  // orbitals at r': T[5][ns]
  L.total = o;
  return L;
}

__device__ __forceinline__ double2 ld_x2(const float* v, int jj)
{
  const float2 f = reinterpret_cast<const float2*>(v)[jj];
  return make_double2((double)f.x, (double)f.y);
}
__device__ __forceinline__ double2 ld_x2(const double* v, int jj) { return reinterpret_cast<const double2*>(v)[jj]; }

__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// dynamic smem: win_layout(...).total doubles.  Requires an empty window on entry (qmc_sweep flushes first).
template <typename T>
__global__ void __launch_bounds__(MOVE_NT, QMC_WIN_MIN_CTAS) window_kernel(CrowdDev d, int k0, int cnt)
{
  extern __shared__ double sm[];
  __shared__ SplineW<T> sw;
  const int w = blockIdx.x, ns = d.ns, kdp = d.kdp, ss = kdp + 1, tid = threadIdx.x;
  const WinLayout L = win_layout(d.N, ns, kdp, (int)sizeof(T));
  double* R_s = sm + L.R;
  double* b_s = sm + L.b;
  double* Sinv_s = sm + L.Sinv;
  double* T_s = sm + L.Tm;
  double* p_s = sm + L.p;
  double* y_s = sm + L.y;
  double* q_s = sm + L.q;
  double* z_s = sm + L.z;
  double* red = sm + L.red;
  double* misc = sm + L.misc;
  int* rows_s = reinterpret_cast<int*>(sm + L.rows);
  T* vgl_s = reinterpret_cast<T*>(sm + L.vgl);
  const MoveScal ms = move_scal_smem(sm + L.mv);

  const int spin = k0 / d.n, kk0 = k0 - spin * d.n;
  const double* blk = d.Binv + (((size_t)w * 2 + spin) * ns + kk0) * ns;
  double* Rg = d.R + (size_t)w * d.N * 3;
  T* cache0 = static_cast<T*>(d.cache) + ((size_t)w * d.N + k0) * 4 * ns;
  double* V = d.V + (size_t)w * kdp * ns;

  // prologue: positions to shared memory; pull the block and the first gradient cache into L2
  for (int j = tid; j < 3 * d.N; j += MOVE_NT) R_s[j] = Rg[j];
  {
    const int lines_blk = cnt * ns * 8 / 128, lines_c = 3 * ns * (int)sizeof(T) / 128;
    for (int j = tid; j < lines_blk + lines_c; j += MOVE_NT)
      prefetch_l2(j < lines_blk ? reinterpret_cast<const char*>(blk) + (size_t)j * 128
                                : reinterpret_cast<const char*>(cache0) + (size_t)(j - lines_blk) * 128);
  }
  int m = 0;
  unsigned long long accmask = 0ull;  // window-local indices accepted so far (uniform across the CTA)
  __syncthreads();

  for (int i = 0; i < cnt; ++i) {
    const int k = k0 + i;
    T* cache = cache0 + (size_t)i * 4 * ns;
    if (i + 1 < cnt) {  // next move's gradient cache: first-touch DRAM lines
      const int lines_c = 3 * ns * (int)sizeof(T) / 128;
      for (int j = tid; j < lines_c; j += MOVE_NT) prefetch_l2(reinterpret_cast<const char*>(cache + 4 * ns) + (size_t)j * 128);
    }
    // ---- row with the window applied (D:C6) ----
    for (int j = tid; j < ns; j += MOVE_NT) b_s[j] = blk[(size_t)i * ns + j];
    if (m > 0) {
      for (int l = tid; l < m; l += MOVE_NT) p_s[l] = T_s[l * kdp + i];  // electron k is not in the window yet
      __syncthreads();
      sinv_matvec(Sinv_s, ss, m, p_s, y_s);
      __syncthreads();
      axpy_rows(b_s, ns, m, y_s, [&](int l) { return blk + (size_t)rows_s[l] * ns; });
    }
    __syncthreads();
    // ---- G_k(R), proposal, orbitals at r', ratio, decision ----
    dev_gold_propose<T>(d, w, k, b_s, cache, R_s, nullptr, ms, red);
    spline_cta<T, MOVE_NT>(d, ms.rn, sw, vgl_s);
    __syncthreads();
    dev_ratio_grad<T>(d, w, k, b_s, vgl_s, R_s, ms, nullptr, nullptr, red);
    if (dev_decide(d, w, k, ms, nullptr)) {
      for (int j = tid; j < 4 * ns; j += MOVE_NT) cache[j] = vgl_s[ns + j];
      if (tid < 3) {
        const double x = ms.rn[tid];
        R_s[3 * k + tid] = x;
        Rg[3 * k + tid] = x;
      }
      for (int j = tid; j < ns; j += MOVE_NT) V[(size_t)m * ns + j] = (double)vgl_s[j];
      // T[m][i'] = blk[i'] . phi' for every row still needed: later moves, this move, accepted rows
      rows_dot<4>(cnt, ns,
                  [&](int ip) { return (ip >= i || ((accmask >> ip) & 1ull)) ? blk + (size_t)ip * ns : nullptr; },
                  [&](int jj) { return ld_x2(vgl_s, jj); },
                  [&](int ip, double acc) { T_s[m * kdp + ip] = acc; });
      __syncthreads();
      for (int l = tid; l < m; l += MOVE_NT) q_s[l] = T_s[m * kdp + rows_s[l]];
      if (tid == 0) misc[0] = T_s[m * kdp + i];
      __syncthreads();
      sinv_border(Sinv_s, ss, m, q_s, y_s, z_s, misc);
      if (tid == 0) rows_s[m] = i;
      accmask |= 1ull << i;
      ++m;
    }
    __syncthreads();
  }

  // epilogue: what the flush needs, in the global layout of the step path
  double* Sinv = d.Sinv + (size_t)w * kdp * kdp;
  for (int e = tid; e < m * m; e += MOVE_NT) {
    const int a = e / m, b = e - a * m;
    Sinv[(size_t)a * kdp + b] = Sinv_s[a * ss + b];
  }
  for (int l = tid; l < m; l += MOVE_NT) d.rows[(size_t)w * kdp + l] = kk0 + rows_s[l];
  if (tid == 0) d.mwin[w] = m;
}

}  // namespace qmc
