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

constexpr int FLUSH_NT = 128;            // 4 warps
constexpr int FLUSH_ROWS_PER_WARP = 16;  // two 8-row MMA blocks
constexpr int FINALIZE_NT = 128;

__device__ __forceinline__ void ld32(const double* p, double (&v)[4])
{
  const double2 a = *reinterpret_cast<const double2*>(p);
  const double2 b = *reinterpret_cast<const double2*>(p + 2);
  v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
}

// Flush, step 1 (per walker, column-local, in place): C <- Z = S^-T C, Z[l][j] = sum_q Sinv[q][l] C[q][j],
// so that the strip kernel needs two GEMMs only: B <- B0 - (B0 V^T - E) Z.  A thread owns one column j
// and up to 32 output rows l in registers, streams C[q][j] once, and reads Sinv from shared memory
// as warp-wide broadcasts; all reads of a column finish (barrier) before it is overwritten.
// 2 k^2 n flop per walker (4 % of the flush at k = 32, n = 384), done once instead of once per strip.
// grid = (ceil(ns / (FINALIZE_NT / LH)), W), LH = KDP / min(KDP, 32); dynamic smem: KDP*KDP doubles
template <int KDP>
__global__ void __launch_bounds__(FINALIZE_NT) flush_finalize_kernel(CrowdDev d)
{
  constexpr int ZL = KDP < 32 ? KDP : 32;
  constexpr int LH = KDP / ZL;
  constexpr int COLS = FINALIZE_NT / LH;
  extern __shared__ double s_sinv[];
  const int w = blockIdx.y;
  const int m = d.mwin[w];
  if (m == 0) return;
  const int ns = d.ns;
  const double* Sinv = d.Sinv + (size_t)w * KDP * KDP;
  for (int e = threadIdx.x; e < KDP * KDP; e += FINALIZE_NT) s_sinv[e] = Sinv[e];
  __syncthreads();
  const int half = threadIdx.x / COLS;
  const int j = blockIdx.x * COLS + (threadIdx.x - half * COLS);
  const int l0 = half * ZL;
  double* C = d.C + (size_t)w * KDP * ns + j;
  double z[ZL];
#pragma unroll
  for (int l = 0; l < ZL; ++l) z[l] = 0.0;
  if (j < ns && l0 < m) {
#pragma unroll 2
    for (int q = 0; q < m; ++q) {
      const double c = C[(size_t)q * ns];
#pragma unroll
      for (int l = 0; l < ZL; ++l) z[l] = fma(s_sinv[q * KDP + l0 + l], c, z[l]);
    }
  }
  __syncthreads();
  if (j < ns) {
#pragma unroll
    for (int l = 0; l < ZL; ++l)
      if (l0 + l < m) C[(size_t)(l0 + l) * ns] = z[l];
  }
}

// ---- operand streams of the strip kernel: a cp.async ring in shared memory ---------------------
// Per 16-column chunk a CTA of 4 warps (64 strip rows) needs
//   - per warp: 16 rows x 128 B of the B0 strip (GEMM-1 A fragments; again as GEMM-2 accumulator init),
//   - per CTA:  the chunk of V (GEMM 1) or of Z (GEMM 2): kdp rows x 128 B, shared by the 4 warps.
// The strip comes from DRAM and V/Z from L2; both latencies are far longer than one chunk of DMMAs,
// so everything is streamed FLUSH_DEPTH-1 chunks ahead with 16-byte cp.async (each warp instruction
// moves full 128-byte row segments) into a ring of stages.  Pieces are placed so that every fragment
// read is one conflict-free LDS.128:
//   strip piece (row r of block i, 16-byte column c)  -> [i][c & 1][4 r + c / 2]      (lane g = r, t = c / 2)
//   V piece (window row l, column c)                  -> [l / 8][c & 1][4 (l % 8) + c / 2]
//   Z piece (window row l, column c)                  -> [l / 8][l & 1][4 c + (l % 8) / 2]  (lane g = c, t = (l % 8) / 2)
constexpr int FLUSH_DEPTH = 6;
constexpr int FLUSH_WARPS = FLUSH_NT / 32;
constexpr int FLUSH_STRIP_BYTES = 2 * 2 * 32 * 16;  // per warp and stage

__device__ __forceinline__ void cp_async16(unsigned smem_addr, const void* gptr)
{
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_addr), "l"(gptr) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <int KB>
struct FlushStage {
  static constexpr int VZ_BYTES = KB * 1024;                              // kdp rows x 128 B
  static constexpr int BYTES = FLUSH_WARPS * FLUSH_STRIP_BYTES + VZ_BYTES;
};

__device__ __forceinline__ void lds32(const unsigned char* p, double (&r)[4])
{
  const double2 a = *reinterpret_cast<const double2*>(p), b = *reinterpret_cast<const double2*>(p + 512);
  r[0] = a.x; r[1] = a.y; r[2] = b.x; r[3] = b.y;
}

// Flush, step 2: B_strip <- B0_strip - (B0_strip V^T - E) Z.  KB = kdp / 8. grid = (ceil(ns / 64), W).
// dynamic smem: FLUSH_DEPTH * FlushStage<KB>::BYTES
template <int KB>
__global__ void __launch_bounds__(FLUSH_NT, 2) flush_kernel(CrowdDev d, int spin)
{
  extern __shared__ __align__(16) unsigned char ring[];
  constexpr int STAGE = FlushStage<KB>::BYTES;
  constexpr int NPV = (KB * 64 + FLUSH_NT - 1) / FLUSH_NT;  // V/Z pieces per thread and chunk
  const int w = blockIdx.y;
  const int m = d.mwin[w];
  if (m == 0) return;
  const int ns = d.ns, kdp = d.kdp, nch = ns / 16;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const int row0 = (blockIdx.x * FLUSH_WARPS + warp) * FLUSH_ROWS_PER_WARP;
  const bool strip_ok = row0 < ns;   // warps past the last strip still help with the V/Z copies and barriers
  double* B = d.Binv + ((size_t)w * 2 + spin) * ns * ns;
  const int* rows = d.rows + (size_t)w * kdp;
  const int mb = (m + 7) >> 3;  // 8-wide blocks of the window that hold accepted moves
  const unsigned ring_s = (unsigned)__cvta_generic_to_shared(ring);

  // ---- per-thread copy plan (loop invariant): 4 strip pieces, NPV pieces of V / Z ----
  const double* s_src[4];
  unsigned s_dst[4];
#pragma unroll
  for (int i = 0; i < 2; ++i)
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      const int p = 32 * j + lane, r = p >> 3, c16 = p & 7;
      s_src[2 * i + j] = B + (size_t)((strip_ok ? row0 : 0) + 8 * i + r) * ns + 2 * c16;
      s_dst[2 * i + j] = (unsigned)(warp * FLUSH_STRIP_BYTES + i * 1024 + (c16 & 1) * 512 + (r * 4 + (c16 >> 1)) * 16);
    }
  const double* v_src[NPV];
  const double* z_src[NPV];
  unsigned v_dst[NPV], z_dst[NPV];
  bool vz_ok[NPV];
#pragma unroll
  for (int it = 0; it < NPV; ++it) {
    const int p = it * FLUSH_NT + threadIdx.x;
    const int l = p >> 3, c16 = p & 7, b = l >> 3, r = l & 7;
    vz_ok[it] = p < KB * 64 && l < m;   // rows at or beyond m keep the zeros written below
    v_src[it] = d.V + ((size_t)w * kdp + (vz_ok[it] ? l : 0)) * ns + 2 * c16;
    z_src[it] = d.C + ((size_t)w * kdp + (vz_ok[it] ? l : 0)) * ns + 2 * c16;
    v_dst[it] = (unsigned)(FLUSH_WARPS * FLUSH_STRIP_BYTES + b * 1024 + (c16 & 1) * 512 + (r * 4 + (c16 >> 1)) * 16);
    z_dst[it] = (unsigned)(FLUSH_WARPS * FLUSH_STRIP_BYTES + b * 1024 + (r & 1) * 512 + (c16 * 4 + (r >> 1)) * 16);
  }
  // zero the ring once: window rows >= m are never copied, so their V slots read as 0 (their Z slots
  // may later hold stale finite V data, which only ever multiplies the exact zeros of nw)
  for (int e = threadIdx.x; e < FLUSH_DEPTH * STAGE / 16; e += FLUSH_NT)
    *reinterpret_cast<double2*>(ring + (size_t)e * 16) = make_double2(0.0, 0.0);
  __syncthreads();

  // seq q in [0, 2 nch): chunk q mod nch; first pass carries V (GEMM 1), second pass Z (GEMM 2)
  auto issue = [&](int q, unsigned st) {
    if (q < 2 * nch) {
      const bool first = q < nch;
      const int off = 16 * (first ? q : q - nch);
      if (strip_ok) {
#pragma unroll
        for (int e = 0; e < 4; ++e) cp_async16(ring_s + st + s_dst[e], s_src[e] + off);
      }
#pragma unroll
      for (int it = 0; it < NPV; ++it)
        if (vz_ok[it]) cp_async16(ring_s + st + (first ? v_dst[it] : z_dst[it]), (first ? v_src[it] : z_src[it]) + off);
    }
    cp_async_commit();  // always, so that group counting stays uniform
  };
#pragma unroll
  for (int q = 0; q < FLUSH_DEPTH - 1; ++q) issue(q, (unsigned)(q * STAGE));

  const unsigned char* my_strip = ring + warp * FLUSH_STRIP_BYTES + lane * 16;
  const unsigned char* my_vz = ring + FLUSH_WARPS * FLUSH_STRIP_BYTES + lane * 16;
  unsigned st_rd = 0, st_wr = (FLUSH_DEPTH - 1) * STAGE;   // stage being consumed / refilled

  // GEMM 1: Wm = B0_strip V^T. acc[i][b] = tile (rows row0+8i.., window columns 8b..8b+7);
  // lane holds (row g, columns 8b+2t, 8b+2t+1).
  double acc[2][KB][2];
#pragma unroll
  for (int i = 0; i < 2; ++i)
#pragma unroll
    for (int b = 0; b < KB; ++b) acc[i][b][0] = acc[i][b][1] = 0.0;
  for (int q = 0; q < nch; ++q) {
    cp_async_wait<FLUSH_DEPTH - 2>();
    __syncthreads();   // stage q landed for everyone; everyone is done reading stage q-1
    issue(q + FLUSH_DEPTH - 1, st_wr);
    if (strip_ok) {
      double a0[4], a1[4], v[KB][4];
      lds32(my_strip + st_rd, a0);
      lds32(my_strip + st_rd + 1024, a1);
#pragma unroll
      for (int b = 0; b < KB; ++b)
        if (b < mb) lds32(my_vz + st_rd + b * 1024, v[b]);
      // k-step outermost: 2 KB independent accumulator chains between dependent DMMAs
#pragma unroll
      for (int kq = 0; kq < 4; ++kq)
#pragma unroll
        for (int b = 0; b < KB; ++b)
          if (b < mb) {
            dmma884(acc[0][b], a0[kq], v[b][kq]);
            dmma884(acc[1][b], a1[kq], v[b][kq]);
          }
    }
    st_rd = st_rd + STAGE == FLUSH_DEPTH * STAGE ? 0u : st_rd + STAGE;
    st_wr = st_wr + STAGE == FLUSH_DEPTH * STAGE ? 0u : st_wr + STAGE;
  }
  // minus E (E[rows[l]][l] = 1), then negate: nw = -(B0 V^T - E)
#pragma unroll
  for (int b = 0; b < KB; ++b) {
    if (b < mb) {
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int l = 8 * b + 2 * t + e;
        const int rl = (l < m) ? rows[l] : -1;
        acc[0][b][e] = (rl == row0 + g ? 1.0 : 0.0) - acc[0][b][e];
        acc[1][b][e] = (rl == row0 + 8 + g ? 1.0 : 0.0) - acc[1][b][e];
      }
    }
  }
  // GEMM 2: B_strip = B0_strip + nw Z, 16 columns at a time.  Even / odd columns of the chunk are
  // separate tiles (a lane ends up with 4 consecutive columns); two accumulator sets (even / odd
  // window blocks) give 8 independent DMMA chains, summed at the end.
  double* o0 = B + (size_t)(row0 + g) * ns + 4 * t;   // the same 32 bytes per row the lane took as accumulators
  double* o1 = o0 + (size_t)8 * ns;
  for (int c = 0; c < nch; ++c) {
    cp_async_wait<FLUSH_DEPTH - 2>();
    __syncthreads();
    issue(nch + c + FLUSH_DEPTH - 1, st_wr);
    if (strip_ok) {
      double x0[4], x1[4];
      double2 z[KB][2];
      lds32(my_strip + st_rd, x0);
      lds32(my_strip + st_rd + 1024, x1);
#pragma unroll
      for (int b = 0; b < KB; ++b)
        if (b < mb) {
          z[b][0] = *reinterpret_cast<const double2*>(my_vz + st_rd + b * 1024);
          z[b][1] = *reinterpret_cast<const double2*>(my_vz + st_rd + b * 1024 + 512);
        }
      double de0[2] = {x0[0], x0[2]}, do0[2] = {x0[1], x0[3]};
      double de1[2] = {x1[0], x1[2]}, do1[2] = {x1[1], x1[3]};
      double ee0[2] = {0.0, 0.0}, eo0[2] = {0.0, 0.0}, ee1[2] = {0.0, 0.0}, eo1[2] = {0.0, 0.0};
#pragma unroll
      for (int kq = 0; kq < 2; ++kq)
#pragma unroll
        for (int b = 0; b < KB; ++b)
          if (b < mb) {
            if (b & 1) {
              dmma884(ee0, acc[0][b][kq], z[b][kq].x);
              dmma884(eo0, acc[0][b][kq], z[b][kq].y);
              dmma884(ee1, acc[1][b][kq], z[b][kq].x);
              dmma884(eo1, acc[1][b][kq], z[b][kq].y);
            } else {
              dmma884(de0, acc[0][b][kq], z[b][kq].x);
              dmma884(do0, acc[0][b][kq], z[b][kq].y);
              dmma884(de1, acc[1][b][kq], z[b][kq].x);
              dmma884(do1, acc[1][b][kq], z[b][kq].y);
            }
          }
      *reinterpret_cast<double2*>(o0 + 16 * c) = make_double2(de0[0] + ee0[0], do0[0] + eo0[0]);
      *reinterpret_cast<double2*>(o0 + 16 * c + 2) = make_double2(de0[1] + ee0[1], do0[1] + eo0[1]);
      *reinterpret_cast<double2*>(o1 + 16 * c) = make_double2(de1[0] + ee1[0], do1[0] + eo1[0]);
      *reinterpret_cast<double2*>(o1 + 16 * c + 2) = make_double2(de1[1] + ee1[1], do1[1] + eo1[1]);
    }
    st_rd = st_rd + STAGE == FLUSH_DEPTH * STAGE ? 0u : st_rd + STAGE;
    st_wr = st_wr + STAGE == FLUSH_DEPTH * STAGE ? 0u : st_wr + STAGE;
  }
  cp_async_wait<0>();
}

}  // namespace qmc
