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

// Mixed precision (D:R6): the same update on fp32-stored rows -- widened on load, updated in fp64, rounded once on store
// (8 n^2 bytes per accepted walker-move).  Two passes over the row (the second one hits L1).
template <typename T>
__global__ void __launch_bounds__(RANK1_NT) rank1_f32_kernel(CrowdDev d, int k)
{
  const int w = blockIdx.y;
  if (!d.accepted[w]) return;
  const int ns = d.ns, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int spin = k / d.n, kk = k - spin * d.n;
  float* B = d.Binv32 + ((size_t)w * 2 + spin) * ns * ns;
  const double* bo = d.brow + (size_t)w * ns;
  const T* phi = static_cast<const T*>(d.vgl) + (size_t)w * 5 * ns;
  const double inv_rho = 1.0 / d.rho_d[w];
  const int row0 = (blockIdx.x * (RANK1_NT / 32) + warp) * RANK1_ROWS_PER_WARP;
  for (int rr = 0; rr < RANK1_ROWS_PER_WARP; ++rr) {
    const int i = row0 + rr;
    if (i >= d.n) break;
    float2* row = reinterpret_cast<float2*>(B + (size_t)i * ns);
    double acc = 0.0;
    for (int jj = lane; jj < ns / 2; jj += 32) {   // same lane partition and order as rank1_kernel
      const float2 x = row[jj];
      acc = fma((double)x.x, (double)phi[2 * jj], acc);
      acc = fma((double)x.y, (double)phi[2 * jj + 1], acc);
    }
    acc = warp_sum(acc);
    const double f = (acc - (i == kk ? 1.0 : 0.0)) * inv_rho;
    for (int jj = lane; jj < ns / 2; jj += 32) {
      const float2 x = row[jj];
      const double2 b2 = *reinterpret_cast<const double2*>(bo + 2 * jj);
      row[jj] = make_float2((float)fma(-f, b2.x, (double)x.x), (float)fma(-f, b2.y, (double)x.y));
    }
  }
}

#ifndef QMC_FLUSH_MIN_CTAS
#define QMC_FLUSH_MIN_CTAS 3
#endif
#ifndef QMC_FLUSH_NT
#define QMC_FLUSH_NT 128
#endif
constexpr int FLUSH_NT = QMC_FLUSH_NT;    // one 16-row strip per warp
constexpr int FLUSH_ROWS_PER_WARP = 16;  // two 8-row MMA blocks
constexpr int FINALIZE_NT = 128;

// Four consecutive elements of the carried inverse in its storage type (D:R6): fp64, or fp32 widened on load and
// rounded to nearest on store.
__device__ __forceinline__ void ld_b4(const double* p, double (&v)[4]) { ld32(p, v); }
__device__ __forceinline__ void ld_b4(const float* p, double (&v)[4])
{
  float4 f;
  asm volatile("ld.global.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(f.x), "=f"(f.y), "=f"(f.z), "=f"(f.w) : "l"(p));
  v[0] = (double)f.x; v[1] = (double)f.y; v[2] = (double)f.z; v[3] = (double)f.w;
}
__device__ __forceinline__ void st_b4(double* p, double a, double b, double c, double d) { st32(p, a, b, c, d); }
__device__ __forceinline__ void st_b4(float* p, double a, double b, double c, double d)
{
  asm volatile("st.global.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(p), "f"((float)a), "f"((float)b), "f"((float)c), "f"((float)d) : "memory");
}
template <typename TB> __device__ __forceinline__ TB* carried_inverse(const CrowdDev& d);
template <> __device__ __forceinline__ double* carried_inverse<double>(const CrowdDev& d) { return d.Binv; }
template <> __device__ __forceinline__ float* carried_inverse<float>(const CrowdDev& d) { return d.Binv32; }

// Flush, step 1 (per walker, column-local): Z = S^-T C, Z[l][j] = sum_q Sinv[q][l] C[q][j], written to
// the d.C buffer, so that the strip kernel needs two GEMMs only: B <- B0 - (B0 V^T - E) Z.  C[q] is read
// where it lives, C[q,:] = B0[rows[q],:] (the window kernel never copies it; the strip kernel has not
// touched B0 yet).  A thread owns one column j and up to 32 output rows l in registers, streams
// C[q][j] once, and reads Sinv from shared memory as warp-wide broadcasts.
// 2 k^2 n flop per walker (4 % of the flush at k = 32, n = 384), done once instead of once per strip.
// grid = (ceil(ns / (FINALIZE_NT / LH)), W), LH = KDP / min(KDP, 32); dynamic smem: KDP*KDP doubles
template <int KDP>
__global__ void __launch_bounds__(FINALIZE_NT) flush_finalize_kernel(CrowdDev d, int spin)
{
  constexpr int ZL = KDP < 32 ? KDP : 32;
  constexpr int LH = KDP / ZL;
  constexpr int COLS = FINALIZE_NT / LH;
  extern __shared__ double s_sinv[];
  const int w = blockIdx.y + d.w0;
  const int m = d.mwin[w];
  if (m == 0) return;
  const int ns = d.ns;
  const double* Sinv = d.Sinv + (size_t)w * KDP * KDP;
  __shared__ int s_rows[KDP];
  for (int e = threadIdx.x; e < KDP * KDP; e += FINALIZE_NT) s_sinv[e] = (e / KDP < m && e % KDP < m) ? Sinv[e] : 0.0;
  for (int e = threadIdx.x; e < KDP; e += FINALIZE_NT) s_rows[e] = e < m ? d.rows[(size_t)w * KDP + e] : 0;
  __syncthreads();
  const int half = threadIdx.x / COLS;
  const int j = blockIdx.x * COLS + (threadIdx.x - half * COLS);
  const int l0 = half * ZL;
  double* C = d.C + (size_t)w * KDP * ns + j;
  const size_t B0 = ((size_t)w * 2 + spin) * ns * ns + j;
  double z[ZL];
#pragma unroll
  for (int l = 0; l < ZL; ++l) z[l] = 0.0;
  if (j < ns && l0 < m) {
#pragma unroll 2
    for (int q = 0; q < m; ++q) {
      const double c = ld_binv(d, B0 + (size_t)s_rows[q] * ns);
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

// Measured alternatives on B200 (cfg 5, W = 4096, round 1):
//  - the DMMA.8x8x4 issue ceiling with this chain structure is 37.2 TFLOP/s, and 34.4 TFLOP/s with the V and strip
//    fragments loaded straight from L1/L2 as here -- the operand path is not the limit, DRAM streaming is: the strip is
//    read twice and the second read misses L2 half the time (13.8 GB of traffic for 9.7 GB algorithmic; skipping the
//    second read shortens the flush by 0.85 ms);
//  - L2 eviction hints on the strip (evict_last on the first read, evict_first on the second read and the store) with
//    or without a persisting-L2 set-aside, and L2 / L1 prefetches of the strip 2-16 chunks ahead: no gain (the
//    set-aside slows the window kernel; with GEMM 2 walking backwards the L2 prefetch costs 0.1 ms);
//  - a K-split form (eight warps share a strip, each keeps its columns in registers, partial products summed through
//    shared memory, strip read once: 10.3 GB of traffic) ran at 5.0 ms instead of 3.3 ms: two block barriers per strip
//    and eight warps per SM leave the DMMA pipe 42 % busy;
//  - 8-row strips (half the L2 reuse distance, twice the V fragment traffic per DMMA): 4.1 ms instead of 3.7 ms;
//  - a pair of warps per strip splitting its columns (partials exchanged through shared memory, second read half a
//    strip after the first): 4.4 ms instead of 3.5 ms -- the exposed load latency at the start of each shorter
//    GEMM loop costs more than the L2 hits save.
// Round 2 (measured on B200 at cfg 5, W = 4096):
//  - the strip staged ONCE in shared memory by bulk asynchronous copies (cp.async.bulk + mbarrier, one copy per row issued
//    by a lane, rows padded by 16 bytes so that the fragment reads are conflict-free; persistent grid, one CTA per SM;
//    both GEMMs take the strip from shared memory, V / Z fragments software-pipelined 4 chunks ahead in registers at 255
//    registers per thread): correct (same tests), DRAM traffic at the algorithmic minimum, and SLOWER -- 8-row strips,
//    4 warps per SM, strip double-buffered (198 KB): 7.1 ms per flush; 8 warps per SM, single-buffered: 5.1 ms; against
//    3.1 ms for this kernel.  With ~200 KB of shared memory the L1 shrinks to ~30 KB, the V and Z fragments (196 KB per
//    walker, read once per strip) come from L2 every time, and 4-8 warps per SM cannot hide that latency next to the
//    DMMAs; 16-row strips need 48 KB per warp, which leaves room for neither a second buffer nor a fifth warp.  The
//    variant was removed again;
//  - storing the inverses in fp32 (mixed precision, half the strip bytes) leaves the time of this kernel unchanged, a fourth
//    CTA per SM at 128 registers spills 472 bytes, ns as a compile-time constant changes nothing: the kernel is bound by
//    the latency of its fragment loads at 12 warps per SM (65 % of its stall samples are the first DMMA of a fragment set
//    waiting for that set), not by DRAM bandwidth and not by instruction issue.
// ---- strip kernel: fragments straight from global memory, software-pipelined in registers -------
// (A shared-memory cp.async ring for the operands was measured slower on B200 in round 1: 2.54 ms vs 2.07 ms per
// flush at cfg 5 / W = 2048 -- the LDS + LDGSTS instruction stream saturates the MIO queue next to
// the DMMAs.)

// Fragment set of one 16-column chunk of GEMM 1: the B0 strip (two 8-row blocks) and KB window blocks of V.
template <int KB>
struct Frag1 {
  double a0[4], a1[4], v[KB][4];
};
template <int KB, typename TB>
__device__ __forceinline__ void load_frag1(Frag1<KB>& f, const TB* a0p, const TB* a1p, const double* vp,
                                           int s, int ns, int m, int mb, int g)
{
  ld_b4(a0p + s, f.a0);
  ld_b4(a1p + s, f.a1);
#pragma unroll
  for (int b = 0; b < KB; ++b) {
    f.v[b][0] = f.v[b][1] = f.v[b][2] = f.v[b][3] = 0.0;
    if (b < mb && 8 * b + g < m) ld32(vp + (size_t)(8 * b) * ns + s, f.v[b]);
  }
}
template <int KB>
__device__ __forceinline__ void mma_frag1(double (&acc)[2][KB][2], const Frag1<KB>& f, int mb)
{
  // k-step outermost: 2 KB independent accumulator chains between dependent DMMAs
#pragma unroll
  for (int q = 0; q < 4; ++q)
#pragma unroll
    for (int b = 0; b < KB; ++b)
      if (b < mb) {
        dmma884(acc[0][b], f.a0[q], f.v[b][q]);
        dmma884(acc[1][b], f.a1[q], f.v[b][q]);
      }
}

// Fragment set of one 16-column chunk of GEMM 2: the B0 strip chunk (accumulator init) and Z rows.
template <int KB>
struct Frag2 {
  double x0[4], x1[4];
  double2 z[KB][2];
};
template <int KB, typename TB>
__device__ __forceinline__ void load_frag2(Frag2<KB>& f, const TB* a0p, const TB* a1p, const double* zp,
                                           int j0, int ns, int m, int mb, int t)
{
  ld_b4(a0p + j0, f.x0);
  ld_b4(a1p + j0, f.x1);
#pragma unroll
  for (int b = 0; b < KB; ++b)
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      f.z[b][q] = make_double2(0.0, 0.0);
      if (b < mb && 8 * b + 2 * t + q < m) f.z[b][q] = *reinterpret_cast<const double2*>(zp + (size_t)(8 * b + q) * ns + j0);
    }
}
template <int KB, typename TB>
__device__ __forceinline__ void mma_store_frag2(const Frag2<KB>& f, const double (&nw)[2][KB][2], int mb, TB* o0,
                                                TB* o1)
{
  // even / odd columns of the chunk are separate tiles (a lane ends up with 4 consecutive columns);
  // two accumulator sets (even / odd window blocks) give 8 independent DMMA chains, summed at the end
  double de0[2] = {f.x0[0], f.x0[2]}, do0[2] = {f.x0[1], f.x0[3]};
  double de1[2] = {f.x1[0], f.x1[2]}, do1[2] = {f.x1[1], f.x1[3]};
  double ee0[2] = {0.0, 0.0}, eo0[2] = {0.0, 0.0}, ee1[2] = {0.0, 0.0}, eo1[2] = {0.0, 0.0};
#pragma unroll
  for (int q = 0; q < 2; ++q)
#pragma unroll
    for (int b = 0; b < KB; ++b)
      if (b < mb) {
        if (b & 1) {
          dmma884(ee0, nw[0][b][q], f.z[b][q].x);
          dmma884(eo0, nw[0][b][q], f.z[b][q].y);
          dmma884(ee1, nw[1][b][q], f.z[b][q].x);
          dmma884(eo1, nw[1][b][q], f.z[b][q].y);
        } else {
          dmma884(de0, nw[0][b][q], f.z[b][q].x);
          dmma884(do0, nw[0][b][q], f.z[b][q].y);
          dmma884(de1, nw[1][b][q], f.z[b][q].x);
          dmma884(do1, nw[1][b][q], f.z[b][q].y);
        }
      }
  st_b4(o0, de0[0] + ee0[0], do0[0] + eo0[0], de0[1] + ee0[1], do0[1] + eo0[1]);
  st_b4(o1, de1[0] + ee1[0], do1[0] + eo1[0], de1[1] + ee1[1], do1[1] + eo1[1]);
}

// Flush, step 1 for the window kernel's eager-block form (window.cuh, R5): the accepted moves
// left V[l] = phi_l and Cp[l] = c_l = b_l / rho_l; with N[j][l] = c_j . phi_l (j < l, strictly upper
// triangular) the Sherman-Morrison chain B_m = B0 - sum_l w_l c_l^T, w_l = B_l phi_l - e_l, telescopes to
// B_m = B0 - (B0 V^T - E) Z with (I + N) Z = Cp.  One CTA per walker, three steps, all on the FP64 tensor pipe but
// the tiny middle one:
//   1. N by DMMA tiles (operand fragments straight from the rows of Cp and V, as in the strip kernel);
//   2. T = (I + N)^-1, unit upper triangular, by back substitution on the identity: one warp, lane = column, the
//      column in registers (496 fused multiply-adds per lane);
//   3. Z = T Cp by DMMA tiles in the strip kernel's GEMM-2 fragment scheme (T from shared memory as the A operand,
//      rows of Cp as the B operand, four consecutive columns of Z per lane and store).
// (Round 1 solved (I + N) Z = Cp by back substitution with one column of Z per thread: 32 dependent values in
// registers next to the DMMA code spilled 440 bytes per thread under the 128-register cap.)
// m^2 n + 2 m^2 n flop per walker.  grid = W; dynamic smem: (1 + FINTRI_NT / 32) KDP (KDP + 1) doubles.
#ifndef QMC_FINTRI_MIN_CTAS
#define QMC_FINTRI_MIN_CTAS 3
#endif
constexpr int FINTRI_NT = 128;
template <int KDP>
__global__ void __launch_bounds__(FINTRI_NT, QMC_FINTRI_MIN_CTAS) flush_finalize_tri_kernel(CrowdDev d, int l0)
{
  // l0 > 0: the window is flushed in sections of KDP accepted moves (section = moves l0 .. l0 + KDP - 1), each section a
  // complete flush of its own applied to the result of the previous one (see launch_flush_kdp)
  static_assert(KDP % 16 == 0 || KDP == 8, "two 8-row blocks per output strip");
  constexpr int KB = KDP / 8, SS = KDP + 1;
  extern __shared__ double s_n[];
  double* s_t = s_n + KDP * SS;
  const int w = blockIdx.x + d.w0;
  const int m = min(d.mwin[w] - l0, KDP);
  if (m <= 0) return;
  const int ns = d.ns, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, t = lane & 3;
  const double* Cp = d.Cp + ((size_t)w * d.kdp + l0) * ns;
  const double* V = d.V + ((size_t)w * d.kdp + l0) * ns;
  double* Z = d.C + ((size_t)w * d.kdp + l0) * ns;
  // ---- 1. N[j][l] = Cp[j] . V[l] for j < l < m.  The contraction (over the ns columns) is split over the warps: a warp
  // takes every fourth 16-column chunk and all (jb <= lb) tiles, so that each warp's chain of fragment loads is ns / 64
  // chunks long instead of ns / 16, and the warps' work is equal (by rows of tiles, warp 0 had four tiles and warp 3
  // one); the partial tiles meet in shared memory and are summed in a fixed order.
  constexpr int NWF = FINTRI_NT / 32;
  double* s_p = s_t + KDP * SS;   // [NWF - 1][KDP][SS] partial tiles of warps 1.. (warp 0 writes s_n)
  for (int e = tid; e < KDP * SS; e += FINTRI_NT) s_n[e] = 0.0;
  for (int e = tid; e < KDP * SS * (NWF - 1); e += FINTRI_NT) s_p[e] = 0.0;
  __syncthreads();
  {
    const int mbn = (m + 7) >> 3;
    double acc[KB][KB][2];
#pragma unroll
    for (int jb = 0; jb < KB; ++jb)
#pragma unroll
      for (int lb = 0; lb < KB; ++lb) acc[jb][lb][0] = acc[jb][lb][1] = 0.0;
    const double* ap = Cp + (size_t)g * ns + 4 * t;
    const double* vp = V + (size_t)g * ns + 4 * t;
#pragma unroll 2   // two chunks of fragment loads in flight
    for (int s = 16 * warp; s < ns; s += 16 * NWF) {
      double a[KB][4], b[KB][4];
#pragma unroll
      for (int jb = 0; jb < KB; ++jb) {
        a[jb][0] = a[jb][1] = a[jb][2] = a[jb][3] = 0.0;
        b[jb][0] = b[jb][1] = b[jb][2] = b[jb][3] = 0.0;
        if (jb < mbn && 8 * jb + g < m) {
          ld32(ap + (size_t)(8 * jb) * ns + s, a[jb]);
          ld32(vp + (size_t)(8 * jb) * ns + s, b[jb]);
        }
      }
#pragma unroll
      for (int q = 0; q < 4; ++q)
#pragma unroll
        for (int jb = 0; jb < KB; ++jb)
#pragma unroll
          for (int lb = jb; lb < KB; ++lb)
            if (lb < mbn) dmma884(acc[jb][lb], a[jb][q], b[lb][q]);
    }
    double* dst = warp == 0 ? s_n : s_p + (size_t)(warp - 1) * KDP * SS;
#pragma unroll
    for (int jb = 0; jb < KB; ++jb)
#pragma unroll
      for (int lb = jb; lb < KB; ++lb)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int j = 8 * jb + g, l = 8 * lb + 2 * t + e;
          if (j < l && l < m) dst[j * SS + l] = acc[jb][lb][e];
        }
  }
  __syncthreads();
  for (int e = tid; e < KDP * SS; e += FINTRI_NT) {
    double sum = s_n[e];
#pragma unroll
    for (int q = 0; q < NWF - 1; ++q) sum += s_p[(size_t)q * KDP * SS + e];
    s_n[e] = sum;
  }
  __syncthreads();
  // ---- 2. T = (I + N)^-1: column c solves (I + N) x = e_c from the bottom up; x[l] = 0 below the diagonal
  if (warp == 0 && lane < KDP) {
    const int c = lane;
    double x[KDP];
#pragma unroll
    for (int l = KDP - 1; l >= 0; --l) {
      double a = 0.0;
#pragma unroll
      for (int j = l + 1; j < KDP; ++j) a = fma(-s_n[l * SS + j], x[j], a);
      x[l] = l < c ? a : (l == c ? 1.0 : 0.0);
    }
#pragma unroll
    for (int l = 0; l < KDP; ++l) s_t[l * SS + c] = x[l];
  }
  __syncthreads();
  // ---- 3. Z = T Cp: a warp takes the 16-row strips of Z and 16-column chunks in turn; the Cp fragments of its next item
  // are loaded before the tiles of the current one are multiplied
  constexpr int NSTRIP = KDP >= 16 ? KDP / 16 : 1, RB = KDP >= 16 ? 2 : 1;
  const int mb = (m + 7) >> 3;
  const int n_items = NSTRIP * (ns / 16);
  auto load_z = [&](int item, double2 (&z)[KB][2]) {
    const int j0 = (item / NSTRIP) * 16;
#pragma unroll
    for (int b2 = 0; b2 < KB; ++b2)
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        z[b2][q] = make_double2(0.0, 0.0);
        if (b2 < mb && 8 * b2 + 2 * t + q < m) z[b2][q] = *reinterpret_cast<const double2*>(Cp + (size_t)(8 * b2 + 2 * t + q) * ns + j0 + 2 * g);
      }
  };
  Frag2<KB> f;
  f.x0[0] = f.x0[1] = f.x0[2] = f.x0[3] = 0.0;
  f.x1[0] = f.x1[1] = f.x1[2] = f.x1[3] = 0.0;
  double2 znext[KB][2];
  if (warp < n_items) load_z(warp, znext);
  for (int item = warp; item < n_items; item += NWF) {
    const int strip = item % NSTRIP, j0 = (item / NSTRIP) * 16;
#pragma unroll
    for (int b2 = 0; b2 < KB; ++b2)
#pragma unroll
      for (int q = 0; q < 2; ++q) f.z[b2][q] = znext[b2][q];
    if (item + NWF < n_items) load_z(item + NWF, znext);
    if (16 * strip >= m) continue;
    // T as the A operand of the strip kernel's GEMM 2: rows 16 strip + 8 i + g, contraction index 8 b + 2 t + e
    double nw[2][KB][2];
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
      for (int b2 = 0; b2 < KB; ++b2)
#pragma unroll
        for (int e = 0; e < 2; ++e)
          nw[i][b2][e] = s_t[(16 * strip + 8 * (i % RB) + g) * SS + 8 * b2 + 2 * t + e];
    double* o0 = Z + (size_t)(16 * strip + g) * ns + 4 * t + j0;
    // KDP = 8 has one row block: the second one repeats it (same values to the same addresses)
    mma_store_frag2<KB>(f, nw, mb, o0, RB == 2 ? o0 + (size_t)8 * ns : o0);
  }
}

// Flush, step 2: B_strip <- B0_strip - (B0_strip V^T - E) Z.  KB = kdp / 8. grid = (ceil(ns / 64), W).
// L0: first move of the section this launch applies (-1: the whole window; a compile-time constant, so the common
// case keeps the register allocation it was tuned with)
// TB: storage type of the carried inverse (double; float = mixed precision, D:R6: fragments widened on load, the
// updated strip rounded to fp32 once on store -- 8 n^2 bytes per walker-flush instead of 16 n^2)
template <int KB, int L0 = -1, typename TB = double>
__global__ void __launch_bounds__(FLUSH_NT, QMC_FLUSH_MIN_CTAS) flush_kernel(CrowdDev d, int spin)
{
  constexpr int l0 = L0 < 0 ? 0 : L0;
  const int w = blockIdx.y + d.w0;
  // L0 < 0: the whole window; L0 >= 0: its section l0 .. l0 + 8 KB - 1
  int m = d.mwin[w];
  if constexpr (L0 < 0) {
    if (m == 0) return;
  } else {
    m = min(m - l0, 8 * KB);
    if (m <= 0) return;
  }
  const int ns = d.ns, kdp = d.kdp;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const int row0 = (blockIdx.x * (FLUSH_NT / 32) + warp) * FLUSH_ROWS_PER_WARP;
  if (row0 >= ns) return;
  TB* B = carried_inverse<TB>(d) + ((size_t)w * 2 + spin) * ns * ns;
  const int* rows = d.rows + (size_t)w * kdp + l0;
  const int mb = (m + 7) >> 3;  // 8-wide blocks of the window that hold accepted moves
  TB* a0p = B + (size_t)(row0 + g) * ns + 4 * t;
  TB* a1p = a0p + (size_t)8 * ns;
  // lane's V fragment base: row g of each window block, columns 4t..4t+3 of the chunk
  const double* vp = d.V + (size_t)w * kdp * ns + (size_t)(g + l0) * ns + 4 * t;
  // lane's Z fragment base: rows 2t (+q) of each window block, columns 2g, 2g+1 of the chunk
  const double* zp = d.C + (size_t)w * kdp * ns + (size_t)(2 * t + l0) * ns + 2 * g;

  // GEMM 1: Wm = B0_strip V^T. acc[i][b] = tile (rows row0+8i.., window columns 8b..8b+7);
  // lane holds (row g, columns 8b+2t, 8b+2t+1).
  double acc[2][KB][2];
#pragma unroll
  for (int i = 0; i < 2; ++i)
#pragma unroll
    for (int b = 0; b < KB; ++b) acc[i][b][0] = acc[i][b][1] = 0.0;
  if (KB > 4) {
    // eight window blocks: one fragment set at a time (two would spill next to the 64 accumulator registers)
    Frag1<KB> fa;
    for (int s = 0; s < ns; s += 16) {
      load_frag1<KB>(fa, a0p, a1p, vp, s, ns, m, mb, g);
      mma_frag1<KB>(acc, fa, mb);
    }
  } else {
    Frag1<KB> fa, fb;
    load_frag1<KB>(fa, a0p, a1p, vp, 0, ns, m, mb, g);
    for (int s = 0; s < ns; s += 32) {
      if (s + 16 < ns) load_frag1<KB>(fb, a0p, a1p, vp, s + 16, ns, m, mb, g);
      mma_frag1<KB>(acc, fa, mb);
      if (s + 16 < ns) {
        if (s + 32 < ns) load_frag1<KB>(fa, a0p, a1p, vp, s + 32, ns, m, mb, g);
        mma_frag1<KB>(acc, fb, mb);
      }
    }
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
  // GEMM 2: B_strip = B0_strip + nw Z, 16 columns at a time
  if (KB > 4) {
    Frag2<KB> fa;
    for (int j0 = ns - 16; j0 >= 0; j0 -= 16) {
      load_frag2<KB>(fa, a0p, a1p, zp, j0, ns, m, mb, t);
      mma_store_frag2<KB>(fa, acc, mb, a0p + j0, a1p + j0);
    }
  } else {
    // chunks in reverse order: the strip lines GEMM 1 read last are the most likely to still be in L2
    Frag2<KB> fa, fb;
    load_frag2<KB>(fa, a0p, a1p, zp, ns - 16, ns, m, mb, t);
    for (int j0 = ns - 16; j0 >= 0; j0 -= 32) {
      if (j0 >= 16) load_frag2<KB>(fb, a0p, a1p, zp, j0 - 16, ns, m, mb, t);
      mma_store_frag2<KB>(fa, acc, mb, a0p + j0, a1p + j0);
      if (j0 >= 16) {
        if (j0 >= 32) load_frag2<KB>(fa, a0p, a1p, zp, j0 - 32, ns, m, mb, t);
        mma_store_frag2<KB>(fb, acc, mb, a0p + j0 - 16, a1p + j0 - 16);
      }
    }
  }
}

// ---- 32-row strips: four 8-row blocks per warp, so every V / Z fragment set feeds twice the DMMAs of the 16-row kernel
// above (64 per set at KB = 4), fragment sets double-buffered in registers (254 registers, two CTAs of four warps per
// SM).  Measured at cfg 5, W = 4096, k = 32 (B200, round 2): 2.96 ms per launch against 3.13 ms, DMMA pipe 70 % busy
// against 67 % (GEMM 2 sums the window blocks in one chain per tile instead of two: rounding-level differences).  The larger strips in flight
// (98 KB per warp, 116 MB over the GPU) miss L2 more often on their second read: 13.2 GB of DRAM traffic against 12.2 GB
// for 9.66 GB algorithmic -- the kernel is bound by the latency of its fragment loads next to the DMMAs, not by DRAM
// bandwidth, so the trade pays.  Single-buffered at 168 registers (three CTAs per SM, 124 B spill) it ran at 3.6 ms,
// single-buffered at 198 registers (two CTAs) at 4.1 ms; CTAs of one or two warps at the same occupancy: no change;
// prefetch.global.L2 of the strip 4 or 8 chunks ahead of the fragment loads (both GEMMs): 3.45 ms against 3.31 ms per
// flush; the first 3 or 6 chunks of every strip (the ones least likely to survive in L2 until GEMM 2 comes back to them)
// kept in otherwise unused shared memory between the two GEMMs, conflict-free 16-byte pieces: 3.70 ms against 3.37 ms
// (shared-memory traffic next to the DMMAs costs more than the DRAM re-reads it saves, as with round 1's operand ring).
// With 4 KB of strip per warp in flight (8 warps per SM, ~1 us of loaded DRAM latency) the kernel moves 4.5 TB/s of mixed
// read / write traffic (0.69 of the copy rate) next to a DMMA pipe that is 68 % busy: both are near what this structure
// can feed; the overfetch of the second strip read (3.6 of its 4.8 GB miss L2) is what is left to remove.
// Used for fp64-stored inverses when ns % 32 == 0 and the window has at least two blocks (KB >= 2); the 16-row kernel
// serves the rest.
#ifndef QMC_FLUSH32_MIN_CTAS
#define QMC_FLUSH32_MIN_CTAS 2
#endif
#ifndef QMC_FLUSH32_NT
#define QMC_FLUSH32_NT 128
#endif
constexpr int FLUSH32_NT = QMC_FLUSH32_NT;
// Window move held at position p of an 8-wide MMA tile.  The accumulator layout of GEMM 1 gives a lane the tile positions
// 2 t and 2 t + 1, and GEMM 2 contracts over them in k-steps (b, q) = positions {2 t + q}: with position p holding move
// 4 (p & 1) + (p >> 1) a k-step covers the four CONSECUTIVE moves 8 b + 4 q .. + 3, so the k-steps of the window's padding
// can be left out in units of four moves instead of eight (m = 27 accepted moves of 32 on average at cfg 5).
__device__ __forceinline__ int win_pos(int p) { return 4 * (p & 1) + (p >> 1); }

template <int KB>
struct Frag1x4 {
  double a[4][4], v[KB][4];
};
template <int KB, typename TB>
__device__ __forceinline__ void load_frag1x4(Frag1x4<KB>& f, const TB* ap, const double* vp, int s, int ns, int m, int mb, int g)
{
#pragma unroll
  for (int i = 0; i < 4; ++i) ld_b4(ap + (size_t)(8 * i) * ns + s, f.a[i]);
#pragma unroll
  for (int b = 0; b < KB; ++b) {
    f.v[b][0] = f.v[b][1] = f.v[b][2] = f.v[b][3] = 0.0;
    if (b < mb && 8 * b + win_pos(g) < m) ld32(vp + (size_t)(8 * b) * ns + s, f.v[b]);
  }
}
template <int KB>
__device__ __forceinline__ void mma_frag1x4(double (&acc)[4][KB][2], const Frag1x4<KB>& f, int mb)
{
#pragma unroll
  for (int q = 0; q < 4; ++q)
#pragma unroll
    for (int b = 0; b < KB; ++b)
      if (b < mb) {
#pragma unroll
        for (int i = 0; i < 4; ++i) dmma884(acc[i][b], f.a[i][q], f.v[b][q]);
      }
}
template <int KB>
struct Frag2x4 {
  double x[4][4];
  double2 z[KB][2];
};
template <int KB, typename TB>
__device__ __forceinline__ void load_frag2x4(Frag2x4<KB>& f, const TB* ap, const double* zp, int j0, int ns, int m, int mb, int t)
{
#pragma unroll
  for (int i = 0; i < 4; ++i) ld_b4(ap + (size_t)(8 * i) * ns + j0, f.x[i]);
#pragma unroll
  for (int b = 0; b < KB; ++b)
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      f.z[b][q] = make_double2(0.0, 0.0);
      if (8 * b + 4 * q + t < m) f.z[b][q] = *reinterpret_cast<const double2*>(zp + (size_t)(8 * b + 4 * q) * ns + j0);
    }
}
template <int KB, typename TB>
__device__ __forceinline__ void mma_store_frag2x4(const Frag2x4<KB>& f, const double (&nw)[4][KB][2], int m, TB* op, int ns)
{
  double de[4][2], dd[4][2];   // even / odd columns of the chunk: eight independent DMMA chains
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    de[i][0] = f.x[i][0]; de[i][1] = f.x[i][2];
    dd[i][0] = f.x[i][1]; dd[i][1] = f.x[i][3];
  }
#pragma unroll
  for (int b = 0; b < KB; ++b)
    if (8 * b < m) {
      // k-step (b, q) = window moves 8 b + 4 q .. + 3 (win_pos): the second one is skipped when none of them was accepted
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        dmma884(de[i], nw[i][b][0], f.z[b][0].x);
        dmma884(dd[i], nw[i][b][0], f.z[b][0].y);
      }
      if (8 * b + 4 < m) {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          dmma884(de[i], nw[i][b][1], f.z[b][1].x);
          dmma884(dd[i], nw[i][b][1], f.z[b][1].y);
        }
      }
    }
#pragma unroll
  for (int i = 0; i < 4; ++i) st_b4(op + (size_t)(8 * i) * ns, de[i][0], dd[i][0], de[i][1], dd[i][1]);
}

// L0, TB: as for flush_kernel.  grid = (ceil(ns / (32 warps per CTA)), W); CTAs of four warps when the strips of a matrix fill
// them, else of one warp (n = 192: 6 strips, n = 96: 3 -- half-empty CTAs hold registers for nothing: cfg 4 42.3 -> 44.3 M,
// cfg 3 67.5 -> 70.3 M moves/s; at n = 384 one-warp CTAs are 0.25 % slower).
template <int KB, int L0 = -1, typename TB = double>
__global__ void __launch_bounds__(FLUSH32_NT, QMC_FLUSH32_MIN_CTAS) flush32_kernel(CrowdDev d, int spin)
{
  constexpr int l0 = L0 < 0 ? 0 : L0;
  const int w = blockIdx.y + d.w0;
  int m = d.mwin[w];
  if constexpr (L0 < 0) {
    if (m == 0) return;
  } else {
    m = min(m - l0, 8 * KB);
    if (m <= 0) return;
  }
  const int ns = d.ns, kdp = d.kdp;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const int row0 = (blockIdx.x * (blockDim.x >> 5) + warp) * 32;   // CTAs of FLUSH32_NT or of 32 threads (launch_strip)
  if (row0 >= ns) return;
  TB* B = carried_inverse<TB>(d) + ((size_t)w * 2 + spin) * ns * ns;
  const int* rows = d.rows + (size_t)w * kdp + l0;
  const int mb = (m + 7) >> 3;
  TB* ap = B + (size_t)(row0 + g) * ns + 4 * t;
  const double* vp = d.V + (size_t)w * kdp * ns + (size_t)(win_pos(g) + l0) * ns + 4 * t;
  const double* zp = d.C + (size_t)w * kdp * ns + (size_t)(t + l0) * ns + 2 * g;
  double acc[4][KB][2];   // acc[i][b][e]: row 8 i + g of the strip, window move 8 b + win_pos(2 t + e) = 8 b + 4 e + t
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int b = 0; b < KB; ++b) acc[i][b][0] = acc[i][b][1] = 0.0;
  {
    Frag1x4<KB> fa, fb;
    load_frag1x4<KB>(fa, ap, vp, 0, ns, m, mb, g);
    for (int s = 0; s < ns; s += 32) {
      if (s + 16 < ns) load_frag1x4<KB>(fb, ap, vp, s + 16, ns, m, mb, g);
      mma_frag1x4<KB>(acc, fa, mb);
      if (s + 16 < ns) {
        if (s + 32 < ns) load_frag1x4<KB>(fa, ap, vp, s + 32, ns, m, mb, g);
        mma_frag1x4<KB>(acc, fb, mb);
      }
    }
  }
#pragma unroll
  for (int b = 0; b < KB; ++b) {
    if (b < mb) {
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int l = 8 * b + 4 * e + t;
        const int rl = (l < m) ? rows[l] : -1;
#pragma unroll
        for (int i = 0; i < 4; ++i) acc[i][b][e] = (rl == row0 + 8 * i + g ? 1.0 : 0.0) - acc[i][b][e];
      }
    }
  }
  {
    // chunks in reverse order: the strip lines GEMM 1 read last are the most likely to still be in L2
    Frag2x4<KB> fa, fb;
    load_frag2x4<KB>(fa, ap, zp, ns - 16, ns, m, mb, t);
    for (int j0 = ns - 16; j0 >= 0; j0 -= 32) {
      if (j0 >= 16) load_frag2x4<KB>(fb, ap, zp, j0 - 16, ns, m, mb, t);
      mma_store_frag2x4<KB>(fa, acc, m, ap + j0, ns);
      if (j0 >= 16) {
        if (j0 >= 32) load_frag2x4<KB>(fa, ap, zp, j0 - 32, ns, m, mb, t);
        mma_store_frag2x4<KB>(fb, acc, m, ap + j0 - 16, ns);
      }
    }
  }
}

}  // namespace qmc
