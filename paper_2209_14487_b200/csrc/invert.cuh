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
  int* rsrc = reinterpret_cast<int*>(colf);         // [ns] row sources of the current panel's trailing update
  __shared__ int s_bad;
  double* X = d.Binv + (size_t)blockIdx.x * ns * ns;
  if (tid == 0) s_bad = 0;
  __syncthreads();
#ifdef QMC_INV_CLOCKS
  long long ph_t[8] = {0, 0, 0, 0, 0, 0, 0, 0}, ph_c = clock64();
#define IPH(x) do { if (tid == 0) { const long long c_ = clock64(); ph_t[x] += c_ - ph_c; ph_c = c_; } } while (0)
#else
#define IPH(x) do {} while (0)
#endif
  for (int c0 = 0; c0 < n; c0 += INVB_NB) {
    const int nb = min(INVB_NB, n - c0);
    // (a) panel into shared memory (zero padded), eliminated there in place
#pragma unroll 8   // eight independent loads in flight per thread (the panel load is a latency chain otherwise)
    for (int e = tid; e < ns * INVB_NB; e += INVB2_NT) {
      const int r = e / INVB_NB, j = e - r * INVB_NB;
      XG[r * INVB2_XS + j] = (r < n && j < nb) ? X[(size_t)r * ns + c0 + j] : 0.0;
    }
    __syncthreads();
    IPH(0);
    // The panel itself is eliminated in sub-panels of INVB_SB columns, the same right-looking scheme one level down:
    // a pivot step touches n x SB elements (a warp takes sixteen rows at a time, lane = (row group, column pair), the
    // multiplier of a row is a shuffle, the row interchange is done on register copies of rows c and p, the search
    // for the next pivot rides on the update), and after each sub-panel the other 32 - SB panel columns get its row
    // swaps and one rank-SB update.  (Eliminating all 32 columns at every pivot step cost 67 of the kernel's 139 ms at
    // cfg 5, W = 4096.)
    constexpr int NW = INVB2_NT / 32, SB = INVB_SB;
    static_assert(INVB_NB == 32 && SB == 8, "lane = (row group, column pair) of an eight-column sub-panel");
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
        // lane = (row group rg, column pair cp): the lane owns columns 2 cp, 2 cp + 1 of its rows as one 16-byte piece, so
        // a row costs one shared-memory load, ONE broadcast of its multiplier and one store per lane (with one column per
        // lane it was twice that; the update loop with its loads, broadcasts and stores is nearly all of a pivot step's
        // 3.8 k cycles).  The lanes of a quarter-warp take rows r and r + 4 (row stride 34 doubles: 64 bytes apart in the
        // banks), so the 16-byte accesses are conflict-free.
        const int cp = lane & 3, rg = lane >> 2, cbase = lane - cp;
        const double2 prow = *reinterpret_cast<const double2*>(XG + p * INVB2_XS + s0 + 2 * cp);
        const double2 crow = *reinterpret_cast<const double2*>(XG + c * INVB2_XS + s0 + 2 * cp);
        const double pv = __shfl_sync(0xffffffffu, (jl & 1) ? prow.y : prow.x, cbase + (jl >> 1));
        // true divisions (see above), two per lane
        const double2 rc = make_double2(((2 * cp == jl) ? 1.0 : prow.x) / pv, ((2 * cp + 1 == jl) ? 1.0 : prow.y) / pv);
        __syncthreads();   // rows c and p are in registers everywhere; the partial maxima have been read
        double best = -1.0;
        int bi = c + 1;
        const bool next_y = (jl + 1) & 1;   // component of column jl + 1 in the lanes cp == (jl + 1) / 2
        for (int rb = warp * 16; rb < n; rb += 16 * NW) {   // warp-uniform trip count; a warp pass takes 16 consecutive rows
          const int r0 = rb + (rg >> 1) + 4 * (rg & 1);
          double2 v[2];
#pragma unroll
          for (int i = 0; i < 2; ++i) {
            const int r = r0 + 8 * i;
            v[i] = (r < n) ? *reinterpret_cast<const double2*>(XG + r * INVB2_XS + s0 + 2 * cp) : make_double2(0.0, 0.0);
            if (r == p) v[i] = crow;   // row p receives the old row c
          }
#pragma unroll
          for (int i = 0; i < 2; ++i) {
            const int r = r0 + 8 * i;
            const double cf = __shfl_sync(0xffffffffu, (jl & 1) ? v[i].y : v[i].x, cbase + (jl >> 1));
            double2 nv = make_double2(fma(-cf, rc.x, (2 * cp == jl) ? 0.0 : v[i].x), fma(-cf, rc.y, (2 * cp + 1 == jl) ? 0.0 : v[i].y));
            if (r == c) nv = rc;
            if (r < n) *reinterpret_cast<double2*>(XG + r * INVB2_XS + s0 + 2 * cp) = nv;
            double a = fabs(next_y ? nv.y : nv.x);
            a = (a == a) ? a : INFINITY;
            const bool take = r > c && r < n && (a > best || (a == best && r < bi));
            best = take ? a : best;
            bi = take ? r : bi;
          }
        }
        if (jl + 1 < sb) {   // column jl + 1 lives in the lanes cp == (jl + 1) / 2 of the eight row groups
          double bj = best;
          int ij = bi;
#pragma unroll
          for (int o = 4; o < 32; o <<= 1) {
            const double ov = __shfl_xor_sync(0xffffffffu, bj, o);
            const int oi = __shfl_xor_sync(0xffffffffu, ij, o);
            if (ov > bj || (ov == bj && oi < ij)) { bj = ov; ij = oi; }
          }
          if (lane == ((jl + 1) >> 1)) { redv[warp] = bj; redi[warp] = ij; }
        }
      }
      if (bad) break;
      __syncthreads();   // the sub-panel holds its Gauss-Jordan operator; piv[] of its columns is visible
      IPH(1);
      if (nb > sb) {
        // the sub-panel's row swaps on the other panel columns (a thread owns a column: no barrier), then its pivot
        // rows, then the rank-sb update X[:, o] <- X[:, o] + (G - E_K) A_K[:, o]  (rows of K: G[K, :] A_K[:, o]) ...
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
        // ... as one FP64 tensor-core GEMM per 16-row tile (k = SB: two MMA k-steps).  Column nn of MMA tile b is panel
        // column f = ((nn >> 1) & 1) + 16 (nn >> 2) + 4 b + 2 (nn & 1): a lane's accumulator pair (nn = 2 t, 2 t + 1) then
        // sits at 34 g + (t & 1) + 16 (t >> 1) + const, which tiles the 16 double-banks exactly twice per access (the
        // shuffle form -- one load, eight shuffles, one store per row -- kept the L1 data pipe three times as busy).
        const int g = lane >> 2, t = lane & 3;
        const int fc = (t & 1) + 16 * (t >> 1);                                   // + 4 b + 2 e
        double bk[2][4];
#pragma unroll
        for (int q2 = 0; q2 < 2; ++q2)
#pragma unroll
          for (int b2 = 0; b2 < 4; ++b2) {
            const int k = 4 * q2 + t, col = ((g >> 1) & 1) + 16 * (g >> 2) + 4 * b2 + 2 * (g & 1);
            bk[q2][b2] = (k < sb && (col < s0 || col >= s0 + sb)) ? AKs[k * INVB_NB + col] : 0.0;
          }
        for (int rt = warp; rt < (n + 15) / 16; rt += NW) {
          double acc[2][4][2];
          double* xr[2];
#pragma unroll
          for (int i = 0; i < 2; ++i) {
            const int r = rt * 16 + 8 * i + g;
            const bool in_k = r >= c0 + s0 && r < c0 + s0 + sb;
            xr[i] = XG + r * INVB2_XS;
#pragma unroll
            for (int b2 = 0; b2 < 4; ++b2)
#pragma unroll
              for (int e = 0; e < 2; ++e) acc[i][b2][e] = in_k ? 0.0 : xr[i][fc + 4 * b2 + 2 * e];
          }
#pragma unroll
          for (int q2 = 0; q2 < 2; ++q2) {
            const double a0 = xr[0][s0 + 4 * q2 + t], a1 = xr[1][s0 + 4 * q2 + t];
#pragma unroll
            for (int b2 = 0; b2 < 4; ++b2) {
              dmma884(acc[0][b2], a0, bk[q2][b2]);
              dmma884(acc[1][b2], a1, bk[q2][b2]);
            }
          }
#pragma unroll
          for (int i = 0; i < 2; ++i)
#pragma unroll
            for (int b2 = 0; b2 < 4; ++b2)
#pragma unroll
              for (int e = 0; e < 2; ++e) {
                const int col = fc + 4 * b2 + 2 * e;
                if (col < s0 || col >= s0 + sb) xr[i][col] = acc[i][b2][e];
              }
        }
        __syncthreads();
      }
      IPH(2);
    }
    if (bad && tid == 0) s_bad = 1;
    // (b) the panel's row swaps on the columns outside the panel are not carried out as swaps: rsrc[r] = the row whose
    // content they move to position r, and the trailing update below reads row rsrc[r] where it writes row r.  Every
    // swap pairs a row of K with a pivot row, so a pivot row's position only ever receives old rows of K; a warp owns
    // its 16 columns, reads the (permuted) rows of K first and writes them last: no row is read after it was written.
    // (As a pass of its own -- 32 dependent load/store pairs per column -- the swaps were 14 % of the kernel; issued
    // from the pivot steps they stalled the pivot chain on their loads.)
    for (int r = tid; r < ns; r += INVB2_NT) rsrc[r] = r;
    __syncthreads();
    if (tid == 0 && !s_bad)
      for (int j = 0; j < nb; ++j) {
        const int c = c0 + j, pp = piv[c], x = rsrc[c];
        rsrc[c] = rsrc[pp];
        rsrc[pp] = x;
      }
    __syncthreads();
    if (s_bad) break;
    IPH(3);
    // (d) trailing update by 16-column blocks: A[:, o] <- A[:, o] + (X_G - E_K) A_K[:, o], rows of K last.
    // The column index of an MMA result may be permuted freely if the B operand uses the same permutation: column nn of
    // tile b is column 4 (nn / 2) + 2 b + (nn % 2) of the block, so a lane's two tiles are four consecutive columns -- one
    // 32-byte load and one 32-byte store per row, four lanes covering one 128-byte line (8-byte stores and 16-byte loads
    // of half lines made the L1 data pipe the busiest unit of this kernel: ncu r2).
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
            const int j = 4 * q + t, o = o0 + 4 * (g >> 1) + 2 * b + (g & 1);
            bb[q][b] = (j < nb && o < n) ? X[(size_t)rsrc[c0 + j] * ns + o] : 0.0;
          }
        // row tiles in order with the tile of K skipped, then the tile of K (its rows of X are not read: acc = 0); the
        // loads of the next tile are issued before the current tile's 64 MMAs, so a warp overlaps its own memory latency
        auto tile_r0 = [&](int rt) { return rt == nrt ? c0 : rt * 32; };
        auto tile_load = [&](int rt, double (&x)[4][4]) {
          const int r0 = tile_r0(rt);
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const int r = r0 + 8 * i + g;
            x[i][0] = x[i][1] = x[i][2] = x[i][3] = 0.0;
            if (rt < nrt && r < n) ld32(X + (size_t)rsrc[r] * ns + o0 + 4 * t, x[i]);
          }
        };
        const int rt_first = c0 == 0 ? 1 : 0;
        double xn[4][4];
        tile_load(rt_first, xn);
        for (int rt = rt_first; rt <= nrt; ++rt) {
          if (rt < nrt && rt * 32 == c0) continue;
          const int r0 = tile_r0(rt);
          double acc[4][2][2];
#pragma unroll
          for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int b = 0; b < 2; ++b) {
              acc[i][b][0] = xn[i][2 * b];
              acc[i][b][1] = xn[i][2 * b + 1];
            }
          int rn = rt + 1;
          if (rn < nrt && rn * 32 == c0) ++rn;
          if (rn <= nrt) tile_load(rn, xn);
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
          for (int i = 0; i < 4; ++i) {
            const int r = r0 + 8 * i + g;   // (padding columns o >= n receive the zeros they already hold)
            if (r < n) st32(X + (size_t)r * ns + o0 + 4 * t, acc[i][0][0], acc[i][0][1], acc[i][1][0], acc[i][1][1]);
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
    IPH(4);
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
#ifdef QMC_INV_CLOCKS
  __syncthreads();
  IPH(5);
  if (tid == 0)
    for (int q = 0; q < 8; ++q) d.pvec[(size_t)blockIdx.x * 8 + q] = (double)ph_t[q];
#endif
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
