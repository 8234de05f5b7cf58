// window.cuh -- qmc_sweep with a delayed update: one launch per delay window, one CTA per walker.
//
// The crowd advances in lock-step per *window* (D:C6 schedule): a CTA owns one walker for the
// cnt <= delay_rank consecutive moves k0 .. k0+cnt-1 (row/proposal, spline, ratio, decision, update
// for each), then the whole crowd flushes (update.cuh).  Walkers never interact inside a window, so
// no kernel boundary is needed between moves: an SM overlaps the DRAM-bound spline gather of one
// walker with the fp64 work of its other resident walkers, the per-walker state (positions, inverse
// row, orbitals at r') lives in shared memory for the whole window, and the launch tail is paid once
// per window instead of twice per move.
//
// Inside the window the kernel uses the *eager-block* form of the delayed update (R5).
// Because the electrons of a window are consecutive, the only inverse rows the window itself needs
// are the cnt rows `blk` = B0[k0 .. k0+cnt); every accepted move l (row k_l, orbitals phi_l, ratio
// rho_l, current row b_l) applies its Sherman-Morrison update (D:C5) to the rows of that block that
// are still to be proposed,
//     Bcur[i'] <- Bcur[i'] - (Bcur[i'] . phi_l) c_l,     c_l = b_l / rho_l,      i' after the move,
// so that the row of the next move is simply Bcur[i] -- no S^-1, no p/q vectors, no axpy over the
// window -- and one pass over (on average) half the block per accepted move is all the window traffic.
// The other n - cnt rows get the same updates at the flush: with V[l] = phi_l, Cp[l] = c_l and the
// strictly upper triangular N[j][l] = c_j . phi_l (j < l),
//     B <- B0 - (B0 V^T - E) Z,      (I + N) Z = Cp,
// which is C6's B0 - (B0 V^T - E) S^-T C with the bordered inverse replaced by its unit-triangular
// factor (flush_finalize_tri_kernel); the two-GEMM strip kernel is the same for both paths.
#pragma once
#include "move.cuh"
#include "update.cuh"

namespace qmc {


// Shared-memory layout of the window kernel, offsets in doubles.
struct WinLayout {
  int R, b, bn, red, mv, gauss, pairk, rows, cbuf, vgl, total;
};
__host__ __device__ inline WinLayout win_layout(int N, int ns, int kdp, int elem, int nt = MOVE_NT)
{
  WinLayout L;
  int o = 0;
  L.R = o; o += 3 * N;       // positions of the walker
  L.b = o; o += ns;          // inverse row of the current move (then c_l = b / rho_D)
  L.bn = o; o += ns;         // inverse row of the next move
  L.red = o; o += (8 * (nt / 32) < 32 ? 32 : 8 * (nt / 32));
  L.mv = o; o += MOVE_MV;
  L.gauss = o; o += 8;       // Box-Muller pieces of the next move
  L.pairk = o; o += 8;       // the pair term (k+1, k) against r_k and against r'_k (window kernel)
  L.rows = o; o += kdp / 2;  // int[kdp]: electron (within the spin block) of accepted move l
  o = (o + 1) & ~1;
#ifdef QMC_WIN_CBUF1
  L.cbuf = o; o += ((3 * ns * elem + 15) / 16) * 2;      // gradient cache of the coming move: T[3][ns]
#else
  L.cbuf = o; o += 2 * ((3 * ns * elem + 15) / 16) * 2;  // gradient cache of this / the next move: 2 x T[3][ns]
#endif
  L.vgl = o; o += (5 * ns * elem + 7) / 8;               // orbitals at r': T[5][ns]
  L.total = o;
  return L;
}

__device__ __forceinline__ double2 ld_x2(const float* v, int jj)
{
  const float2 f = reinterpret_cast<const float2*>(v)[jj];
  return make_double2((double)f.x, (double)f.y);
}
__device__ __forceinline__ double2 ld_x2(const double* v, int jj) { return reinterpret_cast<const double2*>(v)[jj]; }

// nbytes % 16 == 0, both 16-byte aligned; strided over the CTA
template <int NT = MOVE_NT>
__device__ __forceinline__ void cp_async_cta(void* smem, const void* gmem, int nbytes)
{
  for (int o = threadIdx.x * 16; o < nbytes; o += NT * 16)
    cp_async16(static_cast<char*>(smem) + o, static_cast<const char*>(gmem) + o);
}

// ---- the Jastrow sums of a move, taken off the walker's critical path ---------------------------------------------
// A move needs two pair sums (D:C3): at the current position r_k for G_k(R) (proposal) and at r' for the ratio.  Both
// are ~70 dependent fp64 instructions per pair, six pairs per thread: next to the row dots they were 2 x 3000 cycles
// of every move's chain.  Neither depends on what the move itself decides, except through one pair term:
//   - the sum at r' needs only r' and R: it is evaluated right after the proposal, together with the next one, as
//     straight-line code with four pair chains in flight;
//   - the sum at r_{k+1} for the NEXT move is evaluated at the same time over all electrons but k (whose position the
//     pending decision may change); the missing term is evaluated for both outcomes (against r_k and against r'_k)
//     and the one that applies is added after the decision.
struct J2Part {
  double us, g[3];
};
// One pair term, branch-free (the same products and the same order of operations as j2_pair; `on` = false contributes
// exact zeros): straight-line code lets the scheduler interleave several pairs -- a pair is a chain of ~45 dependent
// fp64 instructions, and a thread that walks its pairs one after the other issues one instruction per ~12 cycles.
__device__ __forceinline__ void j2_pair_bf(const CrowdDev& d, const double (&rk)[3], const double* ri, bool on, J2Part& s)
{
  double dd[3], r2 = 0.0;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    double x = rk[c] - ri[c];
    x -= d.box[c] * rint(x * d.inv_box[c]);
    dd[c] = x;
    r2 = fma(x, x, r2);
  }
  on = on && r2 > 1e-280;
  const double inv_r = rsqrt_pos(on ? r2 : 1.0);
  const double r = r2 * inv_r;
  const double inv_den = rcp_pos(fma(d.j2_b, r, 1.0));
  const double a = on ? d.j2_a : 0.0;
  s.us += a * r * inv_den;
  const double f = a * inv_den * inv_den * inv_r;
#pragma unroll
  for (int c = 0; c < 3; ++c) s.g[c] = fma(f, dd[c], s.g[c]);
}

// Thread-strided partials of two pair sums at once: electron k placed at rn against all electrons but k, and (if
// `next`) electron k + 1 at its own position rk1 against all electrons but k and k + 1.  Two electrons per trip, so
// four independent pair chains are in flight per thread.
template <int NT, int NS = 0>
__device__ __forceinline__ void j2_two_sums(const CrowdDev& d, const double* R, int k, const double (&rn)[3], bool next,
                                            const double (&rk1)[3], J2Part& at_rn, J2Part& at_next)
{
  at_rn.us = at_rn.g[0] = at_rn.g[1] = at_rn.g[2] = 0.0;
  at_next.us = at_next.g[0] = at_next.g[1] = at_next.g[2] = 0.0;
  const int N = sh_N<NS>(d);
  for (int i0 = threadIdx.x; i0 < N; i0 += 2 * NT) {
    const int i1 = i0 + NT;
    const bool in1 = i1 < N;
    const double* ra = R + 3 * i0;
    const double* rb = R + 3 * (in1 ? i1 : i0);
    j2_pair_bf(d, rn, ra, i0 != k, at_rn);
    j2_pair_bf(d, rk1, ra, next && i0 != k && i0 != k + 1, at_next);
    j2_pair_bf(d, rn, rb, in1 && i1 != k, at_rn);
    j2_pair_bf(d, rk1, rb, next && in1 && i1 != k && i1 != k + 1, at_next);
  }
}

// G_k(R) and the proposal from the row dots and a precomputed Jastrow partial (see dev_gold_propose for the formulas;
// same products, the pair terms summed in a different order).  extra: the pair term (k, k-1) chosen after the previous
// decision, added by thread 0 (nullptr for the first move of a window).
template <typename T, int NT, int NS = 0>
__device__ __forceinline__ void win_gold_propose(const CrowdDev& d, int k, const double* b_s, const T* cache, const double* R,
                                                 const J2Part& jp, const double* extra, MoveScal ms, double* red,
                                                 const double* gp, SplineW<T>* sw_out)
{
  const int ns = sh_ns<NS>(d), tid = threadIdx.x;
  double v[7] = {0.0, 0.0, 0.0, jp.us, jp.g[0], jp.g[1], jp.g[2]};
  for (int j = tid; j < sh_M<NS>(d); j += NT) {
    const double bj = b_s[j];
    v[0] = fma(bj, (double)cache[j], v[0]);
    v[1] = fma(bj, (double)cache[ns + j], v[1]);
    v[2] = fma(bj, (double)cache[2 * ns + j], v[2]);
  }
  if (extra && tid == 0) {
    v[3] += extra[0]; v[4] += extra[1]; v[5] += extra[2]; v[6] += extra[3];
  }
  block_sum_t0<7, NT>(v, red);
  if (tid < 3) {
    const int c = tid;
    const double g_old = c == 0 ? v[0] + v[4] : (c == 1 ? v[1] + v[5] : v[2] + v[6]);
    const double rkc = R[3 * k + c];
    const double chi = c == 0 ? gp[0] * gp[1] : (c == 1 ? gp[0] * gp[2] : gp[3] * gp[4]);
    const double xx = __dadd_rn(__dmul_rn(d.tau, g_old), __dmul_rn(d.sqrt_tau, chi));
    const double delta = (double)__double2float_rn(xx);
    const double rn = rkc + delta;
    ms.g_old[c] = g_old;
    ms.delta[c] = delta;
    ms.rn[c] = rn;
    if (c == 0) *ms.usum_old = v[3];
    spline_axis<T>(d, c, rn, *sw_out);
  }
}

// rho_D, rho_J and G_k(R') from the row dots and the precomputed Jastrow partial at r' (see dev_ratio_grad).
template <typename T, int NT, int NS = 0>
__device__ __forceinline__ void win_ratio_grad(const CrowdDev& d, const double* b, const T* vgl, const J2Part& jr,
                                               MoveScal ms, double* red)
{
  const int ns = sh_ns<NS>(d), tid = threadIdx.x;
  double v[8] = {0.0, 0.0, 0.0, 0.0, jr.us, jr.g[0], jr.g[1], jr.g[2]};
  for (int j = tid; j < sh_M<NS>(d); j += NT) {
    const double bj = b[j];
    v[0] = fma(bj, (double)vgl[j], v[0]);
    v[1] = fma(bj, (double)vgl[ns + j], v[1]);
    v[2] = fma(bj, (double)vgl[2 * ns + j], v[2]);
    v[3] = fma(bj, (double)vgl[3 * ns + j], v[3]);
  }
  block_sum_t0<8, NT>(v, red);
  if (tid == 0) {
    const double rho_d = v[0];
    *ms.rho_d = rho_d;
    *ms.rho_j = exp(v[4] - *ms.usum_old);
#pragma unroll
    for (int c = 0; c < 3; ++c) ms.g_new[c] = v[1 + c] / rho_d + v[5 + c];
  }
}

// the same by one warp (a warp that would otherwise idle at a barrier)
__device__ __forceinline__ void cp_async_warp(void* smem, const void* gmem, int nbytes)
{
  for (int o = (threadIdx.x & 31) * 16; o < nbytes; o += 32 * 16)
    cp_async16(static_cast<char*>(smem) + o, static_cast<const char*>(gmem) + o);
}

// Sherman-Morrison on the rows of the window block that are still to be proposed (D:C5 restricted to the
// block): for rows r in [r_first, cnt): t = src[r] . phi', dst[r] = src[r] - t c, with phi' = vgl_s[0..ns)
// and c = c_s (both shared memory).  A warp takes two rows at a time, keeps them in registers between the
// dot and the update (rows of up to 64 WIN_NV = 512 columns; longer rows are read twice), and also
// hands row r_first to shared memory (next_s) as the next move's inverse row.
constexpr int WIN_NV = 8;
// TS: type of the source rows (double; float when they are still the fp32-stored B0 rows of the mixed-precision mode)
__device__ __forceinline__ double2 ld_row2(const double* row, int jj) { return reinterpret_cast<const double2*>(row)[jj]; }
__device__ __forceinline__ double2 ld_row2(const float* row, int jj)
{
  const float2 f = reinterpret_cast<const float2*>(row)[jj];
  return make_double2((double)f.x, (double)f.y);
}
template <typename T, int NT, typename TS = double>
__device__ __forceinline__ void block_rows_update(const TS* src, double* dst, int ns, int r_first, int cnt,
                                                  const T* vgl_s, const double* c_s, double* next_s)
{
  constexpr int RB = 2;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nh = ns / 2;
  const double2* c2 = reinterpret_cast<const double2*>(c_s);
  if (nh <= 32 * WIN_NV) {
    for (int r0 = r_first + warp * RB; r0 < cnt; r0 += (NT / 32) * RB) {
      double2 v[RB][WIN_NV];
      double acc[RB];
#pragma unroll
      for (int r = 0; r < RB; ++r) {
        acc[r] = 0.0;
        const TS* rp = src + (size_t)(r0 + r) * ns;
#pragma unroll
        for (int q = 0; q < WIN_NV; ++q) {
          const int jj = lane + 32 * q;
          v[r][q] = (r0 + r < cnt && jj < nh) ? ld_row2(rp, jj) : make_double2(0.0, 0.0);
        }
      }
#pragma unroll
      for (int q = 0; q < WIN_NV; ++q) {
        const int jj = lane + 32 * q;
        if (jj < nh) {
          const double2 x = ld_x2(vgl_s, jj);
#pragma unroll
          for (int r = 0; r < RB; ++r) acc[r] = fma(v[r][q].x, x.x, fma(v[r][q].y, x.y, acc[r]));
        }
      }
#pragma unroll
      for (int r = 0; r < RB; ++r) acc[r] = warp_sum(acc[r]);
#pragma unroll
      for (int r = 0; r < RB; ++r) {
        if (r0 + r < cnt) {
          double2* wp = reinterpret_cast<double2*>(dst + (size_t)(r0 + r) * ns);
          double2* sp = (r0 + r == r_first) ? reinterpret_cast<double2*>(next_s) : nullptr;
#pragma unroll
          for (int q = 0; q < WIN_NV; ++q) {
            const int jj = lane + 32 * q;
            if (jj < nh) {
              const double2 c = c2[jj];
              const double2 o = make_double2(fma(-acc[r], c.x, v[r][q].x), fma(-acc[r], c.y, v[r][q].y));
              wp[jj] = o;
              if (sp) sp[jj] = o;
            }
          }
        }
      }
    }
  } else {
    for (int r = r_first + warp; r < cnt; r += NT / 32) {
      const TS* rp = src + (size_t)r * ns;
      double2* wp = reinterpret_cast<double2*>(dst + (size_t)r * ns);
      double acc = 0.0;
      for (int jj = lane; jj < nh; jj += 32) {
        const double2 x = ld_x2(vgl_s, jj), v = ld_row2(rp, jj);
        acc = fma(v.x, x.x, fma(v.y, x.y, acc));
      }
      acc = warp_sum(acc);
      for (int jj = lane; jj < nh; jj += 32) {
        const double2 c = c2[jj], v = ld_row2(rp, jj);
        const double2 o = make_double2(fma(-acc, c.x, v.x), fma(-acc, c.y, v.y));
        wp[jj] = o;
        if (r == r_first) reinterpret_cast<double2*>(next_s)[jj] = o;
      }
    }
  }
}

// dynamic smem: win_layout(...).total doubles.  Requires an empty window on entry (qmc_sweep flushes first).
// Leaves for the flush: V[l] = phi_l, Cp[l] = c_l, rows[l], mwin (and Bcur in the d.C buffer, dead afterwards).
// NT threads per walker: 128 for full crowds (4 CTAs/SM), 256 / 512 when the crowd leaves SMs idle (a move is then a
// latency chain and wider CTAs shorten every phase of it: +10 % at W = 256, +35 % at W = 64 on cfg 5).
#ifndef QMC_WIN_MINCTAS
#define QMC_WIN_MINCTAS 4
#endif
// NS > 0: the kernel is specialised for n = M = ns = NS (N = 2 NS, a table stride that covers ns): every trip count
// and row stride is a compile-time constant, loops unroll and the index arithmetic folds -- the kernel is bound by its
// instruction stream, a third of which was integer / control overhead (ncu r2).  NS = 0: any shape.
// TB: storage type of the carried inverse (double; float = mixed precision, D:R6: the block's B0 rows are widened
// on load; everything the window itself writes -- Bcur, V, Cp -- stays fp64).
// SB: the window's block of inverse rows (kdp x ns doubles, 98 KB at cfg 5) lives in shared memory instead of the d.C
// buffer -- for the 512-thread class (crowds of at most one walker per SM), where a move is a latency chain and the block-row
// update of an accepted move otherwise waits on L2 round trips; dynamic smem: win_layout(...).total + kdp ns doubles.
template <typename T, int NT, int NS = 0, typename TB = double, bool SB = false>
__global__ void __launch_bounds__(NT, NT == 128 ? QMC_WIN_MINCTAS : 512 / NT) window_kernel(CrowdDev d, int k0, int cnt)
{
  static_assert(!SB || sizeof(TB) == 8, "the shared-memory block is loaded by plain copies of fp64 rows");
  extern __shared__ double sm[];
  __shared__ SplineW<T> sw;
  const int w = blockIdx.x + d.w0, ns = sh_ns<NS>(d), nN = sh_N<NS>(d), kdp = d.kdp, tid = threadIdx.x;
  const WinLayout L = win_layout(nN, ns, kdp, (int)sizeof(T), NT);
  double* R_s = sm + L.R;
  double* b_s = sm + L.b;    // row of the current move
  double* bn_s = sm + L.bn;  // row of the next move
  double* red = sm + L.red;
  double* gauss = sm + L.gauss;
  double* pairk = sm + L.pairk;
  int* rows_s = reinterpret_cast<int*>(sm + L.rows);
  const int cstride = ((3 * ns * (int)sizeof(T) + 15) / 16) * 16 / (int)sizeof(T);
  T* cbuf = reinterpret_cast<T*>(sm + L.cbuf);
  T* vgl_s = reinterpret_cast<T*>(sm + L.vgl);
  const MoveScal ms = move_scal_smem(sm + L.mv);

  const int spin = k0 / sh_n<NS>(d), kk0 = k0 - spin * sh_n<NS>(d);
  const TB* blk = carried_inverse<TB>(d) + (((size_t)w * 2 + spin) * ns + kk0) * ns;  // B0 rows of the window
  constexpr bool B64 = sizeof(TB) == 8;
  double* Bcur = SB ? sm + L.total : d.C + (size_t)w * kdp * ns;          // their current values, once m > 0 (SB: always)
  double* Cp = d.Cp + (size_t)w * kdp * ns;
  double* V = d.V + (size_t)w * kdp * ns;
  double* Rg = d.R + (size_t)w * nN * 3;
  T* cache0 = static_cast<T*>(d.cache) + ((size_t)w * nN + k0) * 4 * ns;
  const int row_bytes = ns * 8, cache_bytes = 3 * ns * (int)sizeof(T);

  // prologue: row and gradient cache of the first move, positions, Gaussians of the first move;
  // the rest of the block is pulled into L2 (first-touch DRAM lines the first accepted move reads)
  if constexpr (B64) cp_async_cta<NT>(b_s, blk, row_bytes);
  else
    for (int j = tid; j < ns; j += NT) b_s[j] = (double)blk[j];
  cp_async_cta<NT>(cbuf, cache0, cache_bytes);
  for (int j = tid; j < 3 * nN; j += NT) R_s[j] = Rg[j];
  if (tid >= 32 && tid < 36) gauss_pieces(d, w, k0, tid - 32, gauss);
  if constexpr (SB) {
    cp_async_cta<NT>(Bcur, blk, cnt * row_bytes);
  } else {
    for (int j = tid; j < (cnt - 1) * ns * (int)sizeof(TB) / 128; j += NT)
      asm volatile("prefetch.global.L2 [%0];" ::"l"(reinterpret_cast<const char*>(blk + ns) + (size_t)j * 128));
  }
  cp_async_wait_all();
  __syncthreads();
  J2Part jnext;   // Jastrow partial of the coming move's electron at its current position
  {
    const double rk0[3] = {R_s[3 * k0], R_s[3 * k0 + 1], R_s[3 * k0 + 2]};
    jnext.us = jnext.g[0] = jnext.g[1] = jnext.g[2] = 0.0;
    j2_partial<NT>(d, R_s, k0, rk0, jnext.us, jnext.g);
  }

#ifdef QMC_PHASE_CLOCKS
  long long ph_t[8] = {0, 0, 0, 0, 0, 0, 0, 0}, ph_c = clock64();
#define PH(x) do { if (tid == 0) { const long long c_ = clock64(); ph_t[x] += c_ - ph_c; ph_c = c_; } } while (0)
#else
#define PH(x) do {} while (0)
#endif
  int m = 0, prev_acc = 0;
  for (int i = 0; i < cnt; ++i) {
    const int k = k0 + i;
#ifdef QMC_WIN_CBUF1
    T* ccur = cbuf;
#else
    T* ccur = cbuf + (i & 1) * cstride;
#endif
    T* cache_g = cache0 + (size_t)i * 4 * ns;
    const bool more = i + 1 < cnt;
    PH(0);
    // ---- G_k(R) and the proposal: row dots + the Jastrow partial prepared during the previous move ----
    win_gold_propose<T, NT, NS>(d, k, b_s, ccur, R_s, jnext, i ? pairk + 4 * prev_acc : nullptr, ms, red, gauss, &sw);
    __syncthreads();   // r' and the spline weights of r' are visible
    PH(1);
    if constexpr (NT >= 256) {
      // small crowds (a move is a latency chain): the 64 stencil rows of r' are pulled into L2 under the Jastrow sums, so
      // that the gather below waits for L2 instead of DRAM.  (At full crowds the same prefetch bought nothing: DESIGN 6.)
      const char* tab = static_cast<const char*>(d.coefs);
      const int lpr = (int)((min((unsigned)ns / Vec16<T>::W, d.tab_vecs) + 7) / 8);   // 128-byte lines of a row that hold orbitals
      for (int j = tid; j < 64 * lpr; j += NT) {
        const int row = j / lpr, l = j - row * lpr;
        const unsigned base = sw.off[0][row >> 4] + sw.off[1][(row >> 2) & 3] + sw.off[2][row & 3];
        asm volatile("prefetch.global.L2 [%0];" ::"l"(tab + (size_t)base * 16 + (size_t)l * 128));
      }
    }
    // ---- both Jastrow sums (at r' for the ratio, at r_{k+1} for the next proposal), four pair chains in flight ----
    J2Part jr;
    const double rn[3] = {ms.rn[0], ms.rn[1], ms.rn[2]};
    const int k1 = more ? k + 1 : k;
    const double rk1[3] = {R_s[3 * k1], R_s[3 * k1 + 1], R_s[3 * k1 + 2]};
    j2_two_sums<NT, NS>(d, R_s, k, rn, more, rk1, jr, jnext);
    PH(2);
    spline_cta<T, NT, NoSideWork, false, true, NS>(d, nullptr, sw, vgl_s);
    __syncthreads();
    PH(3);
    win_ratio_grad<T, NT, NS>(d, b_s, vgl_s, jr, ms, red);   // row dots + block sum; thread 0: rho_D, rho_J, G_k(R')
    PH(4);
    // ---- the decision is one thread's scalar chain (two exp, divisions, Philox): the other warps use the time for
    // what the NEXT move needs and nobody is waiting for -- its Gaussians, the pair term (k+1, k) for both outcomes
    // ([0..3] rejected, [4..7] accepted), its inverse row (valid unless this move is accepted, which rewrites it) and
    // its gradient cache ----
    if (more) {
      const int warp = tid >> 5, lane = tid & 31;
      if (warp == 1 % (NT / 32)) {
        if (lane < 4) gauss_pieces(d, w, k + 1, lane, gauss);
      }
      if (warp == 2 % (NT / 32)) {
        if (lane >= 30) {
          const bool acc_case = lane == 31;
          double us = 0.0, g[3] = {0.0, 0.0, 0.0};
          if (acc_case) j2_pair(d, rk1, rn, us, g);
          else j2_pair(d, rk1, R_s + 3 * k, us, g);
          double* o = pairk + (acc_case ? 4 : 0);
          o[0] = us; o[1] = g[0]; o[2] = g[1]; o[3] = g[2];
        }
      }
      if (warp == 3 % (NT / 32)) {
        if constexpr (SB) {
          const double2* src = reinterpret_cast<const double2*>(Bcur + (size_t)(i + 1) * ns);
          for (int j = lane; j < ns / 2; j += 32) reinterpret_cast<double2*>(bn_s)[j] = src[j];
        } else if (B64 || m) cp_async_warp(bn_s, (m ? Bcur : reinterpret_cast<const double*>(blk)) + (size_t)(i + 1) * ns, row_bytes);
        else
          for (int j = lane; j < ns; j += 32) bn_s[j] = (double)blk[(size_t)(i + 1) * ns + j];
        cp_async_warp(cbuf + ((i + 1) & 1) * cstride, cache_g + 4 * ns, cache_bytes);
      }
    }
    const int acc_ = dev_decide(d, w, k, ms, nullptr);
    prev_acc = acc_;
    PH(5);
    if (acc_) {
      const double inv_rho = 1.0 / *ms.rho_d;
      for (int j = tid; j < ns; j += NT) {
        const double c = b_s[j] * inv_rho;
        b_s[j] = c;
        Cp[(size_t)m * ns + j] = c;
        V[(size_t)m * ns + j] = (double)vgl_s[j];
      }
      for (int j = tid; j < 4 * ns * (int)sizeof(T) / 16; j += NT)   // gradient / Laplacian cache of electron k, 16 bytes at a time
        reinterpret_cast<float4*>(cache_g)[j] = reinterpret_cast<const float4*>(vgl_s + ns)[j];
      if (tid < 3) {
        const double x = ms.rn[tid];
        R_s[3 * k + tid] = x;
        Rg[3 * k + tid] = x;
      }
      if (tid == 0) rows_s[m] = kk0 + i;
      cp_async_wait_all();   // the stale copy of the next row has landed before the update overwrites it
      __syncthreads();
      if constexpr (SB) block_rows_update<T, NT>(Bcur, Bcur, ns, i + 1, cnt, vgl_s, b_s, bn_s);
      else if constexpr (B64) block_rows_update<T, NT>(m ? Bcur : reinterpret_cast<const double*>(blk), Bcur, ns, i + 1, cnt, vgl_s, b_s, bn_s);
      else if (m) block_rows_update<T, NT>(Bcur, Bcur, ns, i + 1, cnt, vgl_s, b_s, bn_s);
      else block_rows_update<T, NT, TB>(blk, Bcur, ns, i + 1, cnt, vgl_s, b_s, bn_s);
      ++m;
    }
    cp_async_wait_all();
    __syncthreads();
    PH(6);
    double* t = b_s; b_s = bn_s; bn_s = t;
  }
#ifdef QMC_PHASE_CLOCKS
  if (tid == 0)
    for (int q = 0; q < 8; ++q) d.pvec[(size_t)w * kdp + q] += (double)ph_t[q];
#endif

  for (int l = tid; l < m; l += NT) d.rows[(size_t)w * kdp + l] = rows_s[l];
  if (tid == 0) d.mwin[w] = m;
}

// ---- qmc_sweep with delay_rank = 1 and small matrices: the whole sweep in one launch -------------------
// Sherman-Morrison after every accepted move (D:C5) touches the full n x n inverse.  For large n that is the
// bandwidth-bound rank1_kernel spread over the whole GPU (update.cuh); for ns <= SWEEP1_MAX_NS (configs 1 and
// 2 of BASELINE.json: n = 4 and 32) a move takes microseconds and four launches per move are pure overhead
// (P:105), so here a CTA owns a walker for the whole sweep and applies the update itself, row by row, with
// exactly rank1_kernel's arithmetic (same lane partition, same fma order: bit-identical inverses).
constexpr int SWEEP1_MAX_NS = 128;

// B'[i,:] = B[i,:] - ((B[i,:].phi' - [i == kk]) / rho_D) b_old for all n rows of one spin block, in place.
// b_old = b_s and phi' = vgl_s[0..ns) in shared memory; row kk_next also goes to next_s (next move's row).
template <typename T>
__device__ __forceinline__ void sm_update_rows(double* B, int ns, int n, int kk, double inv_rho, const T* vgl_s,
                                               const double* b_s, int kk_next, double* next_s)
{
  constexpr int RB = 4, NV = SWEEP1_MAX_NS / 64;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nh = ns / 2;
  double2 ph[NV], bold[NV];
#pragma unroll
  for (int v = 0; v < NV; ++v) {
    const int jj = lane + 32 * v;
    ph[v] = jj < nh ? ld_x2(vgl_s, jj) : make_double2(0.0, 0.0);
    bold[v] = jj < nh ? reinterpret_cast<const double2*>(b_s)[jj] : make_double2(0.0, 0.0);
  }
  for (int i0 = warp * RB; i0 < n; i0 += MOVE_NW * RB) {
    double2 x[RB][NV];
#pragma unroll
    for (int r = 0; r < RB; ++r)
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        const int jj = lane + 32 * v;
        x[r][v] = (i0 + r < n && jj < nh) ? reinterpret_cast<const double2*>(B + (size_t)(i0 + r) * ns)[jj]
                                          : make_double2(0.0, 0.0);
      }
#pragma unroll
    for (int r = 0; r < RB; ++r) {
      const int i = i0 + r;
      if (i >= n) break;
      double acc = 0.0;
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        acc = fma(x[r][v].x, ph[v].x, acc);
        acc = fma(x[r][v].y, ph[v].y, acc);
      }
      acc = warp_sum(acc);
      const double f = (acc - (i == kk ? 1.0 : 0.0)) * inv_rho;
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        const int jj = lane + 32 * v;
        if (jj < nh) {
          x[r][v].x = fma(-f, bold[v].x, x[r][v].x);
          x[r][v].y = fma(-f, bold[v].y, x[r][v].y);
          reinterpret_cast<double2*>(B + (size_t)i * ns)[jj] = x[r][v];
          if (i == kk_next) reinterpret_cast<double2*>(next_s)[jj] = x[r][v];
        }
      }
    }
  }
}

// dynamic smem: win_layout(...).total doubles (same layout as the window kernel).  ns <= SWEEP1_MAX_NS.
template <typename T>
__global__ void __launch_bounds__(MOVE_NT, 512 / MOVE_NT) sweep1_kernel(CrowdDev d)
{
  extern __shared__ double sm[];
  __shared__ SplineW<T> sw;
  const int w = blockIdx.x + d.w0, ns = d.ns, n = d.n, tid = threadIdx.x;
  const WinLayout L = win_layout(d.N, ns, d.kdp, (int)sizeof(T));
  double* R_s = sm + L.R;
  double* b_s = sm + L.b;
  double* bn_s = sm + L.bn;
  double* red = sm + L.red;
  double* gauss = sm + L.gauss;
  const int cstride = ((3 * ns * (int)sizeof(T) + 15) / 16) * 16 / (int)sizeof(T);
  T* cbuf = reinterpret_cast<T*>(sm + L.cbuf);
  T* vgl_s = reinterpret_cast<T*>(sm + L.vgl);
  const MoveScal ms = move_scal_smem(sm + L.mv);
  double* Bw = d.Binv + (size_t)w * 2 * ns * ns;
  double* Rg = d.R + (size_t)w * d.N * 3;
  T* cache0 = static_cast<T*>(d.cache) + (size_t)w * d.N * 4 * ns;
  const int row_bytes = ns * 8, cache_bytes = 3 * ns * (int)sizeof(T);

  cp_async_cta(b_s, Bw, row_bytes);
  cp_async_cta(cbuf, cache0, cache_bytes);
  for (int j = tid; j < 3 * d.N; j += MOVE_NT) R_s[j] = Rg[j];
  if (tid >= 32 && tid < 36) gauss_pieces(d, w, 0, tid - 32, gauss);
  cp_async_wait_all();
  __syncthreads();

  for (int k = 0; k < d.N; ++k) {
    const int spin = k / n, kk = k - spin * n;
    double* B = Bw + (size_t)spin * ns * ns;
    T* ccur = cbuf + (k & 1) * cstride;
    T* cache_g = cache0 + (size_t)k * 4 * ns;
    const bool more = k + 1 < d.N;
    const int spin1 = (k + 1) / n, kk1 = (k + 1) - spin1 * n;
    if (more) {
      cp_async_cta(bn_s, Bw + ((size_t)spin1 * ns + kk1) * ns, row_bytes);
      cp_async_cta(cbuf + ((k + 1) & 1) * cstride, cache_g + 4 * ns, cache_bytes);
    }
    dev_gold_propose<T>(d, w, k, b_s, ccur, R_s, nullptr, ms, red, gauss, &sw);
    spline_cta<T, MOVE_NT>(d, nullptr, sw, vgl_s, [&](int t) {
      if (more && t < 36) gauss_pieces(d, w, k + 1, t - 32, gauss);
    });
    __syncthreads();
    dev_ratio_grad<T>(d, w, k, b_s, vgl_s, R_s, ms, nullptr, nullptr, red);
    cp_async_wait_all();
    if (dev_decide(d, w, k, ms, nullptr)) {
      const double inv_rho = 1.0 / *ms.rho_d;
      for (int j = tid; j < 4 * ns; j += MOVE_NT) cache_g[j] = vgl_s[ns + j];
      if (tid < 3) {
        const double x = ms.rn[tid];
        R_s[3 * k + tid] = x;
        Rg[3 * k + tid] = x;
      }
      sm_update_rows<T>(B, ns, n, kk, inv_rho, vgl_s, b_s, (more && spin1 == spin) ? kk1 : -1, bn_s);
    }
    __syncthreads();
    double* t = b_s; b_s = bn_s; bn_s = t;
  }
}

}  // namespace qmc
