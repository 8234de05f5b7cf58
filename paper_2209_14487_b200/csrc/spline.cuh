// spline.cuh -- tricubic B-spline orbitals: value, gradient, Laplacian.
//
// D:C1: u = x Ng/L, i = floor(u), t = u - i; the four uniform cubic B-spline weights of grid
// points i-1..i+2 (and their first/second derivatives, scaled by 1/h, 1/h^2) per axis;
// phi_j = sum_{a,b,c} A_a B_b C_c P[(ix-1+a) mod Ng][(iy-1+b) mod Ng][(iz-1+c) mod Ng][j].
// The table is orbital-innermost (BJ), so one stencil point is one contiguous row of M values.
//
// Work split (one CTA evaluates one position; the same device function serves qmc_spo_vgl, the
// Slater build at create and the walker-persistent window kernel of qmc_sweep):
//   an item = (16-byte orbital slice, x-plane a): 16 independent 16-byte loads (4 y x 4 z rows),
//   contracted z -> y in registers, scaled by the x weights of plane a.  A warp takes 8 slices x 4 planes
//   (lane = 8 a + slice): a warp request is four runs of 128 contiguous bytes, one per quarter-warp, the
//   four planes of a slice are summed by two xor-shuffles (8, 16), and every thread keeps 16 loads in
//   flight with ~64 data registers -- the 64-loads-per-thread form needed 153 registers (3 CTAs/SM).
#pragma once
#include "common.cuh"

namespace qmc {

// Per-position weights, built once per evaluation in shared memory.
template <typename T>
struct SplineW {
  T w[3][4], dw[3][4], d2w[3][4];
  unsigned off[3][4];  // offsets of the 4 grid planes / lines / points, in 16-byte vectors
};

// Axis c of the weights for coordinate x (one thread per axis).
template <typename T>
__device__ __forceinline__ void spline_axis(const CrowdDev& d, int c, double x, SplineW<T>& s)
{
  unsigned mult = d.orb_stride_v;
  if (c < 2) mult *= (unsigned)d.grid[2];
  if (c < 1) mult *= (unsigned)d.grid[1];
  const int Ng = d.grid[c];
  const double ih = d.inv_h[c];
  const double u = x * ih;
  const double fl = floor(u);
  const double t = u - fl;
  const double t2 = t * t, t3 = t2 * t, omt = 1.0 - t;
  // (multiplications by 1/6 and 1/2: an fp64 division costs ~30 dependent instructions on this serial path)
  constexpr double sixth = 1.0 / 6.0;
  const double hih = 0.5 * ih;
  s.w[c][0] = (T)(omt * omt * omt * sixth);
  s.w[c][1] = (T)((3.0 * t3 - 6.0 * t2 + 4.0) * sixth);
  s.w[c][2] = (T)((-3.0 * t3 + 3.0 * t2 + 3.0 * t + 1.0) * sixth);
  s.w[c][3] = (T)(t3 * sixth);
  s.dw[c][0] = (T)(-omt * omt * hih);
  s.dw[c][1] = (T)((3.0 * t2 - 4.0 * t) * hih);
  s.dw[c][2] = (T)((-3.0 * t2 + 2.0 * t + 1.0) * hih);
  s.dw[c][3] = (T)(t2 * hih);
  const double ih2 = ih * ih;
  s.d2w[c][0] = (T)(omt * ih2);
  s.d2w[c][1] = (T)((3.0 * t - 2.0) * ih2);
  s.d2w[c][2] = (T)((1.0 - 3.0 * t) * ih2);
  s.d2w[c][3] = (T)(t * ih2);
  // (i - 1) mod Ng, floor toward -inf (D:A11); exact in fp64 for |i| < 2^50
  const double a = fl - 1.0;
  const double q = floor(a * d.inv_grid[c]);  // may be off by one at exact multiples: fixed up below
  int i0 = (int)(a - q * (double)Ng);
  if (i0 < 0) i0 += Ng;
  if (i0 >= Ng) i0 -= Ng;
  if (i0 < 0 || i0 >= Ng) i0 = 0;  // non-finite position: stay in bounds, the weights are NaN anyway
#pragma unroll
  for (int m = 0; m < 4; ++m) {
    int g = i0 + m;
    while (g >= Ng) g -= Ng;
    s.off[c][m] = (unsigned)g * mult;
  }
}

// The 16 stencil rows (4 y x 4 z) of x-plane a for one 16-byte orbital slice `chunk`: 16 independent loads.
template <typename T, bool KEEP = false>
__device__ __forceinline__ void spline_plane_load(const T* __restrict__ tab, const SplineW<T>& s, int a, unsigned chunk,
                                                  T (&p)[4][4][Vec16<T>::W])
{
  constexpr int VW = Vec16<T>::W;
  const unsigned base = s.off[0][a] + chunk;
  const unsigned long long pol = l2_evict_first_policy();   // streaming gather: see ld16_stream
#pragma unroll
  for (int b = 0; b < 4; ++b)
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      if (KEEP) ld16_keep(tab + (size_t)(base + s.off[1][b] + s.off[2][c]) * VW, p[b][c]);
      else ld16_stream(tab + (size_t)(base + s.off[1][b] + s.off[2][c]) * VW, p[b][c], pol);
    }
}

// Contribution of x-plane a to the five quantities of the slice, from its 16 loaded rows.
// out[0] = phi, out[1..3] = d/dx, d/dy, d/dz, out[4] = laplacian.
template <typename T>
__device__ __forceinline__ void spline_plane_sum(const SplineW<T>& s, int a, const T (&p)[4][4][Vec16<T>::W],
                                                 T (&out)[5][Vec16<T>::W])
{
  constexpr int VW = Vec16<T>::W;
  T u00[VW], u10[VW], u20[VW], u01[VW], u02[VW];
#pragma unroll
  for (int e = 0; e < VW; ++e) u00[e] = u10[e] = u20[e] = u01[e] = u02[e] = (T)0;
#pragma unroll
  for (int b = 0; b < 4; ++b) {
#pragma unroll
    for (int e = 0; e < VW; ++e) {
      T v0 = s.w[2][0] * p[b][0][e], v1 = s.dw[2][0] * p[b][0][e], v2 = s.d2w[2][0] * p[b][0][e];
#pragma unroll
      for (int c = 1; c < 4; ++c) {
        v0 = fma(s.w[2][c], p[b][c][e], v0);
        v1 = fma(s.dw[2][c], p[b][c][e], v1);
        v2 = fma(s.d2w[2][c], p[b][c][e], v2);
      }
      u00[e] = fma(s.w[1][b], v0, u00[e]);
      u10[e] = fma(s.dw[1][b], v0, u10[e]);
      u20[e] = fma(s.d2w[1][b], v0, u20[e]);
      u01[e] = fma(s.w[1][b], v1, u01[e]);
      u02[e] = fma(s.w[1][b], v2, u02[e]);
    }
  }
  const T wa = s.w[0][a], dwa = s.dw[0][a], d2wa = s.d2w[0][a];
#pragma unroll
  for (int e = 0; e < VW; ++e) {
    out[0][e] = wa * u00[e];
    out[1][e] = dwa * u00[e];
    out[2][e] = wa * u10[e];
    out[3][e] = wa * u01[e];
    out[4][e] = fma(d2wa, u00[e], wa * (u20[e] + u02[e]));
  }
}

// The same contraction for an fp32 table with packed arithmetic (sm_100 FFMA2 / FMUL2 / FADD2: two IEEE operations
// per instruction on a register pair): element for element the same products and sums in the same order as the generic
// version, i.e. bit-identical results with half the floating-point instructions (they were a quarter of the window
// kernel's instruction stream, which is what bounds it: ncu r2).
__device__ __forceinline__ void spline_plane_sum(const SplineW<float>& s, int a, const float (&p)[4][4][4], float (&out)[5][4])
{
  float2 u00[2], u10[2], u20[2], u01[2], u02[2];
#pragma unroll
  for (int h = 0; h < 2; ++h) u00[h] = u10[h] = u20[h] = u01[h] = u02[h] = make_float2(0.f, 0.f);
  float2 wz[4], dwz[4], d2wz[4];
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    wz[c] = make_float2(s.w[2][c], s.w[2][c]);
    dwz[c] = make_float2(s.dw[2][c], s.dw[2][c]);
    d2wz[c] = make_float2(s.d2w[2][c], s.d2w[2][c]);
  }
#pragma unroll
  for (int b = 0; b < 4; ++b) {
    const float2 wy = make_float2(s.w[1][b], s.w[1][b]), dwy = make_float2(s.dw[1][b], s.dw[1][b]),
                 d2wy = make_float2(s.d2w[1][b], s.d2w[1][b]);
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const float2 p0 = make_float2(p[b][0][2 * h], p[b][0][2 * h + 1]);
      float2 v0 = __fmul2_rn(wz[0], p0), v1 = __fmul2_rn(dwz[0], p0), v2 = __fmul2_rn(d2wz[0], p0);
#pragma unroll
      for (int c = 1; c < 4; ++c) {
        const float2 pc = make_float2(p[b][c][2 * h], p[b][c][2 * h + 1]);
        v0 = __ffma2_rn(wz[c], pc, v0);
        v1 = __ffma2_rn(dwz[c], pc, v1);
        v2 = __ffma2_rn(d2wz[c], pc, v2);
      }
      u00[h] = __ffma2_rn(wy, v0, u00[h]);
      u10[h] = __ffma2_rn(dwy, v0, u10[h]);
      u20[h] = __ffma2_rn(d2wy, v0, u20[h]);
      u01[h] = __ffma2_rn(wy, v1, u01[h]);
      u02[h] = __ffma2_rn(wy, v2, u02[h]);
    }
  }
  const float2 wa = make_float2(s.w[0][a], s.w[0][a]), dwa = make_float2(s.dw[0][a], s.dw[0][a]),
               d2wa = make_float2(s.d2w[0][a], s.d2w[0][a]);
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    const float2 o0 = __fmul2_rn(wa, u00[h]), o1 = __fmul2_rn(dwa, u00[h]), o2 = __fmul2_rn(wa, u10[h]),
                 o3 = __fmul2_rn(wa, u01[h]), o4 = __ffma2_rn(d2wa, u00[h], __fmul2_rn(wa, __fadd2_rn(u20[h], u02[h])));
    out[0][2 * h] = o0.x; out[0][2 * h + 1] = o0.y;
    out[1][2 * h] = o1.x; out[1][2 * h + 1] = o1.y;
    out[2][2 * h] = o2.x; out[2][2 * h + 1] = o2.y;
    out[3][2 * h] = o3.x; out[3][2 * h + 1] = o3.y;
    out[4][2 * h] = o4.x; out[4][2 * h + 1] = o4.y;
  }
}

__device__ __forceinline__ float shfl_xor_t(float v, int m) { return __shfl_xor_sync(0xffffffffu, v, m); }
__device__ __forceinline__ double shfl_xor_t(double v, int m) { return __shfl_xor_sync(0xffffffffu, v, m); }

// Sum over the four planes (lanes 8 a + slice) with the owner of each quantity as the only receiver: plane a's lane ends
// up with quantity a of the slice (f0), plane 0's also with the laplacian (f1).  Same pairwise tree per value as two full
// xor-shuffles, (p_a + p_{a^1}) + (p_{a^2} + p_{a^3}), with 5 instead of 10 shuffles per value.
template <typename T>
__device__ __forceinline__ void spline_plane_reduce(int a, const T (&out)[5][Vec16<T>::W], T (&f0)[Vec16<T>::W], T (&f1)[Vec16<T>::W])
{
  constexpr int VW = Vec16<T>::W;
  const bool odd = a & 1, up = a & 2;
  T r0[VW], r1[VW], r2[VW];  // after step 1: even lanes hold q0, q2, q4; odd lanes hold q1, q3 (r2 unused)
#pragma unroll
  for (int e = 0; e < VW; ++e) {
    const T s0 = odd ? out[0][e] : out[1][e], s1 = odd ? out[2][e] : out[3][e], s2 = odd ? out[4][e] : (T)0;
    const T k0 = odd ? out[1][e] : out[0][e], k1 = odd ? out[3][e] : out[2][e], k2 = out[4][e];
    r0[e] = k0 + shfl_xor_t(s0, 8);
    r1[e] = k1 + shfl_xor_t(s1, 8);
    r2[e] = k2 + shfl_xor_t(s2, 8);
  }
  // after step 2: plane 0: q0, q4; plane 1: q1; plane 2: q2; plane 3: q3
#pragma unroll
  for (int e = 0; e < VW; ++e) {
    const T s0 = up ? r0[e] : r1[e], s1 = up ? r2[e] : (T)0;
    const T k0 = up ? r1[e] : r0[e], k1 = r2[e];
    f0[e] = k0 + shfl_xor_t(s0, 16);
    f1[e] = k1 + shfl_xor_t(s1, 16);
  }
}

// All orbitals at position r by the whole CTA (NT threads, NT % 32 == 0).  `s` is shared memory;
// `vgl` (global or shared) receives [5][ns]: phi, d/dx, d/dy, d/dz, laplacian, zero beyond M.
// Contains two __syncthreads(); must be called by all threads of the CTA.
// `side(tid)` runs on the threads of warps >= 1 right after the first round of loads has been issued, i.e. under
// their DRAM latency (a slot for work that is off the caller's critical path).
struct NoSideWork { __device__ __forceinline__ void operator()(int) const {} };
// r == nullptr: the caller has already filled `s` for this position (spline_axis per axis).
// KEEP: loads without the L2 evict-first hint (callers that arrange for L2 re-use).
// PRESYNCED: the caller has already synchronised after filling `s` (and may have done work of its own in between).
template <typename T, int NT, typename Side = NoSideWork, bool KEEP = false, bool PRESYNCED = false, int NS = 0>
__device__ __forceinline__ void spline_cta(const CrowdDev& d, const double* r, SplineW<T>& s, T* vgl, Side side = Side())
{
  constexpr int VW = Vec16<T>::W;
  // lane = 8 a + slice: the eight lanes of a quarter-warp read eight adjacent 16-byte slices of ONE row (one 128-byte
  // line = one L1 wavefront per quarter-warp of a 128-bit load; with the four planes in adjacent lanes a quarter-warp
  // touched four lines and the gather cost four times the wavefronts -- the L1 data pipe was the busiest unit of the
  // window kernel, ncu r2).  The planes of a slice sit 8 and 16 lanes apart.
  const int tid = threadIdx.x, lane = tid & 31, a = lane >> 3, g = (tid >> 5) * 8 + (lane & 7);
  if (!PRESYNCED) __syncthreads();  // previous users of `s` are done / the caller's weights are visible
  if (r) {
    if (tid < 3) spline_axis<T>(d, tid, r[tid], s);
    __syncthreads();
  }
  const T* tab = static_cast<const T*>(d.coefs);
  const unsigned chunks = (unsigned)sh_ns<NS>(d) / VW;
#pragma unroll 1
  for (unsigned c0 = 0; c0 < chunks; c0 += NT / 4) {
    const unsigned chunk = c0 + g;
    T out[5][VW];
    // shape known at compile time with the slices filling every round: no bounds checks, no masking of padding columns
    constexpr bool FULL = NS > 0 && (NS / VW) % (NT / 4) == 0;
    if (FULL || (chunk < sh_tab_vecs<NS>(d) && chunk < chunks)) {
      T p[4][4][VW];
      spline_plane_load<T, KEEP>(tab, s, a, chunk, p);
      if (c0 == 0 && tid >= 32) side(tid);
      spline_plane_sum(s, a, p, out);
    } else {
      if (c0 == 0 && tid >= 32) side(tid);
#pragma unroll
      for (int q = 0; q < 5; ++q)
#pragma unroll
        for (int e = 0; e < VW; ++e) out[q][e] = (T)0;
    }
    T f0[VW], f1[VW];
    spline_plane_reduce<T>(a, out, f0, f1);
#pragma unroll
    for (int e = 0; e < VW; ++e)
      if (!FULL && (int)(chunk * VW) + e >= sh_M<NS>(d)) f0[e] = f1[e] = (T)0;
    if (FULL || chunk < chunks) {
      T* o = vgl + (size_t)chunk * VW;
      st16(o + (size_t)a * sh_ns<NS>(d), f0);
      if (a == 0) st16(o + (size_t)4 * sh_ns<NS>(d), f1);
    }
  }
}

constexpr int SPLINE_NT = 128;

// qmc_spo_vgl step (c): one CTA per walker at r' = d.rnew[w]; output d.vgl[w].
template <typename T>
__global__ void __launch_bounds__(SPLINE_NT, 4) spline_vgl_kernel(CrowdDev d)
{
  __shared__ SplineW<T> s;
  const int w = blockIdx.x;
  spline_cta<T, SPLINE_NT>(d, d.rnew + 3 * (size_t)w, s, static_cast<T*>(d.vgl) + (size_t)w * 5 * d.ns);
}

// qmc_crowd_create / set_positions on small crowds (fewer than 256 positions; larger ones take the cell-sorted build
// below): one CTA per (walker, electron) at the electron's own position; fills the caches and the transposed Slater
// matrix X[j][i] = phi_j(r_i) that the inversion kernel turns into B = (A^-1)^T = (A^T)^-1 (D:C2).
// dynamic smem: 5 ns elements of T.
template <typename T>
__global__ void __launch_bounds__(SPLINE_NT, 4) spline_build_kernel(CrowdDev d)
{
  extern __shared__ double sm_build[];
  __shared__ SplineW<T> s;
  T* v_s = reinterpret_cast<T*>(sm_build);
  const size_t we = (size_t)blockIdx.x;
  const int w = (int)(we / d.N), e_idx = (int)(we - (size_t)w * d.N);
  spline_cta<T, SPLINE_NT>(d, d.R + 3 * we, s, v_s);
  __syncthreads();
  const int spin = e_idx / d.n, i = e_idx - spin * d.n;
  T* cache = static_cast<T*>(d.cache) + we * 4 * d.ns;
  double* X = d.Binv + ((size_t)w * 2 + spin) * d.ns * d.ns;
  for (int j = threadIdx.x; j < 4 * d.ns; j += SPLINE_NT) cache[j] = v_s[d.ns + j];
  for (int j = threadIdx.x; j < d.M; j += SPLINE_NT) X[(size_t)j * d.ns + i] = (double)v_s[j];
}

// X <- X^T for every ns x ns matrix of the crowd, in place: CTA (a, matrix) swaps the 16 x 16 tiles (a, b) and (b, a)
// for b >= a through shared memory (coalesced both ways).  grid = (ns / 16, 2 W), 256 threads.
__global__ void __launch_bounds__(256) transpose_inplace_kernel(CrowdDev d)
{
  __shared__ double t0[16][17], t1[16][17];
  const int ns = d.ns, a = blockIdx.x, tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  double* X = d.Binv + (size_t)blockIdx.y * ns * ns;
  for (int b = a; b < ns / 16; ++b) {
    t0[ty][tx] = X[(size_t)(16 * a + ty) * ns + 16 * b + tx];
    t1[ty][tx] = X[(size_t)(16 * b + ty) * ns + 16 * a + tx];
    __syncthreads();
    X[(size_t)(16 * b + ty) * ns + 16 * a + tx] = t0[tx][ty];
    if (b != a) X[(size_t)(16 * a + ty) * ns + 16 * b + tx] = t1[tx][ty];
    __syncthreads();
  }
}

// ---- counting sort of the (walker, electron) positions by grid cell, z fastest like the table ----------------------
__device__ __forceinline__ int cell_of(const CrowdDev& d, const double* r)
{
  int idx = 0;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    double u = r[c] * d.inv_box[c];
    u -= floor(u);
    int i = (int)(u * d.grid[c]);
    i = i < 0 ? 0 : (i >= d.grid[c] ? d.grid[c] - 1 : i);   // non-finite positions land in the first / last cell
    idx = idx * d.grid[c] + i;
  }
  return idx;
}
__global__ void cell_count_kernel(CrowdDev d, int* bins)
{
  const size_t we = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (we < (size_t)d.W * d.N) atomicAdd(bins + cell_of(d, d.R + 3 * we), 1);
}
// exclusive scan of bins[0 .. nb) in place, one CTA of 1024 threads, each thread a contiguous chunk
__global__ void __launch_bounds__(1024) cell_scan_kernel(int* bins, int nb)
{
  __shared__ int part[1024];
  const int tid = threadIdx.x, per = (nb + 1023) / 1024, lo = min(tid * per, nb), hi = min(lo + per, nb);
  int sum = 0;
  for (int i = lo; i < hi; ++i) sum += bins[i];
  part[tid] = sum;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {
    const int v = tid >= o ? part[tid - o] : 0;
    __syncthreads();
    part[tid] += v;
    __syncthreads();
  }
  int run = part[tid] - sum;
  for (int i = lo; i < hi; ++i) {
    const int v = bins[i];
    bins[i] = run;
    run += v;
  }
}
__global__ void cell_scatter_kernel(CrowdDev d, int* bins, int* order)
{
  const size_t we = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (we < (size_t)d.W * d.N) order[atomicAdd(bins + cell_of(d, d.R + 3 * we), 1)] = (int)we;
}

// The Slater build over positions sorted by grid cell (qmc_crowd_create / set_positions / recompute on crowds of 256
// positions and more).  CTAs in flight together gather overlapping stencils, so the table is streamed from DRAM about
// once instead of once per position, and the positions of one cell share their 64 stencil rows outright: the CTA of a
// cell (grid = cells; its range in `order` is bins[cell - 1] .. bins[cell] after the scatter; empty cells exit) takes its
// positions in runs of up to BUILD_RUN, stages the 64 rows in shared memory ONCE per run (in column segments of
// BUILD_SEG_BYTES per row: 96 KB, two CTAs per SM) and evaluates every position of the run from there -- a thread takes
// one 16-byte orbital slice of one position through all four x-planes, so the planes are summed in registers.  At cfg 5,
// W = 4096 a cell holds 6 positions on average: against one CTA per position with the planes spread over lanes (the
// form the move kernels use, where a position is evaluated alone) the L2 -> SM traffic falls from 308 GB to 50 GB and the
// instruction count by 2.4 (no shuffle tree, weights read once per four planes).  Same arithmetic per value as
// spline_cta -- the same plane sums, added as (p0 + p1) + (p2 + p3) like its shuffle tree -- so the results are
// bit-identical to the per-position form.  The outputs go straight to global memory: the caches [4][ns] and row i of the
// row-major Slater matrix A (one contiguous row per electron -- the CTAs of one walker are not neighbours in time,
// strided 8-byte writes of A^T would not merge in L2 -- transposed in place afterwards by transpose_inplace_kernel).
// A position whose stencil offsets differ from the run's first (the cell index and the spline's own floor are computed
// differently and may disagree on a cell face) starts a new sub-run with its own staging.
constexpr int BUILD_RUN = 16;
constexpr int BUILD_NT = 192;
constexpr int BUILD_SEG_BYTES = 1536;
constexpr size_t BUILD_SMEM = (size_t)64 * BUILD_SEG_BYTES;

__device__ __forceinline__ float add_rn(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ double add_rn(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ void st_phi_row(double* x, const float (&f)[4]) { st32(x, (double)f[0], (double)f[1], (double)f[2], (double)f[3]); }
__device__ __forceinline__ void st_phi_row(double* x, const double (&f)[2]) { *reinterpret_cast<double2*>(x) = make_double2(f[0], f[1]); }

template <typename T>
__global__ void __launch_bounds__(BUILD_NT, 2) spline_build_cells_kernel(CrowdDev d, const int* __restrict__ order,
                                                                         const int* __restrict__ bins)
{
  constexpr int VW = Vec16<T>::W, NT = BUILD_NT;
  constexpr unsigned SEGV = BUILD_SEG_BYTES / 16;   // 16-byte vectors per staged row
  constexpr int PP = NT / SEGV;                     // positions evaluated side by side
  static_assert(NT % SEGV == 0 && PP >= 1, "a thread owns one slice of the segment");
  extern __shared__ __align__(16) unsigned char sm_cells[];
  T* st = reinterpret_cast<T*>(sm_cells);           // [64][SEGV * VW]
  __shared__ SplineW<T> sw[BUILD_RUN];
  __shared__ double* s_x[BUILD_RUN];                // row i of the position's Slater matrix
  __shared__ T* s_cache[BUILD_RUN];
  const int cell = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int start = cell ? bins[cell - 1] : 0, end = bins[cell];   // the cell's range in `order` (after the scatter)
  const T* tab = static_cast<const T*>(d.coefs);
  const unsigned chunks = (unsigned)d.ns / VW;
  const unsigned v = tid % SEGV;
  const int jp = tid / SEGV;
  for (int b0 = start; b0 < end; b0 += BUILD_RUN) {
    const int cnt = min(BUILD_RUN, end - b0);
    __syncthreads();   // the previous run's weights are no longer read
    if (tid < 3 * cnt) {
      const int j = tid / 3, c = tid - 3 * j;
      const size_t we = (size_t)order[b0 + j];
      spline_axis<T>(d, c, d.R[3 * we + c], sw[j]);
      if (c == 0) {
        const int w = (int)(we / d.N), e_idx = (int)(we - (size_t)w * d.N);
        const int spin = e_idx / d.n, i = e_idx - spin * d.n;
        s_x[j] = d.Binv + ((size_t)w * 2 + spin) * d.ns * d.ns + (size_t)i * d.ns;
        s_cache[j] = static_cast<T*>(d.cache) + we * 4 * d.ns;
      }
    }
    __syncthreads();
    for (int q = 0; q < cnt;) {
      int qe = q + 1;
      while (qe < cnt && sw[qe].off[0][0] == sw[q].off[0][0] && sw[qe].off[1][0] == sw[q].off[1][0] &&
             sw[qe].off[2][0] == sw[q].off[2][0])
        ++qe;
      for (unsigned v0 = 0; v0 < chunks; v0 += SEGV) {
        const unsigned nv = min(SEGV, chunks - v0);
        __syncthreads();   // the readers of the previous segment are done
        for (int row = warp; row < 64; row += NT / 32) {   // a warp stages whole rows: contiguous 16-byte pieces
          const unsigned src0 = sw[q].off[0][row >> 4] + sw[q].off[1][(row >> 2) & 3] + sw[q].off[2][row & 3] + v0;
          for (unsigned vv = lane; vv < nv; vv += 32) {
            T* dst = st + ((size_t)row * SEGV + vv) * VW;
            if (v0 + vv < d.tab_vecs) {
              cp_async16(dst, tab + (size_t)(src0 + vv) * VW);
            } else {
#pragma unroll
              for (int e = 0; e < VW; ++e) dst[e] = (T)0;   // columns the table does not hold (all >= M: masked below)
            }
          }
        }
        cp_async_wait_all();
        __syncthreads();
        if (v < nv) {
          const unsigned chunk = v0 + v;
          for (int j = q + jp; j < qe; j += PP) {
            const SplineW<T>& s = sw[j];
            T o01[5][VW], o2[5][VW], res[5][VW];
#pragma unroll
            for (int a = 0; a < 4; ++a) {
              T p[4][4][VW], o[5][VW];
#pragma unroll
              for (int bb = 0; bb < 4; ++bb)
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                  const T* src = st + ((size_t)(16 * a + 4 * bb + c) * SEGV + v) * VW;
#pragma unroll
                  for (int e = 0; e < VW; ++e) p[bb][c][e] = src[e];
                }
              spline_plane_sum(s, a, p, o);
#pragma unroll
              for (int k = 0; k < 5; ++k)
#pragma unroll
                for (int e = 0; e < VW; ++e) {
                  if (a == 0) o01[k][e] = o[k][e];
                  if (a == 1) o01[k][e] = add_rn(o01[k][e], o[k][e]);   // (never contracted with the products behind o)
                  if (a == 2) o2[k][e] = o[k][e];
                  if (a == 3) res[k][e] = add_rn(o01[k][e], add_rn(o2[k][e], o[k][e]));
                }
            }
#pragma unroll
            for (int e = 0; e < VW; ++e)
              if ((int)(chunk * VW) + e >= d.M) res[0][e] = res[1][e] = res[2][e] = res[3][e] = res[4][e] = (T)0;
            st_phi_row(s_x[j] + (size_t)chunk * VW, res[0]);
            T* cache = s_cache[j] + (size_t)chunk * VW;
#pragma unroll
            for (int k = 0; k < 4; ++k) st16(cache + (size_t)k * d.ns, res[k + 1]);
          }
        }
      }
      q = qe;
    }
  }
}

}  // namespace qmc
