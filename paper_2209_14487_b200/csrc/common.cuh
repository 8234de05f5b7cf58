// common.cuh -- device-side view of a crowd and small helpers shared by the kernels.
//
// Layout of the caller-owned workspace:
//   R      fp64 [W][N][3]          positions, not wrapped (D:C1)
//   Binv   fp64 [W][2][ns][ns]     B = (A^-1)^T per spin, row = electron (D:A9); ns = n rounded
//                                  (mixed precision, D:R6: carried as fp32 in Binv32 [W][2][ns][ns])
//                                  up to 16, padding rows/columns are zero and stay zero
//   cache  T    [W][N][4][ns]      d/dx, d/dy, d/dz, laplacian of phi at the electron's current
//                                  position (D:A12, A13); T = table type
//   vgl    T    [W][5][ns]         phi, d/dx, d/dy, d/dz, lap at the proposed position
//   brow   fp64 [W][ns]            inverse row of the moved electron, window applied (D:C6)
//   V, C, Cp fp64 [W][kdp][ns]     delayed window rows (C doubles as Bcur / Z, Cp = c_l of the window
//                                  kernel); kdp = delay rank padded to 8/16/32/64
//   Sinv   fp64 [W][kdp][kdp]      inverse of S = V C^T, grown by bordering
//   per-walker scalars of the move in flight (rnew, delta, g_old, g_new, ...)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace qmc {

struct CrowdDev {
  int W, N, n, M, ns;
  int kd, kdp;
  int walker_id0;
  int w0;  // first walker of this launch (sub-crowds of qmc_sweep run on two streams; 0 otherwise)
  unsigned seed_lo, seed_hi;
  int grid[3];
  double tau, sqrt_tau, j2_a, j2_b;
  double box[3], inv_box[3], inv_h[3], inv_grid[3];
  unsigned orb_stride_v;  // orbital stride of the table in 16-byte vectors
  unsigned tab_vecs;      // vectors of the table that hold orbitals < orb_stride (per grid point)
  const void* coefs;
  double* R;
  double* Binv;
  float* Binv32;  // mixed precision (D:R6): the carried inverses, stored in fp32 [W][2][ns][ns]; Binv is then the
                  // fp64 scratch of the (re)inversion.  nullptr: the inverses are carried in Binv
  void* cache;
  void* vgl;
  double* brow;
  double *rnew, *delta, *g_old, *g_new;      // [W][3]
  double *usum_old, *rho_d, *rho_j, *p, *u;  // [W]
  unsigned char* accepted;                   // [W]
  double *V, *C, *Cp, *Sinv, *pvec, *yvec;
  int* rows;                                 // [W][kdp]
  int* mwin;                                 // [W]
  double* e_elec;                            // [W][N] per-electron kinetic terms (qmc_kinetic_energy); int[W N] build order
  int* cell_bins;                            // [cells + 1] grid-cell histogram / offsets of the Slater build (or null)
  unsigned long long* counters;              // [0] accepted moves
  unsigned* sweep;                           // [1] Philox counter word 2
  int* status;                               // [1] != 0: singular matrix met
};

// Shape accessors of shape-specialised kernels: NS > 0 means n = M = ns = NS and N = 2 NS are compile-time constants
// (and the table's orbital stride covers ns); NS = 0 reads the crowd's own fields.
template <int NS> __device__ __forceinline__ int sh_ns(const CrowdDev& d) { return NS > 0 ? NS : d.ns; }
template <int NS> __device__ __forceinline__ int sh_M(const CrowdDev& d) { return NS > 0 ? NS : d.M; }
template <int NS> __device__ __forceinline__ int sh_n(const CrowdDev& d) { return NS > 0 ? NS : d.n; }
template <int NS> __device__ __forceinline__ int sh_N(const CrowdDev& d) { return NS > 0 ? 2 * NS : d.N; }
template <int NS> __device__ __forceinline__ unsigned sh_tab_vecs(const CrowdDev& d) { return NS > 0 ? 0xffffffffu : d.tab_vecs; }

// Row i of the carried inverse of (walker, spin): read where it is stored, widened to fp64 (non-hot kernels; the hot
// kernels are templated on the storage type).
__device__ __forceinline__ double ld_binv(const CrowdDev& d, size_t idx)
{
  return d.Binv32 ? (double)d.Binv32[idx] : d.Binv[idx];
}

template <typename T> struct Vec16;
template <> struct Vec16<float> { static constexpr int W = 4; };
template <> struct Vec16<double> { static constexpr int W = 2; };

// Streaming 16-byte loads of read-only data with an L2 evict-first policy (the spline table is gathered once per
// move and must not push the per-walker state out of L2: window kernel 4.94 -> 4.63 ms at cfg 5, W = 4096; an
// evict_last policy on the walker's own block rows, tried on top, was slightly slower and is not used).
// pol: createpolicy.fractional.L2::evict_first.
__device__ __forceinline__ unsigned long long l2_evict_first_policy()
{
  unsigned long long pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ void ld16_stream(const float* p, float (&v)[4], unsigned long long pol)
{
  asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.f32 {%0,%1,%2,%3}, [%4], %5;"
               : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]) : "l"(p), "l"(pol));
}
__device__ __forceinline__ void ld16_stream(const double* p, double (&v)[2], unsigned long long pol)
{
  asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;" : "=d"(v[0]), "=d"(v[1]) : "l"(p), "l"(pol));
}
// The same loads without the evict-first hint, for gathers that are arranged to re-use lines in L2 (spline_build_kernel
// visits the positions in grid-cell order).
__device__ __forceinline__ void ld16_keep(const float* p, float (&v)[4])
{
  asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]) : "l"(p));
}
__device__ __forceinline__ void ld16_keep(const double* p, double (&v)[2])
{
  asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(v[0]), "=d"(v[1]) : "l"(p));
}
__device__ __forceinline__ void st16(float* p, const float (&v)[4])
{
  *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
}
__device__ __forceinline__ void st16(double* p, const double (&v)[2])
{
  *reinterpret_cast<double2*>(p) = make_double2(v[0], v[1]);
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Sum NV values over a block of NT threads; every thread gets the totals. sm: NV*NT/32 doubles.
template <int NV, int NT>
__device__ __forceinline__ void block_sum(double (&v)[NV], double* sm)
{
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int i = 0; i < NV; ++i) v[i] = warp_sum(v[i]);
  if (lane == 0) {
#pragma unroll
    for (int i = 0; i < NV; ++i) sm[warp * NV + i] = v[i];
  }
  __syncthreads();
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    double s = 0.0;
#pragma unroll
    for (int w = 0; w < NT / 32; ++w) s += sm[w * NV + i];
    v[i] = s;
  }
  __syncthreads();
}

// Sum NV <= 8 values over a block of NT threads; only threads 0, 1, 2 get the totals (v of the other threads
// is left undefined).  Within a warp the eight sums are reduced together by a butterfly that halves the number
// of live values at each of the first three steps (9 double shuffles instead of 40); every partial is the
// same pairwise tree (xor 16, 8, 4, 2, 1) as warp_sum, so the totals are bit-identical to block_sum's.
// sm: 8*NT/32 doubles.
template <int NV, int NT>
__device__ __forceinline__ void block_sum_t0(double (&v)[NV], double* sm)
{
  static_assert(NV <= 8, "block_sum_t0 reduces at most 8 values");
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double a[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) a[i] = i < NV ? v[i] : 0.0;
  double b[4], c[2], e;
  {
    const bool hi = lane & 16;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const double keep = hi ? a[i + 4] : a[i], send = hi ? a[i] : a[i + 4];
      b[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
    }
  }
  {
    const bool hi = lane & 8;
#pragma unroll
    for (int i = 0; i < 2; ++i) {
      const double keep = hi ? b[i + 2] : b[i], send = hi ? b[i] : b[i + 2];
      c[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
    }
  }
  {
    const bool hi = lane & 4;
    const double keep = hi ? c[1] : c[0], send = hi ? c[0] : c[1];
    e = keep + __shfl_xor_sync(0xffffffffu, send, 4);
  }
  e += __shfl_xor_sync(0xffffffffu, e, 2);
  e += __shfl_xor_sync(0xffffffffu, e, 1);
  // lane now holds quantity q = 4 [bit 4] + 2 [bit 3] + [bit 2]
  const int q = ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1);
  if ((lane & 3) == 0) sm[warp * 8 + q] = e;
  __syncthreads();
  if (threadIdx.x < 3) {
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      double s = 0.0;
#pragma unroll
      for (int w = 0; w < NT / 32; ++w) s += sm[w * 8 + i];
      v[i] = s;
    }
  }
  __syncthreads();
}

// Sum eight values over a warp; every lane gets the eight totals.  Same butterfly (and the same pairwise tree per
// value) as block_sum_t0, followed by eight broadcasts: 17 double shuffles instead of 40.
__device__ __forceinline__ void warp_sum8(double (&v)[8])
{
  const int lane = threadIdx.x & 31;
  double b[4], c[2], e;
  {
    const bool hi = lane & 16;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const double keep = hi ? v[i + 4] : v[i], send = hi ? v[i] : v[i + 4];
      b[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
    }
  }
  {
    const bool hi = lane & 8;
#pragma unroll
    for (int i = 0; i < 2; ++i) {
      const double keep = hi ? b[i + 2] : b[i], send = hi ? b[i] : b[i + 2];
      c[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
    }
  }
  {
    const bool hi = lane & 4;
    const double keep = hi ? c[1] : c[0], send = hi ? c[0] : c[1];
    e = keep + __shfl_xor_sync(0xffffffffu, send, 4);
  }
  e += __shfl_xor_sync(0xffffffffu, e, 2);
  e += __shfl_xor_sync(0xffffffffu, e, 1);
  // a lane holds quantity q = 4 [bit 4] + 2 [bit 3] + [bit 2]
#pragma unroll
  for (int q = 0; q < 8; ++q) v[q] = __shfl_sync(0xffffffffu, e, ((q >> 2) & 1) * 16 + ((q >> 1) & 1) * 8 + (q & 1) * 4);
}

// 1/x and 1/sqrt(x) for normal positive x: the hardware's approximate seed (MUFU.RCP64H / RSQ64H, relative error e with
// |e| < 2^-22) and ONE third-order correction in fma arithmetic -- 1/x = y (1 + e + e^2 + O(e^3)) with e = 1 - x y,
// 1/sqrt(x) = y (1 + e/2 + 3 e^2/8 + O(e^3)) with e = 1 - x y^2 -- i.e. full double precision to within an ulp or two
// (the neglected terms are below 2^-66), without the special-case branches of the library versions.  Used by the
// Jastrow pair terms, whose arguments are well inside the normal range.
__device__ __forceinline__ double rcp_pos(double x)
{
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double e = fma(-x, y, 1.0);
  return fma(y, fma(e, e, e), y);
}
__device__ __forceinline__ double rsqrt_pos(double x)
{
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double e = fma(-(x * y), y, 1.0);
  return fma(y, e * fma(e, 0.375, 0.5), y);
}

// ---- Philox4x32-10 (Salmon et al., SC'11; D:C7). Counter (walker id, k, sweep, tag). ----
__device__ __forceinline__ void philox4x32_10(unsigned c0, unsigned c1, unsigned c2, unsigned c3, unsigned k0,
                                              unsigned k1, unsigned (&out)[4])
{
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    if (r > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
    const unsigned hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const unsigned hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    const unsigned n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

__device__ __forceinline__ double u01(unsigned x) { return ((double)x + 0.5) * (1.0 / 4294967296.0); }

// 16-byte asynchronous copy global -> shared through L2 only (L1 is not involved).  SASS: LDGSTS.
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem)
{
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// 32-byte vector access (sm_100: ld/st.global.v4.f64 -> LDG.E.256 / STG.E.256): one L1 request per lane
// instead of two; p must be 32-byte aligned.
__device__ __forceinline__ void ld32(const double* p, double (&v)[4])
{
  asm volatile("ld.global.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(v[0]), "=d"(v[1]), "=d"(v[2]), "=d"(v[3]) : "l"(p));
}
__device__ __forceinline__ void st32(double* p, double a, double b, double c, double d)
{
  asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}

// FP64 tensor-core tile: D(8x8) += A(8x4, row) B(4x8, col). Lane l holds A[l/4][l%4],
// B[l%4][l/4] and D[l/4][2(l%4) + {0,1}].  SASS: DMMA.8x8x4.
__device__ __forceinline__ void dmma884(double (&c)[2], double a, double b)
{
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c[0]), "+d"(c[1])
               : "d"(a), "d"(b));
}

}  // namespace qmc
