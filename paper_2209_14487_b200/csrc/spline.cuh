// spline.cuh -- tricubic B-spline orbitals: value, gradient, Laplacian.
//
// D:C1: u = x Ng/L, i = floor(u), t = u - i; the four uniform cubic B-spline weights of grid
// points i-1..i+2 (and their first/second derivatives, scaled by 1/h, 1/h^2) per axis;
// phi_j = sum_{a,b,c} A_a B_b C_c P[(ix-1+a) mod Ng][(iy-1+b) mod Ng][(iz-1+c) mod Ng][j].
// The table is orbital-innermost (BJ), so one stencil point is one contiguous row of M values:
// a thread owns one 16-byte slice of the orbital range (4 fp32 / 2 fp64 orbitals) of one walker
// and reads its slice of all 64 rows as 64 independent 16-byte loads; consecutive threads read
// consecutive slices, so every warp request is a run of full 128-byte lines.
// The 64-term sum is contracted z -> y -> x (300 FMA per orbital instead of 320 + weights).
#pragma once
#include "common.cuh"

namespace qmc {

template <typename T>
struct SplineW {
  T w[3][4], dw[3][4], d2w[3][4];
  unsigned off[3][4];  // offsets of the 4 grid planes / lines / points, in 16-byte vectors
};

template <typename T>
__device__ __forceinline__ void spline_setup(const CrowdDev& d, const double* __restrict__ r, SplineW<T>& s)
{
  unsigned mult[3];
  mult[2] = d.orb_stride_v;
  mult[1] = mult[2] * (unsigned)d.grid[2];
  mult[0] = mult[1] * (unsigned)d.grid[1];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const int Ng = d.grid[c];
    const double ih = d.inv_h[c];
    const double u = r[c] * ih;
    const double fl = floor(u);
    const double t = u - fl;
    const double t2 = t * t, t3 = t2 * t, omt = 1.0 - t;
    s.w[c][0] = (T)(omt * omt * omt / 6.0);
    s.w[c][1] = (T)((3.0 * t3 - 6.0 * t2 + 4.0) / 6.0);
    s.w[c][2] = (T)((-3.0 * t3 + 3.0 * t2 + 3.0 * t + 1.0) / 6.0);
    s.w[c][3] = (T)(t3 / 6.0);
    s.dw[c][0] = (T)(-omt * omt / 2.0 * ih);
    s.dw[c][1] = (T)((3.0 * t2 - 4.0 * t) / 2.0 * ih);
    s.dw[c][2] = (T)((-3.0 * t2 + 2.0 * t + 1.0) / 2.0 * ih);
    s.dw[c][3] = (T)(t2 / 2.0 * ih);
    const double ih2 = ih * ih;
    s.d2w[c][0] = (T)(omt * ih2);
    s.d2w[c][1] = (T)((3.0 * t - 2.0) * ih2);
    s.d2w[c][2] = (T)((1.0 - 3.0 * t) * ih2);
    s.d2w[c][3] = (T)(t * ih2);
    // (i - 1) mod Ng, floor toward -inf (D:A11); exact in fp64 for |i| < 2^50
    const double a = fl - 1.0;
    const double q = floor(a / (double)Ng);
    int i0 = (int)(a - q * (double)Ng);
    if (i0 < 0) i0 += Ng;
    if (i0 >= Ng) i0 -= Ng;
    if (i0 < 0 || i0 >= Ng) i0 = 0;  // non-finite position: stay in bounds, the weights are NaN anyway
#pragma unroll
    for (int m = 0; m < 4; ++m) {
      int g = i0 + m;
      while (g >= Ng) g -= Ng;
      s.off[c][m] = (unsigned)g * mult[c];
    }
  }
}

// One 16-byte orbital slice `chunk` (in vectors) of all five quantities.
// out[0] = phi, out[1..3] = d/dx, d/dy, d/dz, out[4] = laplacian.
template <typename T>
__device__ __forceinline__ void spline_eval(const T* __restrict__ tab, const SplineW<T>& s, unsigned chunk,
                                            T (&out)[5][Vec16<T>::W])
{
  constexpr int VW = Vec16<T>::W;
#pragma unroll
  for (int q = 0; q < 5; ++q)
#pragma unroll
    for (int e = 0; e < VW; ++e) out[q][e] = (T)0;
#pragma unroll
  for (int a = 0; a < 4; ++a) {
    T u00[VW], u10[VW], u20[VW], u01[VW], u02[VW];
#pragma unroll
    for (int e = 0; e < VW; ++e) u00[e] = u10[e] = u20[e] = u01[e] = u02[e] = (T)0;
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      const unsigned base = s.off[0][a] + s.off[1][b] + chunk;
      T p[4][VW];
#pragma unroll
      for (int c = 0; c < 4; ++c) ld16(tab + (size_t)(base + s.off[2][c]) * VW, p[c]);
#pragma unroll
      for (int e = 0; e < VW; ++e) {
        T v0 = s.w[2][0] * p[0][e], v1 = s.dw[2][0] * p[0][e], v2 = s.d2w[2][0] * p[0][e];
#pragma unroll
        for (int c = 1; c < 4; ++c) {
          v0 = fma(s.w[2][c], p[c][e], v0);
          v1 = fma(s.dw[2][c], p[c][e], v1);
          v2 = fma(s.d2w[2][c], p[c][e], v2);
        }
        u00[e] = fma(s.w[1][b], v0, u00[e]);
        u10[e] = fma(s.dw[1][b], v0, u10[e]);
        u20[e] = fma(s.d2w[1][b], v0, u20[e]);
        u01[e] = fma(s.w[1][b], v1, u01[e]);
        u02[e] = fma(s.w[1][b], v2, u02[e]);
      }
    }
#pragma unroll
    for (int e = 0; e < VW; ++e) {
      out[0][e] = fma(s.w[0][a], u00[e], out[0][e]);
      out[1][e] = fma(s.dw[0][a], u00[e], out[1][e]);
      out[2][e] = fma(s.w[0][a], u10[e], out[2][e]);
      out[3][e] = fma(s.w[0][a], u01[e], out[3][e]);
      out[4][e] = fma(s.d2w[0][a], u00[e], out[4][e]);
      out[4][e] = fma(s.w[0][a], u20[e] + u02[e], out[4][e]);
    }
  }
}

constexpr int SPLINE_NT = 128;

// qmc_spo_vgl step (c): one thread per (walker, 16-byte orbital slice) at r' = d.rnew[w].
template <typename T>
__global__ void __launch_bounds__(SPLINE_NT) spline_vgl_kernel(CrowdDev d)
{
  constexpr int VW = Vec16<T>::W;
  const unsigned chunks = (unsigned)d.ns / VW;
  const unsigned item = blockIdx.x * SPLINE_NT + threadIdx.x;
  const unsigned w = item / chunks, chunk = item - w * chunks;
  if (w >= (unsigned)d.W) return;
  T out[5][VW];
  if (chunk < d.tab_vecs) {
    SplineW<T> s;
    spline_setup<T>(d, d.rnew + 3 * (size_t)w, s);
    spline_eval<T>(static_cast<const T*>(d.coefs), s, chunk, out);
#pragma unroll
    for (int e = 0; e < VW; ++e)
      if ((int)(chunk * VW) + e >= d.M) {
#pragma unroll
        for (int q = 0; q < 5; ++q) out[q][e] = (T)0;
      }
  } else {
#pragma unroll
    for (int q = 0; q < 5; ++q)
#pragma unroll
      for (int e = 0; e < VW; ++e) out[q][e] = (T)0;
  }
  T* vgl = static_cast<T*>(d.vgl) + (size_t)w * 5 * d.ns + (size_t)chunk * VW;
#pragma unroll
  for (int q = 0; q < 5; ++q) st16(vgl + (size_t)q * d.ns, out[q]);
}

// qmc_crowd_create / set_positions: one thread per (walker, electron, slice) at the electron's
// own position; fills the caches and the transposed Slater matrix X[j][i] = phi_j(r_i) that the
// inversion kernel turns into B = (A^-1)^T = (A^T)^-1 (D:C2).
template <typename T>
__global__ void __launch_bounds__(SPLINE_NT) spline_build_kernel(CrowdDev d)
{
  constexpr int VW = Vec16<T>::W;
  const unsigned chunks = (unsigned)d.ns / VW;
  const size_t item = (size_t)blockIdx.x * SPLINE_NT + threadIdx.x;
  const size_t we = item / chunks;
  const unsigned chunk = (unsigned)(item - we * chunks);
  if (we >= (size_t)d.W * d.N) return;
  const int w = (int)(we / d.N), e_idx = (int)(we - (size_t)w * d.N);
  T out[5][VW];
#pragma unroll
  for (int q = 0; q < 5; ++q)
#pragma unroll
    for (int e = 0; e < VW; ++e) out[q][e] = (T)0;
  if (chunk < d.tab_vecs) {
    SplineW<T> s;
    spline_setup<T>(d, d.R + 3 * we, s);
    spline_eval<T>(static_cast<const T*>(d.coefs), s, chunk, out);
  }
  const int spin = e_idx / d.n, i = e_idx - spin * d.n;
  T* cache = static_cast<T*>(d.cache) + we * 4 * d.ns + (size_t)chunk * VW;
  double* X = d.Binv + ((size_t)w * 2 + spin) * d.ns * d.ns;
#pragma unroll
  for (int e = 0; e < VW; ++e) {
    const int j = (int)(chunk * VW) + e;
    if (j >= d.M) {
#pragma unroll
      for (int q = 0; q < 5; ++q) out[q][e] = (T)0;
    } else {
      X[(size_t)j * d.ns + i] = (double)out[0][e];
    }
  }
#pragma unroll
  for (int q = 0; q < 4; ++q) st16(cache + (size_t)q * d.ns, out[q + 1]);
}

}  // namespace qmc
