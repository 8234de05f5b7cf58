// branch.cuh -- the data movement of DMC branching inside one crowd (Alg. 1 L13 "branch",
// PAPER.md:63, and the 2.4 MB-per-walker states P:66 moves between ranks): walker slot w takes over the complete
// carried state of slot src[w] -- positions, both inverses, the gradient / Laplacian caches -- so that a killed
// walker's slot continues as a copy of a surviving one.  The weights that decide src come from the local energy and
// the population control (Alg. 1 L11-L13), which stay outside the hot path; src is an input.
//
// In place and race-free by contract: every source must be a slot that keeps its own state (src[src[w]] == src[w]),
// checked on the device before anything is written.  Pure streaming copy: 16-byte vectors, sources read once with the
// L2 evict-first policy, bound by HBM (2 x state bytes per copied walker).
#pragma once
#include "common.cuh"

namespace qmc {

constexpr int BRANCH_NT = 256;

// status |= 8 when src is not a valid branching map
__global__ void branch_check_kernel(CrowdDev d, const int* __restrict__ src)
{
  const int w = blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= d.W) return;
  const int s = src[w];
  if (s < 0 || s >= d.W || src[s] != s) atomicOr(d.status, 8);
}

// grid = (chunks, W): CTA (c, w) copies its share of the three state arrays of walker src[w] into walker w
__global__ void __launch_bounds__(BRANCH_NT) branch_copy_kernel(CrowdDev d, const int* __restrict__ src,
                                                                size_t cache_bytes_per_walker)
{
  const int w = blockIdx.y, s = src[w];
  if (s == w) return;
  const unsigned long long pol = l2_evict_first_policy();
  const size_t n_inv = (size_t)2 * d.ns * d.ns / 2;          // 16-byte vectors of the two inverses
  const size_t n_cache = cache_bytes_per_walker / 16;
  const size_t n_pos = ((size_t)d.N * 3) / 2;                // N is even: 3 N doubles = 3 N / 2 vectors
  const size_t tid = (size_t)blockIdx.x * BRANCH_NT + threadIdx.x, stride = (size_t)gridDim.x * BRANCH_NT;
  {
    const double* sp = d.Binv + (size_t)s * n_inv * 2;
    double* dp = d.Binv + (size_t)w * n_inv * 2;
    size_t i = tid;
    for (; i + 3 * stride < n_inv; i += 4 * stride) {  // four independent 16-byte loads in flight per thread
      double v0[2], v1[2], v2[2], v3[2];
      ld16_stream(sp + 2 * i, v0, pol);
      ld16_stream(sp + 2 * (i + stride), v1, pol);
      ld16_stream(sp + 2 * (i + 2 * stride), v2, pol);
      ld16_stream(sp + 2 * (i + 3 * stride), v3, pol);
      st16(dp + 2 * i, v0);
      st16(dp + 2 * (i + stride), v1);
      st16(dp + 2 * (i + 2 * stride), v2);
      st16(dp + 2 * (i + 3 * stride), v3);
    }
    for (; i < n_inv; i += stride) {
      double v[2];
      ld16_stream(sp + 2 * i, v, pol);
      st16(dp + 2 * i, v);
    }
  }
  {
    const double* sp = reinterpret_cast<const double*>(static_cast<const char*>(d.cache) + (size_t)s * cache_bytes_per_walker);
    double* dp = reinterpret_cast<double*>(static_cast<char*>(d.cache) + (size_t)w * cache_bytes_per_walker);
    size_t i = tid;
    for (; i + 3 * stride < n_cache; i += 4 * stride) {
      double v0[2], v1[2], v2[2], v3[2];
      ld16_stream(sp + 2 * i, v0, pol);
      ld16_stream(sp + 2 * (i + stride), v1, pol);
      ld16_stream(sp + 2 * (i + 2 * stride), v2, pol);
      ld16_stream(sp + 2 * (i + 3 * stride), v3, pol);
      st16(dp + 2 * i, v0);
      st16(dp + 2 * (i + stride), v1);
      st16(dp + 2 * (i + 2 * stride), v2);
      st16(dp + 2 * (i + 3 * stride), v3);
    }
    for (; i < n_cache; i += stride) {
      double v[2];
      ld16_stream(sp + 2 * i, v, pol);
      st16(dp + 2 * i, v);
    }
  }
  {
    const double* sp = d.R + (size_t)s * d.N * 3;
    double* dp = d.R + (size_t)w * d.N * 3;
    for (size_t i = tid; i < n_pos; i += stride) {
      double v[2];
      ld16_stream(sp + 2 * i, v, pol);
      st16(dp + 2 * i, v);
    }
  }
}

}  // namespace qmc
