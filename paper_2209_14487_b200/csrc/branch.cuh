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

// 16-byte streaming copy of nvec vectors, strided over the grid's x dimension, four loads in flight per thread
__device__ __forceinline__ void stream_copy16(double* dp, const double* sp, size_t nvec, unsigned long long pol)
{
  const size_t stride = (size_t)gridDim.x * BRANCH_NT;
  size_t i = (size_t)blockIdx.x * BRANCH_NT + threadIdx.x;
  for (; i + 3 * stride < nvec; i += 4 * stride) {
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
  for (; i < nvec; i += stride) {
    double v[2];
    ld16_stream(sp + 2 * i, v, pol);
    st16(dp + 2 * i, v);
  }
}

// The carried state of one walker as three byte ranges (all multiples of 16 bytes: ns, N are even).
struct WalkerState {
  size_t inv_bytes, cache_bytes, pos_bytes;
  __host__ __device__ size_t total() const { return inv_bytes + cache_bytes + pos_bytes; }
};
__host__ __device__ inline WalkerState walker_state(const CrowdDev& d, size_t elem)
{
  // the carried inverses in their storage type (fp64, or fp32 in the mixed-precision mode D:R6)
  return WalkerState{(size_t)2 * d.ns * d.ns * (d.Binv32 ? 4 : 8), (size_t)d.N * 4 * d.ns * elem, (size_t)d.N * 3 * 8};
}

// grid = (chunks, W): CTA (c, w) copies its share of the three state arrays of walker src[w] into walker w
__global__ void __launch_bounds__(BRANCH_NT) branch_copy_kernel(CrowdDev d, const int* __restrict__ src, WalkerState ws)
{
  const int w = blockIdx.y, s = src[w];
  if (s == w) return;
  const unsigned long long pol = l2_evict_first_policy();
  double* inv = d.Binv32 ? reinterpret_cast<double*>(d.Binv32) : d.Binv;
  stream_copy16(inv + (size_t)w * (ws.inv_bytes / 8), inv + (size_t)s * (ws.inv_bytes / 8), ws.inv_bytes / 16, pol);
  stream_copy16(reinterpret_cast<double*>(static_cast<char*>(d.cache) + (size_t)w * ws.cache_bytes),
                reinterpret_cast<const double*>(static_cast<const char*>(d.cache) + (size_t)s * ws.cache_bytes),
                ws.cache_bytes / 16, pol);
  stream_copy16(d.R + (size_t)w * (ws.pos_bytes / 8), d.R + (size_t)s * (ws.pos_bytes / 8), ws.pos_bytes / 16, pol);
}

// Walker states to / from a packed buffer (the message of the DMC load balance, Alg. 1 L14):
// buf[i] = [inverses | caches | positions] of walker slots[i] (EXPORT) or the reverse (IMPORT).  grid = (chunks, n).
template <bool EXPORT>
__global__ void __launch_bounds__(BRANCH_NT) walker_pack_kernel(CrowdDev d, const int* __restrict__ slots, char* buf,
                                                                WalkerState ws)
{
  const int i = blockIdx.y, w = slots[i];
  const unsigned long long pol = l2_evict_first_policy();
  double* b_inv = reinterpret_cast<double*>(buf + (size_t)i * ws.total());
  double* b_cache = reinterpret_cast<double*>(buf + (size_t)i * ws.total() + ws.inv_bytes);
  double* b_pos = reinterpret_cast<double*>(buf + (size_t)i * ws.total() + ws.inv_bytes + ws.cache_bytes);
  double* w_inv = (d.Binv32 ? reinterpret_cast<double*>(d.Binv32) : d.Binv) + (size_t)w * (ws.inv_bytes / 8);
  double* w_cache = reinterpret_cast<double*>(static_cast<char*>(d.cache) + (size_t)w * ws.cache_bytes);
  double* w_pos = d.R + (size_t)w * (ws.pos_bytes / 8);
  if (EXPORT) {
    stream_copy16(b_inv, w_inv, ws.inv_bytes / 16, pol);
    stream_copy16(b_cache, w_cache, ws.cache_bytes / 16, pol);
    stream_copy16(b_pos, w_pos, ws.pos_bytes / 16, pol);
  } else {
    stream_copy16(w_inv, b_inv, ws.inv_bytes / 16, pol);
    stream_copy16(w_cache, b_cache, ws.cache_bytes / 16, pol);
    stream_copy16(w_pos, b_pos, ws.pos_bytes / 16, pol);
  }
}

// status |= 8 for a slot outside [0, W) or listed twice (marks: W zeroed ints, left dirty -- the caller clears them)
__global__ void slots_check_kernel(CrowdDev d, int n, const int* __restrict__ slots, int* marks)
{
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int w = slots[i];
  if (w < 0 || w >= d.W) { atomicOr(d.status, 8); return; }
  if (atomicAdd(marks + w, 1) != 0) atomicOr(d.status, 8);
}

// CTAs per walker of the state copies: about 32 16-byte vectors per thread
inline int state_chunks(const WalkerState& ws)
{
  const size_t vecs = ws.total() / 16;
  int chunks = (int)((vecs + (size_t)BRANCH_NT * 32 - 1) / ((size_t)BRANCH_NT * 32));
  return chunks < 1 ? 1 : (chunks > 64 ? 64 : chunks);
}

// *out += number of slots with src[w] != w
__global__ void branch_count_kernel(int W, const int* __restrict__ src, int* out)
{
  const int w = blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned b = __ballot_sync(0xffffffffu, w < W && src[w] != w);
  if ((threadIdx.x & 31) == 0 && b) atomicAdd(out, __popc(b));
}

}  // namespace qmc
