// qmc_crowd.cu -- host side of libqmc_crowd.so: the C ABI of include/qmc_crowd.h.
// Argument checking, workspace carving, kernel launches and the lock-step sweep schedule
// (Alg. 3; flush schedule D:C6).  Every step of the path runs in the kernels of
// spline.cuh / move.cuh / update.cuh / invert.cuh; there is no CPU fallback.
#include "../../include/qmc_crowd.h"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "common.cuh"
#include "invert.cuh"
#include "move.cuh"
#include "spline.cuh"
#include "energy.cuh"
#include "update.cuh"
#include "window.cuh"
#include "branch.cuh"

using namespace qmc;

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char* fmt, ...)
{
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return code;
}

#define CUDA_TRY(expr)                                                                              \
  do {                                                                                              \
    cudaError_t e_ = (expr);                                                                        \
    if (e_ != cudaSuccess) return fail(QMC_ERR_CUDA, "%s: %s (%s:%d)", #expr, cudaGetErrorString(e_), __FILE__, __LINE__); \
  } while (0)

#define LAUNCH_CHECK(c)                                                                             \
  do {                                                                                              \
    ++(c)->launches;                                                                                \
    cudaError_t e_ = cudaGetLastError();                                                            \
    if (e_ != cudaSuccess) return fail(QMC_ERR_CUDA, "kernel launch: %s (%s:%d)", cudaGetErrorString(e_), __FILE__, __LINE__); \
  } while (0)

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct ProfScope;

enum StepState { ST_IDLE = 0, ST_HAVE_VGL = 1, ST_HAVE_RATIO = 2 };

}  // namespace

struct qmc_crowd {
  qmc_crowd_desc desc;
  CrowdDev dev;
  cudaStream_t stream;
  int is_f64;
  size_t elem;             // sizeof(table element)
  int state, state_k;
  int win_spin;            // spin block of the open window, -1 if none
  std::vector<int> win_rows;  // electrons (within the spin block) proposed since the last flush
  uint64_t proposed, flushes, launches;
  uint32_t sweep_host;
  int use_graph;
  int n_sub;                        // sub-crowds of qmc_sweep (delay_rank > 1), each on its own stream; 0 = automatic
  int strip_rows;                   // QMC_OPT_STRIP_ROWS: 0 = automatic, 16 / 32 = forced
  int smem_optin;                   // cudaDevAttrMaxSharedMemoryPerBlockOptin of the device
  int recompute_every;              // qmc_sweep recomputes the inverses every this many sweeps (0 = never)
  int n_sm;                         // SMs of the device (sizes the automatic sub-crowd choice)
  cudaStream_t sub_stream[4];
  cudaEvent_t ev_fork, ev_join[4];
  uint64_t graph_launches, graph_flushes;  // per replay of the captured sweep
  cudaGraphExec_t graph_exec;
  // QMC_OPT_PROFILE: CUDA-event pairs around every kernel of the plain-launch sweep
  int profile;
  std::vector<cudaEvent_t> ev;      // pool, pairs (begin, end)
  std::vector<int> ev_class;        // kernel class of pair i
  size_t ev_used;                   // pairs recorded since the last qmc_crowd_get_profile
  double prof_ms[QMC_N_KERNEL_CLASSES];
  uint64_t prof_cnt[QMC_N_KERNEL_CLASSES];
};

namespace {

// Records an event pair around the launches issued while it is alive (profile mode only).
struct ProfScope {
  qmc_crowd* c;
  size_t idx;
  bool on;
  ProfScope(qmc_crowd* c_, int cls) : c(c_), idx(0), on(c_->profile != 0)
  {
    if (!on) return;
    if (c->ev_used * 2 + 2 > c->ev.size()) {
      cudaEvent_t a = nullptr, b = nullptr;
      if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) { on = false; return; }
      c->ev.push_back(a);
      c->ev.push_back(b);
      c->ev_class.push_back(cls);
    }
    idx = c->ev_used++;
    c->ev_class[idx] = cls;
    cudaEventRecord(c->ev[2 * idx], c->stream);
  }
  ~ProfScope()
  {
    if (on) cudaEventRecord(c->ev[2 * idx + 1], c->stream);
  }
};

int padded_rank(int kd)
{
  int p = 8;
  while (p < kd) p *= 2;
  return p;
}

// Carves the workspace; with base == nullptr only measures. Returns total bytes.
size_t carve(const qmc_crowd_desc* ds, CrowdDev* d, char* base)
{
  const size_t W = (size_t)ds->n_walkers, N = (size_t)ds->n_elec, n = N / 2;
  const size_t ns = align_up(n, 16);
  const size_t kdp = (size_t)padded_rank(ds->delay_rank);
  const size_t el = ds->coef_dtype ? 8 : 4;
  size_t off = 0;
  auto take = [&](size_t bytes) {
    char* p = base ? base + off : nullptr;
    off = align_up(off + bytes, 256);
    return p;
  };
  char* R = take(W * N * 3 * 8);
  char* Binv = take(W * 2 * ns * ns * 8);
  char* Binv32 = ds->inverse_dtype ? take(W * 2 * ns * ns * 4) : nullptr;
  char* cache = take(W * N * 4 * ns * el);
  char* vgl = take(W * 5 * ns * el);
  char* brow = take(W * ns * 8);
  char* rnew = take(W * 3 * 8);
  char* delta = take(W * 3 * 8);
  char* g_old = take(W * 3 * 8);
  char* g_new = take(W * 3 * 8);
  char* usum_old = take(W * 8);
  char* rho_d = take(W * 8);
  char* rho_j = take(W * 8);
  char* p = take(W * 8);
  char* u = take(W * 8);
  char* accepted = take(W);
  char* acc_sink = take(W);
  char* V = take(ds->delay_rank > 1 ? W * kdp * ns * 8 : 8);
  char* C = take(ds->delay_rank > 1 ? W * kdp * ns * 8 : 8);
  char* Cp = take(ds->delay_rank > 1 ? W * kdp * ns * 8 : 8);
  char* Sinv = take(ds->delay_rank > 1 ? W * kdp * kdp * 8 : 8);
  char* pvec = take(W * kdp * 8);
  char* yvec = take(W * kdp * 8);
  char* rows = take(W * kdp * 4);
  char* mwin = take(W * 4);
  char* e_elec = take(W * N * 8);
  char* counters = take(4 * 8);
  char* sweep = take(4);
  char* status = take(4);
  const size_t cells = (size_t)ds->grid[0] * ds->grid[1] * ds->grid[2];
  char* cell_bins = cells <= ((size_t)1 << 22) ? take((cells + 1) * 4) : nullptr;   // Slater build in grid-cell order
  if (d) {
    d->R = (double*)R; d->Binv = (double*)Binv; d->Binv32 = (float*)Binv32; d->cache = cache; d->vgl = vgl; d->brow = (double*)brow;
    d->rnew = (double*)rnew; d->delta = (double*)delta; d->g_old = (double*)g_old; d->g_new = (double*)g_new;
    d->usum_old = (double*)usum_old; d->rho_d = (double*)rho_d; d->rho_j = (double*)rho_j;
    d->p = (double*)p; d->u = (double*)u; d->accepted = (unsigned char*)accepted;
    d->V = (double*)V; d->C = (double*)C; d->Cp = (double*)Cp; d->Sinv = (double*)Sinv; d->pvec = (double*)pvec; d->yvec = (double*)yvec;
    d->e_elec = (double*)e_elec;
    d->cell_bins = (cells <= ((size_t)1 << 22)) ? (int*)cell_bins : nullptr;
    d->rows = (int*)rows; d->mwin = (int*)mwin; d->counters = (unsigned long long*)counters;
    d->sweep = (unsigned*)sweep; d->status = (int*)status;
    (void)acc_sink;
  }
  return off;
}

int check_desc(const qmc_crowd_desc* ds)
{
  if (!ds) return fail(QMC_ERR_INVALID_ARG, "desc is NULL");
  if (ds->n_elec < 2 || (ds->n_elec & 1)) return fail(QMC_ERR_INVALID_ARG, "n_elec must be even and >= 2");
  if (ds->n_orb != ds->n_elec / 2) return fail(QMC_ERR_INVALID_ARG, "n_orb must equal n_elec/2");
  if (ds->n_walkers < 1) return fail(QMC_ERR_INVALID_ARG, "n_walkers must be >= 1");
  // several kernels put W (or 2 W) in gridDim.y, which CUDA limits to 65535
  if (ds->n_walkers > 32767) return fail(QMC_ERR_INVALID_ARG, "n_walkers must be <= 32767 per crowd (split the population into crowds)");
  if (ds->coef_dtype != 0 && ds->coef_dtype != 1) return fail(QMC_ERR_INVALID_ARG, "coef_dtype must be 0 or 1");
  if (ds->delay_rank < 1 || ds->delay_rank > 64) return fail(QMC_ERR_INVALID_ARG, "delay_rank must be in [1,64]");
  if (ds->inverse_dtype != 0 && ds->inverse_dtype != 1) return fail(QMC_ERR_INVALID_ARG, "inverse_dtype must be 0 (fp64) or 1 (fp32 storage)");
  if (ds->inverse_dtype == 1 && ds->delay_rank > 32)
    return fail(QMC_ERR_INVALID_ARG, "fp32-stored inverses need delay_rank <= 32 (one flush pass = one rounding)");
  const int vw = ds->coef_dtype ? 2 : 4;
  if (ds->orb_stride < ds->n_orb || ds->orb_stride % vw) return fail(QMC_ERR_INVALID_ARG, "orb_stride must be >= n_orb and a multiple of %d", vw);
  double tab = (double)ds->orb_stride / vw;
  for (int c = 0; c < 3; ++c) {
    if (ds->grid[c] < 1) return fail(QMC_ERR_INVALID_ARG, "grid must be >= 1");
    if (!(ds->box[c] > 0.0) || !std::isfinite(ds->box[c])) return fail(QMC_ERR_INVALID_ARG, "box must be positive");
    tab *= ds->grid[c];
  }
  if (tab >= 4294967296.0) return fail(QMC_ERR_INVALID_ARG, "coefficient table larger than 2^32 16-byte vectors");
  if (!(ds->tau > 0.0) || !std::isfinite(ds->tau)) return fail(QMC_ERR_INVALID_ARG, "tau must be positive");
  return QMC_OK;
}

}  // namespace

// ------------------------------------------------------------------------------------------
// launch helpers (all on c->stream)
// ------------------------------------------------------------------------------------------
namespace {

template <typename T>
int launch_build_t(qmc_crowd* c)
{
  const CrowdDev& d = c->dev;
  const size_t blocks = (size_t)d.W * d.N;
  if (blocks > 0x7fffffffull) return fail(QMC_ERR_INVALID_ARG, "crowd too large for one build launch");
  const size_t smem = (size_t)5 * d.ns * sizeof(T);
  const int* order = nullptr;
#ifndef QMC_BUILD_UNSORTED
  if (d.cell_bins && blocks >= 256) {
    // positions in grid-cell order (counting sort; the order inside a cell is arbitrary and does not matter: every
    // CTA writes only its own electron's outputs).  The order lives in the e_elec scratch (W N doubles).
    const int cells = d.grid[0] * d.grid[1] * d.grid[2];
    int* ord = reinterpret_cast<int*>(d.e_elec);
    CUDA_TRY(cudaMemsetAsync(d.cell_bins, 0, (size_t)(cells + 1) * 4, c->stream));
    cell_count_kernel<<<(unsigned)((blocks + 255) / 256), 256, 0, c->stream>>>(d, d.cell_bins);
    cell_scan_kernel<<<1, 1024, 0, c->stream>>>(d.cell_bins, cells);
    cell_scatter_kernel<<<(unsigned)((blocks + 255) / 256), 256, 0, c->stream>>>(d, d.cell_bins, ord);
    LAUNCH_CHECK(c);
    c->launches += 3;
    order = ord;
  }
#endif
  if (order)
    spline_build_cells_kernel<T><<<(unsigned)(d.grid[0] * d.grid[1] * d.grid[2]), BUILD_NT, BUILD_SMEM, c->stream>>>(d, order, d.cell_bins);
  else spline_build_kernel<T><<<(unsigned)blocks, SPLINE_NT, smem, c->stream>>>(d);
  LAUNCH_CHECK(c);
  if (order) {   // the sorted build writes A row-major: transpose to the A^T the inversion expects
    transpose_inplace_kernel<<<dim3((unsigned)(d.ns / 16), (unsigned)(2 * d.W)), 256, 0, c->stream>>>(d);
    LAUNCH_CHECK(c);
  }
  return QMC_OK;
}

// spline at all electron positions -> caches + A^T; Gauss-Jordan; status check (synchronises)
int rebuild(qmc_crowd* c)
{
  const CrowdDev& d = c->dev;
  CUDA_TRY(cudaMemsetAsync(d.Binv, 0, (size_t)d.W * 2 * d.ns * d.ns * 8, c->stream));
  CUDA_TRY(cudaMemsetAsync(d.mwin, 0, (size_t)d.W * 4, c->stream));
  CUDA_TRY(cudaMemsetAsync(d.status, 0, 4, c->stream));
  c->launches += 3;
  int st = c->is_f64 ? launch_build_t<double>(c) : launch_build_t<float>(c);
  if (st) return st;
  const size_t b2smem = invert_blocked2_smem(d.ns);
  if (b2smem <= 227 * 1024 && d.ns <= 2 * INVB2_NT) {
    invert_blocked2_kernel<<<(unsigned)(d.W * 2), INVB2_NT, b2smem, c->stream>>>(d);
  } else {
    // matrices too large for the shared-memory panel: the unblocked Gauss-Jordan (same pivots, 2 n sweeps of the matrix)
    const size_t smem = (size_t)(2 * d.ns + 2 * (INV_NT / 32)) * 8 + (size_t)d.ns * 4 + 64;
    invert_kernel<<<(unsigned)(d.W * 2), INV_NT, smem, c->stream>>>(d);
  }
  LAUNCH_CHECK(c);
  if (d.Binv32) {   // D:R6: the fp64 inverse is rounded once into the carried fp32 copy
    const size_t total = (size_t)d.W * 2 * d.ns * d.ns;
    narrow_kernel<<<(unsigned)std::min<size_t>((total / 4 + 255) / 256, 148 * 32), 256, 0, c->stream>>>(d.Binv32, d.Binv, total);
    LAUNCH_CHECK(c);
  }
  int status = 0;
  CUDA_TRY(cudaMemcpyAsync(&status, d.status, 4, cudaMemcpyDeviceToHost, c->stream));
  CUDA_TRY(cudaStreamSynchronize(c->stream));
  c->state = ST_IDLE;
  c->win_spin = -1;
  c->win_rows.clear();
  if (status != 0) return fail(QMC_ERR_SINGULAR, "a Slater matrix has a zero or non-finite pivot");
  return QMC_OK;
}

// dynamic smem of every move kernel: the largest need of the three device functions
size_t move_smem(const CrowdDev& d)
{
  const size_t row = (size_t)d.ns + 2 * d.kdp + MOVE_RED, acc = (size_t)d.ns + 3 * d.kdp + 16;
  return (row > acc ? row : acc) * 8;
}

template <typename T>
int launch_row_propose_t(qmc_crowd* c, int k, const double* rnew)
{
  row_propose_kernel<T><<<c->dev.W, MOVE_NT, move_smem(c->dev), c->stream>>>(c->dev, k, rnew);
  LAUNCH_CHECK(c);
  return QMC_OK;
}

template <typename T>
int launch_spline_t(qmc_crowd* c)
{
  const CrowdDev& d = c->dev;
  spline_vgl_kernel<T><<<(unsigned)d.W, SPLINE_NT, 0, c->stream>>>(d);
  LAUNCH_CHECK(c);
  return QMC_OK;
}

template <typename T>
int launch_ratio_t(qmc_crowd* c, int k, double* ratio, double* grad)
{
  ratio_grad_kernel<T><<<c->dev.W, MOVE_NT, move_smem(c->dev), c->stream>>>(c->dev, k, ratio, grad);
  LAUNCH_CHECK(c);
  return QMC_OK;
}

template <typename T>
int launch_rank1_t(qmc_crowd* c, int k)
{
  const CrowdDev& d = c->dev;
  const int rows_per_cta = (RANK1_NT / 32) * RANK1_ROWS_PER_WARP;
  dim3 grid((d.n + rows_per_cta - 1) / rows_per_cta, d.W);
  const int nv = (d.ns + 63) / 64;
  if (d.Binv32) {
    rank1_f32_kernel<T><<<grid, RANK1_NT, 0, c->stream>>>(d, k);
    LAUNCH_CHECK(c);
    return QMC_OK;
  }
  switch (nv) {
    case 1: rank1_kernel<T, 1><<<grid, RANK1_NT, 0, c->stream>>>(d, k); break;
    case 2: rank1_kernel<T, 2><<<grid, RANK1_NT, 0, c->stream>>>(d, k); break;
    case 3: rank1_kernel<T, 3><<<grid, RANK1_NT, 0, c->stream>>>(d, k); break;
    case 4: rank1_kernel<T, 4><<<grid, RANK1_NT, 0, c->stream>>>(d, k); break;
    case 5: case 6: rank1_kernel<T, 6><<<grid, RANK1_NT, 0, c->stream>>>(d, k); break;
    case 7: case 8: rank1_kernel<T, 8><<<grid, RANK1_NT, 0, c->stream>>>(d, k); break;
    default: rank1_generic_kernel<T><<<grid, RANK1_NT, 0, c->stream>>>(d, k); break;
  }
  LAUNCH_CHECK(c);
  return QMC_OK;
}

template <typename T>
int launch_accept_t(qmc_crowd* c, int k, unsigned char* acc_out)
{
  {
    ProfScope ps(c, QMC_K_ACCEPT);
    accept_kernel<T><<<c->dev.W, MOVE_NT, move_smem(c->dev), c->stream>>>(c->dev, k, acc_out);
    LAUNCH_CHECK(c);
  }
  if (c->dev.kd == 1) {
    ProfScope ps(c, QMC_K_RANK1);
    return launch_rank1_t<T>(c, k);
  }
  return QMC_OK;
}

// The strip kernel of a flush (section L0 of the window, -1 = all of it): 32-row strips where the shape allows them
template <int KB, int L0, typename TB>
void launch_strip(const CrowdDev& d, int spin, int wn, cudaStream_t st, int strip_rows)
{
  // (fp32-stored inverses keep the 16-row kernel: with the conversions next to 254 registers the 32-row form was slower,
  // 3.70 against 3.5 ms per flush at cfg 5, W = 4096)
  if constexpr (KB >= 2 && sizeof(TB) == 8) {
    // small crowds keep 16-row strips: below ~2 waves of 32-row strip warps (8 per SM) the shorter chains of twice as many
    // warps win (cfg 5, k = 32: W = 64 +1.4 %, W = 128 +4 %; from W = 256 on the 32-row kernel is faster)
    const bool want32 = strip_rows ? strip_rows == 32 : (size_t)wn * (d.ns / 32) >= 2368;
    if (d.ns % 32 == 0 && want32) {
      const int nt = (d.ns / 32) % (FLUSH32_NT / 32) == 0 ? FLUSH32_NT : 32;
      dim3 grid32((d.ns + nt - 1) / nt, wn);
      flush32_kernel<KB, L0, TB><<<grid32, nt, 0, st>>>(d, spin);
      return;
    }
  }
  const int rows_per_cta = (FLUSH_NT / 32) * FLUSH_ROWS_PER_WARP;
  dim3 grid((d.ns + rows_per_cta - 1) / rows_per_cta, wn);
  flush_kernel<KB, L0, TB><<<grid, FLUSH_NT, 0, st>>>(d, spin);
}

template <int KDP>
void launch_flush_kdp(const CrowdDev& d, int spin, bool from_window, int wn, cudaStream_t st, int strip_rows)
{
  if (from_window && KDP > 32) {
    // Two sections of 32 moves, each a complete flush applied to the result of the one before: the sequential
    // Sherman-Morrison updates B_{l+1} = B_l - (B_l phi_l - e_l) c_l^T compose section by section (c_l is the current
    // row over rho_l, whatever came before), and a section's Z solves only its own triangular block.  The strip kernel
    // with four window blocks keeps its double-buffered operands in registers (eight spill or lose the double
    // buffer): 11.1 -> 7.7 ms per flush of 64 moves at cfg 5, W = 4096.
    flush_finalize_tri_kernel<32><<<wn, FINTRI_NT, (size_t)(1 + FINTRI_NT / 32) * 32 * 33 * 8, st>>>(d, 0);
    launch_strip<4, 0, double>(d, spin, wn, st, strip_rows);
    flush_finalize_tri_kernel<32><<<wn, FINTRI_NT, (size_t)(1 + FINTRI_NT / 32) * 32 * 33 * 8, st>>>(d, 32);
    launch_strip<4, 32, double>(d, spin, wn, st, strip_rows);
    return;
  }
  if (from_window) {
    if constexpr (KDP <= 32) flush_finalize_tri_kernel<KDP><<<wn, FINTRI_NT, (size_t)(1 + FINTRI_NT / 32) * KDP * (KDP + 1) * 8, st>>>(d, 0);
  } else {
    const int fcols = FINALIZE_NT / (KDP > 32 ? KDP / 32 : 1);
    dim3 fgrid((d.ns + fcols - 1) / fcols, wn);
    flush_finalize_kernel<KDP><<<fgrid, FINALIZE_NT, (size_t)KDP * KDP * 8, st>>>(d, spin);
  }
  if constexpr (KDP <= 32) {
    if (d.Binv32) {   // D:R6, delay_rank <= 32: one pass, one rounding
      launch_strip<KDP / 8, -1, float>(d, spin, wn, st, strip_rows);
      return;
    }
  }
  if constexpr (KDP <= 32) launch_strip<KDP / 8, -1, double>(d, spin, wn, st, strip_rows);
  else flush_kernel<KDP / 8><<<dim3((d.ns + (FLUSH_NT / 32) * FLUSH_ROWS_PER_WARP - 1) / ((FLUSH_NT / 32) * FLUSH_ROWS_PER_WARP), wn), FLUSH_NT, 0, st>>>(d, spin);
}

// Flush of walkers [w0, w0 + wn) on stream st (the whole crowd on the crowd's stream by default).
int launch_flush(qmc_crowd* c, int spin, bool from_window = false, int w0 = 0, int wn = -1, cudaStream_t st = nullptr)
{
  CrowdDev d = c->dev;
  if (wn < 0) { wn = d.W; st = c->stream; }
  d.w0 = w0;
  ProfScope ps(c, QMC_K_FLUSH);
  switch (d.kdp) {
    case 8: launch_flush_kdp<8>(d, spin, from_window, wn, st, c->strip_rows); break;
    case 16: launch_flush_kdp<16>(d, spin, from_window, wn, st, c->strip_rows); break;
    case 32: launch_flush_kdp<32>(d, spin, from_window, wn, st, c->strip_rows); break;
    case 64: launch_flush_kdp<64>(d, spin, from_window, wn, st, c->strip_rows); break;
    default: return fail(QMC_ERR_INVALID_ARG, "unsupported padded delay rank %d", d.kdp);
  }
  ++c->launches;
  LAUNCH_CHECK(c);
  CUDA_TRY(cudaMemsetAsync(d.mwin + w0, 0, (size_t)wn * 4, st));
  ++c->launches;
  if (w0 == 0) ++c->flushes;
  return QMC_OK;
}

// propose + spline for electron k (qmc_spo_vgl without the optional copies)
int step_vgl(qmc_crowd* c, int k, const double* rnew)
{
  int st;
  {
    ProfScope ps(c, QMC_K_ROW_PROPOSE);
    st = c->is_f64 ? launch_row_propose_t<double>(c, k, rnew) : launch_row_propose_t<float>(c, k, rnew);
  }
  if (st) return st;
  ProfScope ps(c, QMC_K_SPLINE_VGL);
  return c->is_f64 ? launch_spline_t<double>(c) : launch_spline_t<float>(c);
}
int step_ratio(qmc_crowd* c, int k, double* ratio, double* grad)
{
  ProfScope ps(c, QMC_K_RATIO_GRAD);
  return c->is_f64 ? launch_ratio_t<double>(c, k, ratio, grad) : launch_ratio_t<float>(c, k, ratio, grad);
}
int step_accept(qmc_crowd* c, int k, unsigned char* acc)
{
  return c->is_f64 ? launch_accept_t<double>(c, k, acc) : launch_accept_t<float>(c, k, acc);
}

template <typename T>
int launch_ratio_accept_t(qmc_crowd* c, int k)
{
  ProfScope ps(c, QMC_K_RATIO_ACCEPT);
  ratio_accept_kernel<T><<<c->dev.W, MOVE_NT, move_smem(c->dev), c->stream>>>(c->dev, k);
  LAUNCH_CHECK(c);
  return QMC_OK;
}

size_t window_smem(const CrowdDev& d, size_t elem, int nt = MOVE_NT) { return (size_t)win_layout(d.N, d.ns, d.kdp, (int)elem, nt).total * 8; }

// Threads per walker of the window kernel: a crowd that leaves SMs idle gets wider CTAs (shorter move chain).
// W = the whole crowd's size (sub-crowds of qmc_sweep keep their crowd's class, so QMC_OPT_SUBCROWDS is bit-invariant).
int window_threads(int wn) { return wn <= 148 ? 512 : (wn <= 296 ? 256 : 128); }

template <typename T>
int launch_window_t(qmc_crowd* c, int k0, int cnt, int w0, int wn, cudaStream_t st)
{
  ProfScope ps(c, QMC_K_WINDOW);
  CrowdDev d = c->dev;
  d.w0 = w0;
  const int nt = window_threads(d.W);
  const size_t smem = window_smem(d, sizeof(T), nt);
  // shape-specialised instances for the BASELINE.json shapes with n a multiple of 16 (cfgs 3, 4, 5): see window.cuh
  const bool shape_ok = sizeof(T) == 4 && d.n == d.ns && d.M == d.n && d.tab_vecs >= (unsigned)d.ns / 4;
  const bool spec = nt == 128 && shape_ok;
  // 512-thread class (one walker per SM): the block rows in shared memory when they fit next to the move's own state
  const size_t smem_sb = smem + (size_t)d.kdp * d.ns * 8;
  const bool sb_ok = smem_sb + 1024 <= (size_t)c->smem_optin;
  if (d.Binv32) {   // mixed precision (D:R6): the block's B0 rows are fp32
    if (spec && d.ns == 384) window_kernel<T, 128, 384, float><<<wn, 128, smem, st>>>(d, k0, cnt);
    else if (nt == 512) window_kernel<T, 512, 0, float><<<wn, 512, smem, st>>>(d, k0, cnt);
    else if (nt == 256) window_kernel<T, 256, 0, float><<<wn, 256, smem, st>>>(d, k0, cnt);
    else window_kernel<T, 128, 0, float><<<wn, 128, smem, st>>>(d, k0, cnt);
  } else if (spec && d.ns == 384) window_kernel<T, 128, 384><<<wn, 128, smem, st>>>(d, k0, cnt);
  else if (spec && d.ns == 192) window_kernel<T, 128, 192><<<wn, 128, smem, st>>>(d, k0, cnt);
  else if (spec && d.ns == 96) window_kernel<T, 128, 96><<<wn, 128, smem, st>>>(d, k0, cnt);
  else if (shape_ok && d.ns == 384 && nt == 256) window_kernel<T, 256, 384><<<wn, 256, smem, st>>>(d, k0, cnt);   // small crowds of cfg 5
  else if (shape_ok && d.ns == 384 && nt == 512 && sb_ok) window_kernel<T, 512, 384, double, true><<<wn, 512, smem_sb, st>>>(d, k0, cnt);
  else if (shape_ok && d.ns == 384 && nt == 512) window_kernel<T, 512, 384><<<wn, 512, smem, st>>>(d, k0, cnt);
  else switch (nt) {   // the class of the WHOLE crowd: a split into sub-crowds never changes a reduction tree
    case 512:
      if (sb_ok) window_kernel<T, 512, 0, double, true><<<wn, 512, smem_sb, st>>>(d, k0, cnt);
      else window_kernel<T, 512><<<wn, 512, smem, st>>>(d, k0, cnt);
      break;
    case 256: window_kernel<T, 256><<<wn, 256, smem, st>>>(d, k0, cnt); break;
    default: window_kernel<T, 128><<<wn, 128, smem, st>>>(d, k0, cnt); break;
  }
  LAUNCH_CHECK(c);
  return QMC_OK;
}

// Dynamic shared memory above 48 KB is an opt-in attribute of each kernel, and it is process-wide: it is raised ONCE
// per device to what the device allows (minus the kernel's static shared memory), never to one crowd's need, so that
// crowds of different shapes in one process cannot lower it under each other's launches.
cudaError_t raise_smem_limit(const void* fn, int optin)
{
  cudaFuncAttributes a;
  cudaError_t e = cudaFuncGetAttributes(&a, fn);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, optin - (int)a.sharedSizeBytes);
}

template <typename T>
cudaError_t raise_smem_limits_t(int optin)
{
  const void* fns[] = {(const void*)row_propose_kernel<T>, (const void*)ratio_grad_kernel<T>, (const void*)accept_kernel<T>,
                       (const void*)ratio_accept_kernel<T>, (const void*)window_kernel<T, 128>,
                       (const void*)window_kernel<T, 128, 384>, (const void*)window_kernel<T, 128, 192>,
                       (const void*)window_kernel<T, 128, 96>, (const void*)window_kernel<T, 256, 384>,
                       (const void*)window_kernel<T, 512, 384>, (const void*)window_kernel<T, 128, 384, float>,
                       (const void*)window_kernel<T, 128, 0, float>, (const void*)window_kernel<T, 256, 0, float>,
                       (const void*)window_kernel<T, 512, 0, float>,
                       (const void*)window_kernel<T, 256>, (const void*)window_kernel<T, 512>,
                       (const void*)window_kernel<T, 512, 384, double, true>, (const void*)window_kernel<T, 512, 0, double, true>,
                       (const void*)sweep1_kernel<T>, (const void*)spline_build_kernel<T>, (const void*)spline_build_cells_kernel<T>,
                       (const void*)kinetic_kernel<T>};
  for (const void* f : fns) {
    cudaError_t e = raise_smem_limit(f, optin);
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

cudaError_t raise_smem_limits()
{
  static bool done[64] = {};
  int dev = 0, optin = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev >= 0 && dev < 64 && done[dev]) return cudaSuccess;
  e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  if (e != cudaSuccess) return e;
  if ((e = raise_smem_limits_t<float>(optin)) != cudaSuccess) return e;
  if ((e = raise_smem_limits_t<double>(optin)) != cudaSuccess) return e;
  if ((e = raise_smem_limit((const void*)invert_blocked2_kernel, optin)) != cudaSuccess) return e;
  if ((e = raise_smem_limit((const void*)invert_kernel, optin)) != cudaSuccess) return e;
  if (dev >= 0 && dev < 64) done[dev] = true;
  return cudaSuccess;
}

// One full sweep with the D:C6 flush schedule; no host synchronisation (capturable).
// delay_rank > 1: per delay window ONE walker-persistent kernel (all moves of the window) + the flush.
// delay_rank = 1: per move spline(k), ratio(k) + accept(k), the rank-1 update, row/proposal of k+1
// (which must see the updated inverse).
int sweep_once(qmc_crowd* c)
{
  const CrowdDev& d = c->dev;
  int st = QMC_OK;
  if (d.kd > 1) {
    // Walkers never interact, so the crowd may advance as independent sub-crowds (the paper's crowds on separate
    // streams, Alg. 4 / P:135): with two of them the DMMA-bound flush of one overlaps the window kernel of the other.
    // Each sub-crowd is in lock-step with itself; results do not depend on the split (same walkers, same counters).
    // Automatic choice (measured): two sub-crowds pay when the crowd is 1-4 waves of window CTAs
    // (4 per SM), where the flush of one half runs under the other half's partial last wave; larger crowds fill the
    // GPU with every kernel and smaller ones must not be shortened further.
    const int slots = 4 * c->n_sm;
    const int want = c->n_sub ? c->n_sub : (d.W > slots && d.W <= 4 * slots ? 2 : 1);
    const int nsub = (want > 1 && !c->profile && d.W >= 2 * want) ? want : 1;
    cudaStream_t s0 = c->stream;
    if (nsub > 1) {
      CUDA_TRY(cudaEventRecord(c->ev_fork, s0));
      for (int i = 1; i < nsub; ++i) CUDA_TRY(cudaStreamWaitEvent(c->sub_stream[i], c->ev_fork, 0));
    }
    for (int i = 0; i < nsub; ++i) {
      const int w0 = (int)((long long)d.W * i / nsub), w1 = (int)((long long)d.W * (i + 1) / nsub);
      cudaStream_t ss = i == 0 ? s0 : c->sub_stream[i];
      for (int spin = 0; spin < 2; ++spin)
        for (int kk0 = 0; kk0 < d.n; kk0 += d.kd) {
          const int cnt = d.n - kk0 < d.kd ? d.n - kk0 : d.kd;
          st = c->is_f64 ? launch_window_t<double>(c, spin * d.n + kk0, cnt, w0, w1 - w0, ss)
                         : launch_window_t<float>(c, spin * d.n + kk0, cnt, w0, w1 - w0, ss);
          if (st) return st;
          st = launch_flush(c, spin, true, w0, w1 - w0, ss);
          if (st) return st;
        }
      if (i > 0) {
        CUDA_TRY(cudaEventRecord(c->ev_join[i], ss));
        CUDA_TRY(cudaStreamWaitEvent(s0, c->ev_join[i], 0));
      }
    }
    bump_sweep_kernel<<<1, 1, 0, c->stream>>>(d.sweep);
    LAUNCH_CHECK(c);
    return QMC_OK;
  }
  if (d.ns <= SWEEP1_MAX_NS && !d.Binv32) {
    // small matrices: the whole sweep in one walker-persistent launch (window.cuh, sweep1_kernel)
    ProfScope ps(c, QMC_K_WINDOW);
    if (c->is_f64) sweep1_kernel<double><<<d.W, MOVE_NT, window_smem(d, 8), c->stream>>>(d);
    else sweep1_kernel<float><<<d.W, MOVE_NT, window_smem(d, 4), c->stream>>>(d);
    LAUNCH_CHECK(c);
    bump_sweep_kernel<<<1, 1, 0, c->stream>>>(d.sweep);
    LAUNCH_CHECK(c);
    return QMC_OK;
  }
  {
    ProfScope ps(c, QMC_K_ROW_PROPOSE);
    st = c->is_f64 ? launch_row_propose_t<double>(c, 0, nullptr) : launch_row_propose_t<float>(c, 0, nullptr);
  }
  if (st) return st;
  for (int k = 0; k < d.N; ++k) {
    {
      ProfScope ps(c, QMC_K_SPLINE_VGL);
      st = c->is_f64 ? launch_spline_t<double>(c) : launch_spline_t<float>(c);
    }
    if (st) return st;
    st = c->is_f64 ? launch_ratio_accept_t<double>(c, k) : launch_ratio_accept_t<float>(c, k);
    if (st) return st;
    {
      ProfScope ps(c, QMC_K_RANK1);
      st = c->is_f64 ? launch_rank1_t<double>(c, k) : launch_rank1_t<float>(c, k);
      if (st) return st;
    }
    if (k + 1 < d.N) {
      ProfScope ps(c, QMC_K_ROW_PROPOSE);
      st = c->is_f64 ? launch_row_propose_t<double>(c, k + 1, nullptr) : launch_row_propose_t<float>(c, k + 1, nullptr);
      if (st) return st;
    }
  }
  bump_sweep_kernel<<<1, 1, 0, c->stream>>>(d.sweep);
  LAUNCH_CHECK(c);
  return QMC_OK;
}

template <typename TD, typename TS>
int launch_pack(qmc_crowd* c, TD* dst, const TS* src, size_t nb, int rows, int cols, size_t sb, size_t sr, int scatter)
{
  const size_t total = nb * (size_t)rows * cols;
  if (total == 0) return QMC_OK;
  size_t blocks = (total + 255) / 256;
  if (blocks > 148 * 64) blocks = 148 * 64;
  pack_kernel<TD, TS><<<(unsigned)blocks, 256, 0, c->stream>>>(dst, src, nb, rows, cols, sb, sr, scatter);
  LAUNCH_CHECK(c);
  return QMC_OK;
}

}  // namespace

// ------------------------------------------------------------------------------------------
// C ABI
// ------------------------------------------------------------------------------------------
extern "C" {

const char* qmc_last_error(void) { return g_err; }
const char* qmc_version(void) { return "qmc_crowd_b200 0.1 (sm_100a)"; }

size_t qmc_crowd_workspace_bytes(const qmc_crowd_desc* desc)
{
  if (check_desc(desc) != QMC_OK) return 0;
  return carve(desc, nullptr, nullptr);
}

int qmc_crowd_create(const qmc_crowd_desc* desc, const double* pos_dev, qmc_crowd_t** out)
{
  if (!out) return fail(QMC_ERR_INVALID_ARG, "out is NULL");
  *out = nullptr;
  int st = check_desc(desc);
  if (st) return st;
  if (!pos_dev) return fail(QMC_ERR_INVALID_ARG, "pos_dev is NULL");
  if (!desc->coefs || ((uintptr_t)desc->coefs & 15)) return fail(QMC_ERR_INVALID_ARG, "coefs must be a 16-byte aligned device pointer");
  const size_t need = carve(desc, nullptr, nullptr);
  if (!desc->workspace || ((uintptr_t)desc->workspace & 255) || desc->workspace_bytes < need)
    return fail(QMC_ERR_WORKSPACE, "workspace must be 256-byte aligned and >= %zu bytes", need);
  int ndev = 0;
  CUDA_TRY(cudaGetDeviceCount(&ndev));
  if (ndev < 1) return fail(QMC_ERR_CUDA, "no CUDA device");

  qmc_crowd* c = new (std::nothrow) qmc_crowd();
  if (!c) return fail(QMC_ERR_INVALID_ARG, "out of host memory");
  c->desc = *desc;
  c->stream = (cudaStream_t)desc->stream;
  c->is_f64 = desc->coef_dtype;
  c->elem = desc->coef_dtype ? 8 : 4;
  c->state = ST_IDLE; c->state_k = -1; c->win_spin = -1;
  c->proposed = c->flushes = c->launches = 0;
  c->sweep_host = 0;
  c->use_graph = 1;
  c->n_sub = 0;
  c->strip_rows = 0;
  c->recompute_every = 0;
  {
    int devid = 0;
    c->n_sm = 148;
    if (cudaGetDevice(&devid) == cudaSuccess) cudaDeviceGetAttribute(&c->n_sm, cudaDevAttrMultiProcessorCount, devid);
    c->smem_optin = 48 * 1024;
    if (cudaGetDevice(&devid) == cudaSuccess) cudaDeviceGetAttribute(&c->smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, devid);
  }
  for (int i = 0; i < 4; ++i) { c->sub_stream[i] = nullptr; c->ev_join[i] = nullptr; }
  c->ev_fork = nullptr;
  c->graph_launches = c->graph_flushes = 0;
  c->graph_exec = nullptr;
  c->profile = 0;
  c->ev_used = 0;
  for (int i = 0; i < QMC_N_KERNEL_CLASSES; ++i) { c->prof_ms[i] = 0.0; c->prof_cnt[i] = 0; }
  CrowdDev& d = c->dev;
  memset(&d, 0, sizeof(d));
  d.W = desc->n_walkers; d.N = desc->n_elec; d.n = d.N / 2; d.M = desc->n_orb;
  d.ns = (int)align_up((size_t)d.n, 16);
  d.kd = desc->delay_rank; d.kdp = padded_rank(d.kd);
  d.walker_id0 = desc->walker_id0;
  d.seed_lo = (unsigned)(desc->seed & 0xffffffffu); d.seed_hi = (unsigned)(desc->seed >> 32);
  d.tau = desc->tau; d.sqrt_tau = std::sqrt(desc->tau); d.j2_a = desc->j2_a; d.j2_b = desc->j2_b;
  const int vw = desc->coef_dtype ? 2 : 4;
  for (int a = 0; a < 3; ++a) {
    d.grid[a] = desc->grid[a];
    d.box[a] = desc->box[a];
    d.inv_box[a] = 1.0 / desc->box[a];
    d.inv_h[a] = (double)desc->grid[a] / desc->box[a];
    d.inv_grid[a] = 1.0 / (double)desc->grid[a];
  }
  d.orb_stride_v = (unsigned)(desc->orb_stride / vw);
  d.tab_vecs = d.orb_stride_v;
  d.coefs = desc->coefs;
  carve(desc, &d, (char*)desc->workspace);

  auto bail = [&](int code) { qmc_crowd_destroy(c); return code; };
  cudaError_t e = cudaMemsetAsync(desc->workspace, 0, need, c->stream);
  if (e != cudaSuccess) return bail(fail(QMC_ERR_CUDA, "workspace memset: %s", cudaGetErrorString(e)));
  e = cudaMemcpyAsync(d.R, pos_dev, (size_t)d.W * d.N * 3 * 8, cudaMemcpyDeviceToDevice, c->stream);
  if (e != cudaSuccess) return bail(fail(QMC_ERR_CUDA, "position copy: %s", cudaGetErrorString(e)));
  c->launches += 2;
  for (int i = 1; i < 4; ++i) {
    if (cudaStreamCreateWithFlags(&c->sub_stream[i], cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_join[i], cudaEventDisableTiming) != cudaSuccess)
      return bail(fail(QMC_ERR_CUDA, "sub-crowd stream: %s", cudaGetErrorString(cudaGetLastError())));
  }
  if (cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming) != cudaSuccess)
    return bail(fail(QMC_ERR_CUDA, "sub-crowd event: %s", cudaGetErrorString(cudaGetLastError())));
  {
    const int sm = (int)move_smem(d), wsm = (int)window_smem(d, c->elem, 512);
    if (wsm > 227 * 1024 || sm > 227 * 1024)
      return bail(fail(QMC_ERR_INVALID_ARG, "n_elec / delay_rank too large: the per-walker state (%d bytes) exceeds shared memory", wsm));
    e = raise_smem_limits();
    if (e != cudaSuccess) return bail(fail(QMC_ERR_CUDA, "smem attribute: %s", cudaGetErrorString(e)));
  }
  st = rebuild(c);
  if (st) return bail(st);
  *out = c;
  return QMC_OK;
}

int qmc_crowd_destroy(qmc_crowd_t* c)
{
  if (!c) return QMC_OK;
  if (c->graph_exec) cudaGraphExecDestroy(c->graph_exec);
  for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
  for (int i = 1; i < 4; ++i) {
    if (c->sub_stream[i]) cudaStreamDestroy(c->sub_stream[i]);
    if (c->ev_join[i]) cudaEventDestroy(c->ev_join[i]);
  }
  if (c->ev_fork) cudaEventDestroy(c->ev_fork);
  delete c;
  return QMC_OK;
}

int qmc_spo_vgl(qmc_crowd_t* c, int k, const double* rnew_dev, void* phi, void* dphi, void* d2phi)
{
  if (!c) return fail(QMC_ERR_INVALID_ARG, "crowd is NULL");
  const CrowdDev& d = c->dev;
  if (k < 0 || k >= d.N) return fail(QMC_ERR_INVALID_ARG, "k out of range");
  const int spin = k / d.n, kk = k % d.n;
  if (d.kd > 1 && !c->win_rows.empty()) {
    if (spin != c->win_spin || (int)c->win_rows.size() >= d.kd)
      return fail(QMC_ERR_STATE, "delayed window is due for qmc_flush_delayed before electron %d", k);
    for (int r : c->win_rows)
      if (r == kk) return fail(QMC_ERR_STATE, "electron %d was already proposed in the open delayed window", k);
  }
  int st = step_vgl(c, k, rnew_dev);
  if (st) return st;
  c->state = ST_HAVE_VGL;
  c->state_k = k;
  const size_t ns = (size_t)d.ns;
  if (c->is_f64) {
    const double* v = (const double*)d.vgl;
    if (phi && (st = launch_pack(c, (double*)phi, v, d.W, 1, d.M, 5 * ns, ns, 0))) return st;
    if (dphi && (st = launch_pack(c, (double*)dphi, v + ns, d.W, 3, d.M, 5 * ns, ns, 0))) return st;
    if (d2phi && (st = launch_pack(c, (double*)d2phi, v + 4 * ns, d.W, 1, d.M, 5 * ns, ns, 0))) return st;
  } else {
    const float* v = (const float*)d.vgl;
    if (phi && (st = launch_pack(c, (float*)phi, v, d.W, 1, d.M, 5 * ns, ns, 0))) return st;
    if (dphi && (st = launch_pack(c, (float*)dphi, v + ns, d.W, 3, d.M, 5 * ns, ns, 0))) return st;
    if (d2phi && (st = launch_pack(c, (float*)d2phi, v + 4 * ns, d.W, 1, d.M, 5 * ns, ns, 0))) return st;
  }
  return QMC_OK;
}

int qmc_ratio_grad(qmc_crowd_t* c, int k, double* ratio, double* grad)
{
  if (!c) return fail(QMC_ERR_INVALID_ARG, "crowd is NULL");
  if (c->state != ST_HAVE_VGL || c->state_k != k)
    return fail(QMC_ERR_STATE, "qmc_ratio_grad(%d) must follow qmc_spo_vgl(%d)", k, k);
  int st = step_ratio(c, k, ratio, grad);
  if (st) return st;
  c->state = ST_HAVE_RATIO;
  return QMC_OK;
}

int qmc_accept_reject(qmc_crowd_t* c, int k, uint8_t* accepted)
{
  if (!c) return fail(QMC_ERR_INVALID_ARG, "crowd is NULL");
  if (c->state != ST_HAVE_RATIO || c->state_k != k)
    return fail(QMC_ERR_STATE, "qmc_accept_reject(%d) must follow qmc_ratio_grad(%d)", k, k);
  int st = step_accept(c, k, accepted);
  if (st) return st;
  c->state = ST_IDLE;
  c->proposed += (uint64_t)c->dev.W;
  if (c->dev.kd > 1) {
    c->win_spin = k / c->dev.n;
    c->win_rows.push_back(k % c->dev.n);
  }
  return QMC_OK;
}

int qmc_flush_delayed(qmc_crowd_t* c)
{
  if (!c) return fail(QMC_ERR_INVALID_ARG, "crowd is NULL");
  if (c->state != ST_IDLE) return fail(QMC_ERR_STATE, "qmc_flush_delayed in the middle of a move");
  if (c->dev.kd == 1 || c->win_rows.empty()) return QMC_OK;
  int st = launch_flush(c, c->win_spin);
  if (st) return st;
  c->win_rows.clear();
  c->win_spin = -1;
  return QMC_OK;
}

int qmc_sweep(qmc_crowd_t* c, int n_sweeps)
{
  if (!c) return fail(QMC_ERR_INVALID_ARG, "crowd is NULL");
  if (n_sweeps < 0) return fail(QMC_ERR_INVALID_ARG, "n_sweeps < 0");
  if (c->state != ST_IDLE) return fail(QMC_ERR_STATE, "qmc_sweep in the middle of a move");
  int st = qmc_flush_delayed(c);
  if (st) return st;
  if (c->use_graph && !c->profile && !c->graph_exec && n_sweeps > 0) {
    // capture one sweep; the sweep index lives in device memory so the graph is replayable
    cudaStream_t cap = nullptr;
    CUDA_TRY(cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking));
    cudaStream_t user = c->stream;
    const uint64_t launches0 = c->launches, flushes0 = c->flushes;
    cudaGraph_t graph = nullptr;
    cudaError_t e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
    if (e == cudaSuccess) {
      c->stream = cap;
      st = sweep_once(c);
      c->stream = user;
      e = cudaStreamEndCapture(cap, &graph);
    }
    c->graph_launches = c->launches - launches0;
    c->graph_flushes = c->flushes - flushes0;
    c->launches = launches0;
    c->flushes = flushes0;
    if (st == QMC_OK && e == cudaSuccess) e = cudaGraphInstantiate(&c->graph_exec, graph, 0);
    if (graph) cudaGraphDestroy(graph);
    cudaStreamDestroy(cap);
    if (st) return st;
    if (e != cudaSuccess) { c->graph_exec = nullptr; return fail(QMC_ERR_CUDA, "graph capture: %s", cudaGetErrorString(e)); }
  }
  const CrowdDev& d = c->dev;
  for (int s = 0; s < n_sweeps; ++s) {
    if (c->use_graph && !c->profile) {
      CUDA_TRY(cudaGraphLaunch(c->graph_exec, c->stream));
      c->launches += c->graph_launches;
      c->flushes += c->graph_flushes;
    } else {
      st = sweep_once(c);
      if (st) return st;
    }
    c->proposed += (uint64_t)d.W * d.N;
    ++c->sweep_host;
    if (c->recompute_every > 0 && c->sweep_host % (uint32_t)c->recompute_every == 0) {
      st = rebuild(c);
      if (st) return st;
    }
  }
  return QMC_OK;
}

int qmc_recompute_inverse(qmc_crowd_t* c)
{
  if (!c) return fail(QMC_ERR_INVALID_ARG, "crowd is NULL");
  if (c->state != ST_IDLE) return fail(QMC_ERR_STATE, "qmc_recompute_inverse in the middle of a move");
  return rebuild(c);
}

int qmc_sweep_host(qmc_crowd_t* c, double* pos_host, int n_sweeps, uint64_t* stats_host)
{
  if (!c || !pos_host) return fail(QMC_ERR_INVALID_ARG, "NULL argument");
  if (c->state != ST_IDLE) return fail(QMC_ERR_STATE, "qmc_sweep_host in the middle of a move");
  const CrowdDev& d = c->dev;
  const size_t bytes = (size_t)d.W * d.N * 3 * 8;
  CUDA_TRY(cudaMemcpyAsync(d.R, pos_host, bytes, cudaMemcpyHostToDevice, c->stream));
  int st = rebuild(c);
  if (st) return st;
  st = qmc_sweep(c, n_sweeps);
  if (st) return st;
  CUDA_TRY(cudaMemcpyAsync(pos_host, d.R, bytes, cudaMemcpyDeviceToHost, c->stream));
  unsigned long long acc = 0;
  CUDA_TRY(cudaMemcpyAsync(&acc, d.counters, 8, cudaMemcpyDeviceToHost, c->stream));
  CUDA_TRY(cudaStreamSynchronize(c->stream));
  if (stats_host) { stats_host[0] = c->proposed; stats_host[1] = acc; stats_host[2] = c->flushes; }
  return QMC_OK;
}

int qmc_crowd_get_positions(qmc_crowd_t* c, double* pos_dev)
{
  if (!c || !pos_dev) return fail(QMC_ERR_INVALID_ARG, "NULL argument");
  const CrowdDev& d = c->dev;
  CUDA_TRY(cudaMemcpyAsync(pos_dev, d.R, (size_t)d.W * d.N * 3 * 8, cudaMemcpyDeviceToDevice, c->stream));
  CUDA_TRY(cudaStreamSynchronize(c->stream));
  return QMC_OK;
}

int qmc_crowd_set_positions(qmc_crowd_t* c, const double* pos_dev)
{
  if (!c || !pos_dev) return fail(QMC_ERR_INVALID_ARG, "NULL argument");
  if (c->state != ST_IDLE) return fail(QMC_ERR_STATE, "set_positions in the middle of a move");
  const CrowdDev& d = c->dev;
  CUDA_TRY(cudaMemcpyAsync(d.R, pos_dev, (size_t)d.W * d.N * 3 * 8, cudaMemcpyDeviceToDevice, c->stream));
  return rebuild(c);
}

int qmc_crowd_get_inverse(qmc_crowd_t* c, int spin, double* binv_dev)
{
  if (!c || !binv_dev || spin < 0 || spin > 1) return fail(QMC_ERR_INVALID_ARG, "bad argument");
  const CrowdDev& d = c->dev;
  const size_t ns = (size_t)d.ns;
  int st = d.Binv32 ? launch_pack(c, binv_dev, d.Binv32 + (size_t)spin * ns * ns, d.W, d.n, d.n, 2 * ns * ns, ns, 0)
                    : launch_pack(c, binv_dev, d.Binv + (size_t)spin * ns * ns, d.W, d.n, d.n, 2 * ns * ns, ns, 0);
  if (st) return st;
  CUDA_TRY(cudaStreamSynchronize(c->stream));
  return QMC_OK;
}

int qmc_crowd_set_inverse(qmc_crowd_t* c, int spin, const double* binv_dev)
{
  if (!c || !binv_dev || spin < 0 || spin > 1) return fail(QMC_ERR_INVALID_ARG, "bad argument");
  if (c->state != ST_IDLE || !c->win_rows.empty()) return fail(QMC_ERR_STATE, "set_inverse needs an empty window");
  const CrowdDev& d = c->dev;
  const size_t ns = (size_t)d.ns;
  int st = d.Binv32 ? launch_pack(c, d.Binv32 + (size_t)spin * ns * ns, binv_dev, d.W, d.n, d.n, 2 * ns * ns, ns, 1)
                    : launch_pack(c, d.Binv + (size_t)spin * ns * ns, binv_dev, d.W, d.n, d.n, 2 * ns * ns, ns, 1);
  if (st) return st;
  CUDA_TRY(cudaStreamSynchronize(c->stream));
  return QMC_OK;
}

int qmc_crowd_get_caches(qmc_crowd_t* c, void* dphi_dev, void* d2phi_dev)
{
  if (!c) return fail(QMC_ERR_INVALID_ARG, "crowd is NULL");
  const CrowdDev& d = c->dev;
  const size_t ns = (size_t)d.ns, nb = (size_t)d.W * d.N;
  int st = QMC_OK;
  if (c->is_f64) {
    const double* s = (const double*)d.cache;
    if (dphi_dev) st = launch_pack(c, (double*)dphi_dev, s, nb, 3, d.M, 4 * ns, ns, 0);
    if (!st && d2phi_dev) st = launch_pack(c, (double*)d2phi_dev, s + 3 * ns, nb, 1, d.M, 4 * ns, ns, 0);
  } else {
    const float* s = (const float*)d.cache;
    if (dphi_dev) st = launch_pack(c, (float*)dphi_dev, s, nb, 3, d.M, 4 * ns, ns, 0);
    if (!st && d2phi_dev) st = launch_pack(c, (float*)d2phi_dev, s + 3 * ns, nb, 1, d.M, 4 * ns, ns, 0);
  }
  if (st) return st;
  CUDA_TRY(cudaStreamSynchronize(c->stream));
  return QMC_OK;
}

int qmc_crowd_get_window(qmc_crowd_t* c, int32_t* m_dev, int32_t* rows_dev, double* v_dev, double* c_dev, double* sinv_dev)
{
  if (!c) return fail(QMC_ERR_INVALID_ARG, "crowd is NULL");
  const CrowdDev& d = c->dev;
  if (d.kd == 1) return fail(QMC_ERR_STATE, "no delayed window with delay_rank 1");
  const size_t ns = (size_t)d.ns, kdp = (size_t)d.kdp;
  int st = QMC_OK;
  if (m_dev) st = launch_pack(c, m_dev, d.mwin, 1, 1, d.W, 0, 0, 0);
  if (!st && rows_dev) st = launch_pack(c, rows_dev, d.rows, d.W, 1, d.kd, kdp, kdp, 0);
  if (!st && v_dev) st = launch_pack(c, v_dev, d.V, d.W, d.kd, d.n, kdp * ns, ns, 0);
  if (!st && c_dev) st = launch_pack(c, c_dev, d.C, d.W, d.kd, d.n, kdp * ns, ns, 0);
  if (!st && sinv_dev) st = launch_pack(c, sinv_dev, d.Sinv, d.W, d.kd, d.kd, kdp * kdp, kdp, 0);
  if (st) return st;
  CUDA_TRY(cudaStreamSynchronize(c->stream));
  return QMC_OK;
}

int qmc_crowd_get_move(qmc_crowd_t* c, double* rnew, double* delta, double* g_old, double* g_new, double* rho_d,
                       double* rho_j, double* p, double* u, double* brow)
{
  if (!c) return fail(QMC_ERR_INVALID_ARG, "crowd is NULL");
  const CrowdDev& d = c->dev;
  const size_t W = (size_t)d.W;
  auto cp = [&](double* dst, const double* src, size_t cnt) -> cudaError_t {
    return dst ? cudaMemcpyAsync(dst, src, cnt * 8, cudaMemcpyDeviceToDevice, c->stream) : cudaSuccess;
  };
  CUDA_TRY(cp(rnew, d.rnew, 3 * W));
  CUDA_TRY(cp(delta, d.delta, 3 * W));
  CUDA_TRY(cp(g_old, d.g_old, 3 * W));
  CUDA_TRY(cp(g_new, d.g_new, 3 * W));
  CUDA_TRY(cp(rho_d, d.rho_d, W));
  CUDA_TRY(cp(rho_j, d.rho_j, W));
  CUDA_TRY(cp(p, d.p, W));
  CUDA_TRY(cp(u, d.u, W));
  if (brow) {
    int st = launch_pack(c, brow, d.brow, W, 1, d.n, (size_t)d.ns, (size_t)d.ns, 0);
    if (st) return st;
  }
  CUDA_TRY(cudaStreamSynchronize(c->stream));
  return QMC_OK;
}

int qmc_kinetic_energy(qmc_crowd_t* c, double* ekin_dev, double* e_elec_dev)
{
  if (!c || !ekin_dev) return fail(QMC_ERR_INVALID_ARG, "NULL argument");
  if (c->state != ST_IDLE) return fail(QMC_ERR_STATE, "qmc_kinetic_energy in the middle of a move");
  if (!c->win_rows.empty()) return fail(QMC_ERR_STATE, "qmc_kinetic_energy needs a flushed window (call qmc_flush_delayed)");
  const CrowdDev& d = c->dev;
  const size_t smem = (size_t)(3 * d.N) * 8;
  dim3 grid((d.N + EKIN_EPB - 1) / EKIN_EPB, d.W);
  {
    ProfScope ps(c, QMC_K_KINETIC);
    if (c->is_f64) {
      kinetic_kernel<double><<<grid, EKIN_NT, smem, c->stream>>>(d, d.e_elec);
    } else {
      kinetic_kernel<float><<<grid, EKIN_NT, smem, c->stream>>>(d, d.e_elec);
    }
    LAUNCH_CHECK(c);
    kinetic_sum_kernel<<<(d.W + 3) / 4, 128, 0, c->stream>>>(d.W, d.N, d.e_elec, ekin_dev);
    LAUNCH_CHECK(c);
  }
  if (e_elec_dev) CUDA_TRY(cudaMemcpyAsync(e_elec_dev, d.e_elec, (size_t)d.W * d.N * 8, cudaMemcpyDeviceToDevice, c->stream));
  return QMC_OK;
}

int qmc_crowd_branch(qmc_crowd_t* c, const int32_t* src_dev, int* n_copied)
{
  if (!c || !src_dev) return fail(QMC_ERR_INVALID_ARG, "NULL argument");
  if (c->state != ST_IDLE) return fail(QMC_ERR_STATE, "qmc_crowd_branch in the middle of a move");
  int st = qmc_flush_delayed(c);
  if (st) return st;
  const CrowdDev& d = c->dev;
  // validate the map on the device; d.status doubles as the flag, d.mwin[0] (zero: the window is empty) as the counter
  CUDA_TRY(cudaMemsetAsync(d.status, 0, 4, c->stream));
  branch_check_kernel<<<(d.W + 255) / 256, 256, 0, c->stream>>>(d, src_dev);
  LAUNCH_CHECK(c);
  branch_count_kernel<<<(d.W + 255) / 256, 256, 0, c->stream>>>(d.W, src_dev, d.mwin);
  LAUNCH_CHECK(c);
  int flag = 0, cnt = 0;
  CUDA_TRY(cudaMemcpyAsync(&flag, d.status, 4, cudaMemcpyDeviceToHost, c->stream));
  CUDA_TRY(cudaMemcpyAsync(&cnt, d.mwin, 4, cudaMemcpyDeviceToHost, c->stream));
  CUDA_TRY(cudaMemsetAsync(d.status, 0, 4, c->stream));
  CUDA_TRY(cudaMemsetAsync(d.mwin, 0, 4, c->stream));
  CUDA_TRY(cudaStreamSynchronize(c->stream));
  if (flag) return fail(QMC_ERR_INVALID_ARG, "src is not a branching map: entries must lie in [0, W) and sources must keep their own state");
  if (n_copied) *n_copied = cnt;
  if (cnt == 0) return QMC_OK;
  {
    ProfScope ps(c, QMC_K_BRANCH);
    const WalkerState ws = walker_state(d, c->elem);
    branch_copy_kernel<<<dim3(state_chunks(ws), d.W), BRANCH_NT, 0, c->stream>>>(d, src_dev, ws);
    LAUNCH_CHECK(c);
  }
  return QMC_OK;
}

size_t qmc_crowd_walker_state_bytes(const qmc_crowd_t* c)
{
  if (!c) return 0;
  return walker_state(c->dev, c->elem).total();
}

namespace {
int walker_pack(qmc_crowd_t* c, int n, const int32_t* slots_dev, void* buf_dev, bool do_export)
{
  if (!c || n < 0 || (n > 0 && (!slots_dev || !buf_dev))) return fail(QMC_ERR_INVALID_ARG, "bad argument");
  if (c->state != ST_IDLE) return fail(QMC_ERR_STATE, "walker export / import in the middle of a move");
  if (((uintptr_t)buf_dev & 15) != 0) return fail(QMC_ERR_INVALID_ARG, "buffer must be 16-byte aligned");
  int st = qmc_flush_delayed(c);
  if (st) return st;
  const CrowdDev& d = c->dev;
  if (n == 0) return QMC_OK;
  if (n > d.W) return fail(QMC_ERR_INVALID_ARG, "more slots than walkers");
  // slots must be in range and distinct; d.mwin (all zero: the window is empty) holds the marks
  CUDA_TRY(cudaMemsetAsync(d.status, 0, 4, c->stream));
  slots_check_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(d, n, slots_dev, d.mwin);
  LAUNCH_CHECK(c);
  int flag = 0;
  CUDA_TRY(cudaMemcpyAsync(&flag, d.status, 4, cudaMemcpyDeviceToHost, c->stream));
  CUDA_TRY(cudaMemsetAsync(d.status, 0, 4, c->stream));
  CUDA_TRY(cudaMemsetAsync(d.mwin, 0, (size_t)d.W * 4, c->stream));
  CUDA_TRY(cudaStreamSynchronize(c->stream));
  if (flag) return fail(QMC_ERR_INVALID_ARG, "slots must lie in [0, W) and be distinct");
  ProfScope ps(c, QMC_K_BRANCH);
  const WalkerState ws = walker_state(d, c->elem);
  if (do_export) walker_pack_kernel<true><<<dim3(state_chunks(ws), n), BRANCH_NT, 0, c->stream>>>(d, slots_dev, (char*)buf_dev, ws);
  else walker_pack_kernel<false><<<dim3(state_chunks(ws), n), BRANCH_NT, 0, c->stream>>>(d, slots_dev, (char*)buf_dev, ws);
  LAUNCH_CHECK(c);
  return QMC_OK;
}
}  // namespace

int qmc_crowd_export_walkers(qmc_crowd_t* c, int n, const int32_t* slots_dev, void* buf_dev)
{
  return walker_pack(c, n, slots_dev, buf_dev, true);
}

int qmc_crowd_import_walkers(qmc_crowd_t* c, int n, const int32_t* slots_dev, const void* buf_dev)
{
  return walker_pack(c, n, slots_dev, const_cast<void*>(buf_dev), false);
}

int qmc_crowd_set_sweep_index(qmc_crowd_t* c, uint32_t s)
{
  if (!c) return fail(QMC_ERR_INVALID_ARG, "crowd is NULL");
  set_u32_kernel<<<1, 1, 0, c->stream>>>(c->dev.sweep, s);
  LAUNCH_CHECK(c);
  c->sweep_host = s;
  return QMC_OK;
}

int qmc_crowd_stats(qmc_crowd_t* c, uint64_t* proposed, uint64_t* accepted, uint64_t* flushes)
{
  if (!c) return fail(QMC_ERR_INVALID_ARG, "crowd is NULL");
  unsigned long long acc = 0;
  CUDA_TRY(cudaMemcpyAsync(&acc, c->dev.counters, 8, cudaMemcpyDeviceToHost, c->stream));
  CUDA_TRY(cudaStreamSynchronize(c->stream));
  if (proposed) *proposed = c->proposed;
  if (accepted) *accepted = acc;
  if (flushes) *flushes = c->flushes;
  return QMC_OK;
}

int qmc_crowd_get_profile(qmc_crowd_t* c, double* ms, uint64_t* count)
{
  if (!c) return fail(QMC_ERR_INVALID_ARG, "crowd is NULL");
  CUDA_TRY(cudaStreamSynchronize(c->stream));
  for (size_t i = 0; i < c->ev_used; ++i) {
    float t = 0.f;
    CUDA_TRY(cudaEventElapsedTime(&t, c->ev[2 * i], c->ev[2 * i + 1]));
    c->prof_ms[c->ev_class[i]] += (double)t;
    c->prof_cnt[c->ev_class[i]] += 1;
  }
  c->ev_used = 0;
  for (int i = 0; i < QMC_N_KERNEL_CLASSES; ++i) {
    if (ms) ms[i] = c->prof_ms[i];
    if (count) count[i] = c->prof_cnt[i];
    c->prof_ms[i] = 0.0;
    c->prof_cnt[i] = 0;
  }
  return QMC_OK;
}

uint64_t qmc_crowd_launch_count(const qmc_crowd_t* c) { return c ? c->launches : 0; }

int qmc_crowd_set_option(qmc_crowd_t* c, int option, int value)
{
  if (!c) return fail(QMC_ERR_INVALID_ARG, "crowd is NULL");
  if (option == QMC_OPT_GRAPH) { c->use_graph = value ? 1 : 0; return QMC_OK; }
  if (option == QMC_OPT_PROFILE) { c->profile = value ? 1 : 0; return QMC_OK; }
  if (option == QMC_OPT_SUBCROWDS) {
    if (value < 0 || value > 4) return fail(QMC_ERR_INVALID_ARG, "sub-crowds must be in [0,4] (0 = automatic)");
    c->n_sub = value;
    if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
    return QMC_OK;
  }
  if (option == QMC_OPT_STRIP_ROWS) {
    if (value != 0 && value != 16 && value != 32) return fail(QMC_ERR_INVALID_ARG, "strip rows must be 0 (automatic), 16 or 32");
    c->strip_rows = value;
    if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
    return QMC_OK;
  }
  if (option == QMC_OPT_RECOMPUTE_EVERY) {
    if (value < 0) return fail(QMC_ERR_INVALID_ARG, "recompute period must be >= 0");
    c->recompute_every = value;
    return QMC_OK;
  }
  return fail(QMC_ERR_INVALID_ARG, "unknown option %d", option);
}

}  // extern "C"

// ------------------------------------------------------------------------------------------
// qmc_spo_vgl_static: the orbital evaluation with its scratch in a static device array (include/qmc_crowd.h)
// ------------------------------------------------------------------------------------------
namespace {

// The internal [n_pos][5][ns] result buffer of the spline kernel (what d.vgl is in a crowd's workspace).  In HOST code
// this name is a host-side stand-in, not a device address: host code uses static_scratch_address() below.
static __device__ __align__(256) unsigned char g_static_scratch[QMC_STATIC_SCRATCH_BYTES];

// Variant of spline_vgl_kernel: one CTA per position r[b], result into vgl[b] (the static array), no crowd state.
template <typename T>
__global__ void __launch_bounds__(qmc::SPLINE_NT, 4) spline_vgl_static_kernel(qmc::CrowdDev d, const double* __restrict__ r,
                                                                              T* __restrict__ vgl)
{
  __shared__ qmc::SplineW<T> s;
  const size_t b = blockIdx.x;
  qmc::spline_cta<T, qmc::SPLINE_NT>(d, r + 3 * b, s, vgl + b * 5 * d.ns);
}

// Device address of g_static_scratch on the current device: looked up once per device, with that device current.
int static_scratch_address(void** out)
{
  static void* addr[64] = {};
  static std::mutex mu;
  int dev = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return fail(QMC_ERR_INVALID_ARG, "device ordinal %d out of range", dev);
  std::lock_guard<std::mutex> lock(mu);
  if (!addr[dev]) {
    void* p = nullptr;
    CUDA_TRY(cudaGetSymbolAddress(&p, g_static_scratch));
    if (!p) return fail(QMC_ERR_CUDA, "cudaGetSymbolAddress returned a null address for the static scratch");
    addr[dev] = p;
  }
  *out = addr[dev];
  return QMC_OK;
}

template <typename T>
int spo_vgl_static_t(const qmc::CrowdDev& d, int n_pos, const double* r_dev, T* vgl, T* phi, T* dphi, T* d2phi, cudaStream_t stream)
{
  spline_vgl_static_kernel<T><<<(unsigned)n_pos, qmc::SPLINE_NT, 0, stream>>>(d, r_dev, vgl);
  const size_t ns = (size_t)d.ns;
  struct Out { T* dst; const T* src; int rows; } outs[3] = {{phi, vgl, 1}, {dphi, vgl + ns, 3}, {d2phi, vgl + 4 * ns, 1}};
  for (const Out& o : outs) {
    if (!o.dst) continue;
    const size_t total = (size_t)n_pos * o.rows * d.M;
    const size_t blocks = std::min<size_t>((total + 255) / 256, 148 * 64);
    qmc::pack_kernel<T, T><<<(unsigned)blocks, 256, 0, stream>>>(o.dst, o.src, (size_t)n_pos, o.rows, d.M, 5 * ns, ns, 0);
  }
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(QMC_ERR_CUDA, "kernel launch: %s (%s:%d)", cudaGetErrorString(e), __FILE__, __LINE__);
  return QMC_OK;
}

}  // namespace

extern "C" int qmc_spo_vgl_static(int32_t n_orb, const int32_t* grid, const double* box, int32_t coef_dtype,
                                  const void* coefs_dev, int64_t orb_stride, int32_t n_pos, const double* r_dev,
                                  void* phi, void* dphi, void* d2phi, void* stream)
{
  using namespace qmc;
  if (!grid || !box) return fail(QMC_ERR_INVALID_ARG, "grid / box is NULL");
  if (n_orb < 1) return fail(QMC_ERR_INVALID_ARG, "n_orb must be >= 1");
  if (coef_dtype != 0 && coef_dtype != 1) return fail(QMC_ERR_INVALID_ARG, "coef_dtype must be 0 or 1");
  const int vw = coef_dtype ? 2 : 4;
  if (orb_stride < n_orb || orb_stride % vw) return fail(QMC_ERR_INVALID_ARG, "orb_stride must be >= n_orb and a multiple of %d", vw);
  double tab = (double)orb_stride / vw;
  for (int c = 0; c < 3; ++c) {
    if (grid[c] < 1) return fail(QMC_ERR_INVALID_ARG, "grid must be >= 1");
    if (!(box[c] > 0.0) || !std::isfinite(box[c])) return fail(QMC_ERR_INVALID_ARG, "box must be positive");
    tab *= grid[c];
  }
  if (tab >= 4294967296.0) return fail(QMC_ERR_INVALID_ARG, "coefficient table larger than 2^32 16-byte vectors");
  if (n_pos < 0) return fail(QMC_ERR_INVALID_ARG, "n_pos must be >= 0");
  if (n_pos == 0) return QMC_OK;
  if (!coefs_dev || !r_dev) return fail(QMC_ERR_INVALID_ARG, "coefs_dev / r_dev is NULL");
  const size_t ns = align_up((size_t)n_orb, 16), elem = coef_dtype ? 8 : 4;
  const size_t need = (size_t)n_pos * 5 * ns * elem;
  if (need > (size_t)QMC_STATIC_SCRATCH_BYTES)
    return fail(QMC_ERR_WORKSPACE, "qmc_spo_vgl_static: %d positions x %d orbitals need %zu bytes of scratch, the static array holds %zu "
                "(at most %zu positions per call for this table)", n_pos, n_orb, need, (size_t)QMC_STATIC_SCRATCH_BYTES,
                (size_t)QMC_STATIC_SCRATCH_BYTES / (5 * ns * elem));
  void* scratch = nullptr;
  int st = static_scratch_address(&scratch);
  if (st) return st;
  CrowdDev d;
  memset(&d, 0, sizeof(d));
  d.W = n_pos; d.M = n_orb; d.n = n_orb; d.N = 2 * n_orb; d.ns = (int)ns;
  for (int a = 0; a < 3; ++a) {
    d.grid[a] = grid[a];
    d.box[a] = box[a];
    d.inv_box[a] = 1.0 / box[a];
    d.inv_h[a] = (double)grid[a] / box[a];
    d.inv_grid[a] = 1.0 / (double)grid[a];
  }
  d.orb_stride_v = (unsigned)(orb_stride / vw);
  d.tab_vecs = d.orb_stride_v;
  d.coefs = coefs_dev;
  cudaStream_t s = (cudaStream_t)stream;
  return coef_dtype ? spo_vgl_static_t<double>(d, n_pos, r_dev, (double*)scratch, (double*)phi, (double*)dphi, (double*)d2phi, s)
                    : spo_vgl_static_t<float>(d, n_pos, r_dev, (float*)scratch, (float*)phi, (float*)dphi, (float*)d2phi, s);
}
