/*
 * qmc_crowd.h -- C ABI of the B200-native crowd move (libqmc_crowd.so).
 *
 * One thing is built here: the particle-by-particle electron move of arXiv:2209.14487
 * applied to a whole crowd of walkers in lock-step.  Citations:
 *   P:n   = /root/reference/PAPER.md line n
 *   BJ    = BASELINE.json north_star
 *   D:Cx / D:Ax = DESIGN.md "Readings" (restated from SURVEY.md 8(c))
 *
 *   Alg. 1 lines 5-9: propose, ratio, gradient at the new position, accept/reject.
 *   Alg. 3 / Alg. 4: every routine serves all walkers of the crowd in
 *   one batched call and all walkers advance in lock-step for each single particle move.
 *   a crowd is a sub-population advanced in lock-step; one crowd is the legacy
 *   single-stream case.  The arithmetic inside each call is named by BJ; the formula each call
 *   evaluates is given with the call.
 *
 * Conventions
 *   - plain C types only; nothing throws; every call returns a qmc_status (QMC_OK = 0) and the
 *     text of the last failure on this host thread is kept for qmc_last_error().
 *   - "DEVICE" pointers are CUDA device pointers of the current device, "HOST" pointers are host
 *     memory.  BORROWED pointers must outlive the crowd; the library never frees them.
 *   - the library allocates NO device memory: the caller hands it one workspace
 *     (size from qmc_crowd_workspace_bytes) and the coefficient table (BJ: "PyTorch only for
 *     device memory and streams").
 *   - all step calls are asynchronous on desc.stream unless stated otherwise.
 *   - N electrons, n = N/2 per spin, M = n orbitals shared by both spins (D:A5), W walkers.
 *     Electrons [0,n) are spin-up (determinant 0), [n,N) spin-down (determinant 1).
 *   - there is no CPU fallback anywhere: without a CUDA device every call that touches the
 *     device fails with QMC_ERR_CUDA.
 */
#ifndef QMC_CROWD_H
#define QMC_CROWD_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct qmc_crowd qmc_crowd_t; /* opaque; owned by the library (host struct only) */

typedef enum {
  QMC_OK = 0,
  QMC_ERR_INVALID_ARG = 1, /* NULL pointer, bad size, unsupported shape                         */
  QMC_ERR_CUDA = 2,        /* a CUDA call failed (text in qmc_last_error)                       */
  QMC_ERR_WORKSPACE = 3,   /* workspace NULL, misaligned (256 B) or too small                   */
  QMC_ERR_SINGULAR = 4,    /* a Slater matrix had a zero / non-finite pivot (D:A16)             */
  QMC_ERR_STATE = 5        /* step calls out of order, or a flush the schedule requires is due  */
} qmc_status;

typedef struct {
  int32_t n_elec;      /* N, even, >= 2                                                          */
  int32_t n_orb;       /* M, must equal N/2 (D:A5)                                               */
  int32_t grid[3];     /* Ng per axis, >= 1                                                      */
  int32_t coef_dtype;  /* 0 = fp32 table (orbitals evaluated in fp32), 1 = fp64 table            */
  double box[3];       /* L per axis, orthorhombic periodic cell                                 */
  const void* coefs;   /* DEVICE, BORROWED: P[gx][gy][gz][orb_stride], orbital index innermost   */
                       /* (BJ: "coefficients stored orbital-innermost"), 16-byte aligned         */
  int64_t orb_stride;  /* elements between grid points: >= n_orb, multiple of 4 (fp32) / 2 (fp64)*/
  double j2_a, j2_b;   /* two-body Jastrow u(r) = a r / (1 + b r)  (D:C3)                        */
  double tau;          /* time step of the drift-diffusion proposal (D:C4)                       */
  int32_t n_walkers;   /* W >= 1                                                                 */
  int32_t walker_id0;  /* global id of walker 0: Philox counter word 0 is walker_id0 + w (D:C7), */
                       /* so splitting a population into crowds does not change any trajectory   */
  int32_t delay_rank;  /* 1 = Sherman-Morrison rank-1 (D:C5); 2..64 = delayed rank-k (D:C6)      */
  int32_t inverse_dtype; /* 0 = the carried inverses are fp64 (BASELINE.json configs).  1 = mixed    */
                       /* precision (SURVEY 8(f) item 3, D:R6): the carried inverses are STORED in  */
                       /* fp32 -- rounded to nearest after every operation that writes them         */
                       /* (inversion, rank-1 update, flush) -- and every dot product and update is  */
                       /* evaluated in fp64 on the stored values; halves the dominant bytes of the  */
                       /* update kernels.  Needs delay_rank <= 32 (a flush is then ONE pass, one    */
                       /* rounding).  Companion: QMC_OPT_RECOMPUTE_EVERY (fp64 re-inversion).       */
  uint64_t seed;       /* Philox key (lo, hi)                                                    */
  void* workspace;     /* DEVICE, BORROWED, 256-byte aligned                                     */
  size_t workspace_bytes; /* >= qmc_crowd_workspace_bytes(&desc)                                 */
  void* stream;        /* cudaStream_t (0 = legacy default stream), BORROWED                     */
} qmc_crowd_desc;

/* Bytes of device workspace a crowd of this shape needs (positions, transposed inverses,
 * per-electron gradient/Laplacian caches, delayed window, per-move scratch). 0 on a bad desc. */
size_t qmc_crowd_workspace_bytes(const qmc_crowd_desc* desc);

/* BJ "qmc_crowd_create".  Copies pos_dev (DEVICE, [W][N][3] fp64) into the workspace, evaluates
 * the Slater matrices A^s_ij = phi_j(r_{s n + i}) of both spins with the spline kernel (D:C1,C2),
 * inverts them on the device by Gauss-Jordan with partial pivoting into the stored form
 * B = (A^-1)^T (row = electron, D:A9), fills the per-electron caches of grad phi / lap phi
 * (D:A12, A13), and synchronises the stream.  Returns QMC_ERR_SINGULAR (and no crowd) when a
 * pivot is zero or not finite. */
int qmc_crowd_create(const qmc_crowd_desc* desc, const double* pos_dev, qmc_crowd_t** out);
int qmc_crowd_destroy(qmc_crowd_t* crowd);

/* ---- one electron index k for ALL walkers of the crowd (Alg. 3 line 3) -------------
 * The three calls must be issued in this order for the same k; otherwise QMC_ERR_STATE.
 * With delay_rank > 1 a flush is due after every delay_rank proposed moves of a spin block
 * and at the end of each spin block (D:C6 schedule); qmc_spo_vgl returns QMC_ERR_STATE if that
 * flush was not issued (qmc_sweep does it itself).                                            */

/* BJ "qmc_spo_vgl" = Alg. 1 line 5 (reading D:A1) followed by the orbital evaluation.
 *  (a) current inverse row b of electron k with the pending delayed window applied (D:C6),
 *      G_k(R) = b . grad phi(r_k) [cache] + grad_k ln Psi_J(R)   (D:C2, C3, A13);
 *  (b) if rnew_dev == NULL: Delta = fl32(tau G_k(R) + sqrt(tau) chi), chi from Philox
 *      counter (walker id, k, sweep, 0), r' = r_k + Delta (D:C4, C7);
 *      else r' = rnew_dev[w] (DEVICE, [W][3] fp64) and Delta = r' - r_k (teacher forcing);
 *  (c) phi_j(r'), grad phi_j(r'), lap phi_j(r') for j < M: the 4x4x4 tricubic B-spline stencil
 *      (D:C1), evaluated in the table's precision.
 * phi / dphi / d2phi: optional DEVICE outputs (NULL to skip), element type = table type,
 * compact layouts [W][M], [W][3][M], [W][M].                                                  */
int qmc_spo_vgl(qmc_crowd_t* crowd, int k, const double* rnew_dev, void* phi, void* dphi, void* d2phi);

/* BJ "qmc_ratio_grad" = Alg. 1 lines 7-8.  rho_D = b . phi(r') (matrix-determinant
 * lemma, D:C2); rho_J = exp(sum_{i!=k} u(|r'-r_i|) - u(|r_k-r_i|)) (D:C3);
 * ratio[w] = rho_D rho_J;  grad[w] = (b . grad phi(r'))/rho_D + grad_k ln Psi_J(R').
 * ratio: DEVICE [W] fp64 or NULL; grad: DEVICE [W][3] fp64 or NULL.                           */
int qmc_ratio_grad(qmc_crowd_t* crowd, int k, double* ratio, double* grad);

/* BJ "qmc_accept_reject" = Alg. 1 line 9 (reading D:A3).  p = rho^2 exp(logGb - logGf)
 * with the applied Delta (D:C4); u from Philox counter (walker id, k, sweep, 1); accept <=> u < p,
 * non-finite p or rho_D == 0 rejects.  On accept: r_k <- r', caches <- new, and the inverse is
 * updated by Sherman-Morrison (delay_rank 1, D:C5) or the move is appended to the delayed
 * window (D:C6).  On reject nothing changes.  accepted: DEVICE [W] uint8 or NULL.      */
int qmc_accept_reject(qmc_crowd_t* crowd, int k, uint8_t* accepted);

/* BJ "qmc_flush_delayed" (D:C6): B <- B0 - (B0 V^T - E) S^-T C for every walker with a
 * non-empty window (FP64 DMMA), then empties the windows.  No-op for delay_rank 1 or when
 * nothing was proposed since the last flush.                                                  */
int qmc_flush_delayed(qmc_crowd_t* crowd);

/* BJ "qmc_sweep": n_sweeps full sweeps k = 0..N-1 (P:73 particle-by-particle; Alg. 3 lines 2-4)
 * of propose / vgl / ratio / accept with the flush schedule of D:C6; the sweep index (Philox
 * counter word 2) advances by one per sweep.  Ends flushed.  Asynchronous.
 * Same moves, decisions and positions as the step calls issued in that order; with delay_rank > 1 the
 * crowd advances in lock-step per delay window (a walker's moves of a window run back to back, DESIGN.md
 * R5) and the inverses agree with the step-call path to rounding (1e-10).  Requires the per-walker state
 * of a move (about 42 KB at N = 768) to fit shared memory: N up to a few thousand.                     */
int qmc_sweep(qmc_crowd_t* crowd, int n_sweeps);

/* Host-buffer form of the same path (bench.py "e2e"): copies pos_host (HOST, [W][N][3] fp64)
 * to the device, rebuilds Slater matrices / inverses / caches from it (as qmc_crowd_create),
 * runs n_sweeps sweeps, copies the positions back into pos_host and the three counters
 * (proposed, accepted, flushes; totals since create) into stats_host[3].  Synchronous.       */
int qmc_sweep_host(qmc_crowd_t* crowd, double* pos_host, int n_sweeps, uint64_t* stats_host);

/* Kinetic part of the local energy of every walker at its current configuration (Alg. 1 line 11, PAPER.md:59 and
 * :77 "local energy ... expensive"; the potential part needs pseudopotentials / Ewald sums and
 * is out of scope):  ekin[w] = -1/2 sum_k lap_k Psi / Psi,  lap_k Psi / Psi = lap_k ln Psi + |grad_k ln Psi|^2,
 * Psi = D_up D_dn Psi_J, atomic units.  Uses the carried inverses, the per-electron gradient / Laplacian caches and
 * the positions; changes no state.  ekin_dev: DEVICE [W] fp64 (required); e_elec_dev: DEVICE [W][N] fp64 per-electron
 * terms or NULL.  Asynchronous on desc.stream.  QMC_ERR_STATE in the middle of a move or with an open delayed window
 * (call qmc_flush_delayed first; qmc_sweep always returns flushed).                                              */
int qmc_kinetic_energy(qmc_crowd_t* crowd, double* ekin_dev, double* e_elec_dev);

/* Periodic recompute of the inverses (first half; the usual answer to the round-off drift of
 * repeated Sherman-Morrison / delayed updates; "update the internal data of a walker" names
 * the carried data this replaces): rebuilds both Slater matrices of every walker from the crowd's CURRENT positions
 * (B-spline values and the gradient / Laplacian caches of every electron), inverts them with partial pivoting in fp64
 * and drops any open delayed window -- the same code path as qmc_crowd_create / qmc_crowd_set_positions, so the
 * result is bit-identical to a crowd created at those positions.  Counters and the sweep index are kept.
 * Synchronises desc.stream.  QMC_ERR_STATE in the middle of a move; QMC_ERR_SINGULAR as for qmc_crowd_create (the
 * crowd is then unusable until qmc_crowd_set_positions succeeds).                                             */
int qmc_recompute_inverse(qmc_crowd_t* crowd);

/* DMC branching, data movement only (Alg. 1 L13 "branch"; P:66 for the walker
 * states it moves): walker slot w takes over the whole carried state of slot src[w] -- positions, both inverses,
 * gradient / Laplacian caches.  src is a DEVICE int32 array of W entries, BORROWED; every source must keep its own
 * state (src[src[w]] == src[w], which includes src[w] == w for walkers that are not replaced); an invalid map returns
 * QMC_ERR_INVALID_ARG and changes nothing.  Random-number streams stay with the slot (PAPER.md gives no rule; D:A3
 * keys Philox on the global walker id), so a copy diverges from its source at the next move.  Counters and the sweep
 * index are kept; an open delayed window is flushed first.  Synchronises desc.stream (the map is validated on the
 * device before the copy).  n_copied (HOST, may be NULL) receives the number of slots that were overwritten.    */
int qmc_crowd_branch(qmc_crowd_t* crowd, const int32_t* src_dev, int* n_copied);

/* Walker states as messages (second half; the DMC load balance of Alg. 1 L14,
 * PAPER.md:66, P:71 moves whole walkers between ranks).  A packed state is qmc_crowd_walker_state_bytes(crowd) bytes:
 * [both inverses, fp64 [2][ns][ns] | gradient / Laplacian caches, table dtype [N][4][ns] | positions, fp64 [N][3]];
 * it can be imported only into a crowd created with the same n_elec, n_orb and coefficient dtype (same byte count).
 * export: buf[i] <- state of slot slots[i]; import: slot slots[i] <- buf[i], i < n.  slots: DEVICE int32 [n], in
 * [0, W) and distinct (else QMC_ERR_INVALID_ARG, nothing copied); buf: DEVICE, 16-byte aligned, n packed states,
 * BORROWED.  An open delayed window is flushed first; the validation synchronises desc.stream, the copy itself is
 * asynchronous on it.  The transport between ranks is the caller's (paper_2209_14487_b200/dist.py sends the packed
 * buffers point-to-point on the NCCL backend).                                                                 */
size_t qmc_crowd_walker_state_bytes(const qmc_crowd_t* crowd);
int qmc_crowd_export_walkers(qmc_crowd_t* crowd, int n, const int32_t* slots_dev, void* buf_dev);
int qmc_crowd_import_walkers(qmc_crowd_t* crowd, int n, const int32_t* slots_dev, const void* buf_dev);

/* ---- state access for tests: synchronous copies on desc.stream -------------------------- */
int qmc_crowd_get_positions(qmc_crowd_t* crowd, double* pos_dev /* DEVICE [W][N][3] */);
int qmc_crowd_set_positions(qmc_crowd_t* crowd, const double* pos_dev); /* rebuilds, may be SINGULAR */
/* transposed inverse of one spin, compact DEVICE [W][n][n]; with a window open this is B0 */
int qmc_crowd_get_inverse(qmc_crowd_t* crowd, int spin, double* binv_dev);
int qmc_crowd_set_inverse(qmc_crowd_t* crowd, int spin, const double* binv_dev); /* window must be empty */
/* per-electron caches, element type = table type, compact DEVICE [W][N][3][M] and [W][N][M] */
int qmc_crowd_get_caches(qmc_crowd_t* crowd, void* dphi_dev, void* d2phi_dev);
/* delayed window: m[W] int32, rows[W][k] int32, V[W][k][n], C[W][k][n], Sinv[W][k][k] fp64
 * (k = delay_rank; entries at or beyond m[w] are unspecified); any pointer may be NULL      */
int qmc_crowd_get_window(qmc_crowd_t* crowd, int32_t* m_dev, int32_t* rows_dev, double* v_dev, double* c_dev,
                         double* sinv_dev);
/* everything the last move computed, one entry per walker, DEVICE, any pointer may be NULL:
 * rnew[W][3], delta[W][3], g_old[W][3], g_new[W][3], rho_d[W], rho_j[W], p[W], u[W] fp64,
 * brow[W][n] = inverse row used for the move                                               */
int qmc_crowd_get_move(qmc_crowd_t* crowd, double* rnew, double* delta, double* g_old, double* g_new, double* rho_d,
                       double* rho_j, double* p, double* u, double* brow);
int qmc_crowd_set_sweep_index(qmc_crowd_t* crowd, uint32_t s);
/* totals since create; synchronous */
int qmc_crowd_stats(qmc_crowd_t* crowd, uint64_t* proposed, uint64_t* accepted, uint64_t* flushes);
/* kernels + memset nodes this crowd has launched since create (host counter, for bench.py) */
uint64_t qmc_crowd_launch_count(const qmc_crowd_t* crowd);
/* option 0 (QMC_OPT_GRAPH): 1 = qmc_sweep replays one captured CUDA graph per sweep (default),
 * 0 = plain stream launches.                                                                */
int qmc_crowd_set_option(qmc_crowd_t* crowd, int option, int value);
#define QMC_OPT_GRAPH 0
/* option 1 (QMC_OPT_PROFILE): 1 = qmc_sweep and the step calls issue plain launches with a CUDA
 * event pair around every kernel (measurement aid for bench.py's roofline; adds event overhead,
 * so throughput numbers are never taken in this mode).                                        */
#define QMC_OPT_PROFILE 1
/* option 2 (QMC_OPT_SUBCROWDS): number of sub-crowds (1..4; 0 = automatic, the default: 2 for crowds of one to four
 * waves of window CTAs, else 1) qmc_sweep advances on separate internal
 * streams when delay_rank > 1 (crowds on independent streams overlap); walkers are independent and the
 * threads-per-walker class of the window kernel is chosen from the size of the WHOLE crowd, so results do not depend
 * on it bit for bit.  (Separate crowds of different sizes may run different classes -- 512 / 256 / 128 threads per
 * walker for W <= 148 / <= 296 / more -- whose block sums differ at the rounding level: positions and decisions still
 * agree through the fp32-quantised displacement (D:A7), inverses to ~1e-13.)  The sub-crowds are forked from and joined
 * back into desc.stream every sweep.                                                                              */
#define QMC_OPT_SUBCROWDS 2
/* option 3 (QMC_OPT_RECOMPUTE_EVERY): qmc_sweep / qmc_sweep_host call qmc_recompute_inverse after every `value`-th
 * sweep (counted on the crowd's sweep index, so the schedule does not depend on how sweeps are batched into calls);
 * 0 = never (default).                                                                                          */
#define QMC_OPT_RECOMPUTE_EVERY 3
/* option 4 (QMC_OPT_STRIP_ROWS): rows of the inverse a warp of the flush strip kernel owns: 0 = automatic (default: 32 for
 * fp64-stored inverses with ns % 32 == 0, a delay rank >= 16 and a crowd of at least two waves of 32-row strips, else 16),
 * 16 or 32 = forced where the shape allows it (32 needs ns % 32 == 0, fp64 storage and a delay rank >= 16; otherwise 16
 * is used).  Both kernels compute the same update (rounding-level differences); tests force each one. */
#define QMC_OPT_STRIP_ROWS 4

/* kernel classes of the hot path, index into qmc_crowd_get_profile's arrays */
enum {
  QMC_K_ROW_PROPOSE = 0, /* inverse row with window applied + G_k(R) + proposal (step a0)        */
  QMC_K_SPLINE_VGL = 1,  /* tricubic B-spline value/gradient/Laplacian (step a1)                 */
  QMC_K_RATIO_GRAD = 2,  /* determinant + Jastrow ratio and gradient (step a2)                   */
  QMC_K_ACCEPT = 3,      /* Metropolis decision, cache update, window append (steps a3, a4')     */
  QMC_K_RANK1 = 4,       /* Sherman-Morrison rank-1 update (step a4)                             */
  QMC_K_FLUSH = 5,       /* delayed rank-k flush, FP64 DMMA (step a5)                            */
  QMC_K_RATIO_ACCEPT = 6,/* qmc_sweep, delay_rank 1, large n: ratio_grad + accept of electron k  */
  QMC_K_WINDOW = 7,      /* qmc_sweep: all moves of one delay window (or, delay_rank 1 and small n, of a sweep), CTA per walker */
  QMC_K_KINETIC = 8,     /* qmc_kinetic_energy                                                   */
  QMC_K_BRANCH = 9,      /* qmc_crowd_branch, qmc_crowd_export / import_walkers (state copies)   */
  QMC_N_KERNEL_CLASSES = 10
};
/* Device time (ms, CUDA events on desc.stream) and launch count per kernel class accumulated in
 * profile mode since the previous call; resets the accumulators.  Synchronous.  ms and count
 * are HOST arrays of QMC_N_KERNEL_CLASSES entries (either may be NULL).                       */
int qmc_crowd_get_profile(qmc_crowd_t* crowd, double* ms, uint64_t* count);

/* ---- an entry point that allocates nothing and needs no crowd and no workspace -------------------
 * For callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): the orbital evaluation of qmc_spo_vgl step (c) -- D:C1, the 4x4x4 tricubic B-spline stencil, value /
 * gradient / laplacian of all M orbitals -- at n_pos caller-given positions, with the kernel's internal result buffer
 * ([n_pos][5][ns] table elements, ns = M rounded up to 16) in a file-scope `static __device__` array of
 * QMC_STATIC_SCRATCH_BYTES instead of a workspace.  Every GPU that loads the library holds that array until exit.
 *   n_orb, grid, box, coef_dtype, coefs_dev, orb_stride: the table, as in qmc_crowd_desc (coefs_dev DEVICE, BORROWED);
 *   r_dev:  DEVICE [n_pos][3] fp64, not wrapped (periodicity comes from the index arithmetic, D:C1);
 *   phi / dphi / d2phi: optional DEVICE outputs (NULL to skip), element type = table type, compact layouts
 *           [n_pos][M], [n_pos][3][M], [n_pos][M] -- the layouts and the values of qmc_spo_vgl's outputs;
 *   stream: cudaStream_t, BORROWED; the call is asynchronous on it.
 * Returns QMC_ERR_WORKSPACE (and launches nothing) when n_pos * 5 * ns * sizeof(element) exceeds
 * QMC_STATIC_SCRATCH_BYTES, QMC_ERR_INVALID_ARG for a malformed table description or NULL inputs; n_pos == 0 is a no-op.
 * Calls no cudaMalloc / cudaFree and no allocating library routine (the first call on a device looks the array's device
 * address up with cudaGetSymbolAddress, once per device).  ALL calls of a process on one device share the one array:
 * calls that overlap on the GPU (different streams, or graphs replayed concurrently) race; serialise them.  The array
 * keeps the last call's contents; every element a call reads it has written itself first, so nothing needs clearing. */
#define QMC_STATIC_SCRATCH_BYTES (4u << 20)
int qmc_spo_vgl_static(int32_t n_orb, const int32_t* grid /*[3]*/, const double* box /*[3]*/, int32_t coef_dtype,
                       const void* coefs_dev, int64_t orb_stride, int32_t n_pos, const double* r_dev,
                       void* phi, void* dphi, void* d2phi, void* stream);

const char* qmc_last_error(void); /* thread-local, never NULL */
const char* qmc_version(void);

#ifdef __cplusplus
}
#endif
#endif
