/*
 * qmc_oracle.h -- ORACLE: plain, slow, obviously-correct CPU restatement of the
 * particle-by-particle electron move for a crowd of walkers.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or helper with paper_2209_14487_b200/csrc (the CUDA path) and neither
 * side includes the other.
 *
 * What it follows (P:n = /root/reference/PAPER.md line n; BJ = BASELINE.json north_star;
 * S8c = SURVEY.md section 8(c) readings, restated in DESIGN.md "Readings"):
 *   - loop structure: Alg. 1 lines 4-9 applied to all walkers of a crowd in
 *     lock-step, Alg. 3 / Alg. 4;
 *   - the arithmetic inside the loop is named by BJ (tricubic B-spline orbitals, Slater
 *     determinant ratio via the inverse row, two-body Pade Jastrow, Metropolis with a
 *     drift-diffusion proposal, Sherman-Morrison or delayed rank-k update, Philox);
 *     the paper prints no formula for any of it, so each function states the textbook
 *     definition it writes out (S8c C1..C7).
 *
 * All arithmetic is fp64, plain loops, compiled -O2 -ffp-contract=off, no BLAS/LAPACK.
 * OpenMP is used in exactly one place: the loop over walkers of oracle_crowd_sweep
 * (the shape of the paper's CPU driver, Alg. 2).
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"):
 *   philox ........ Random123 known-answer vectors (tests/golden/philox4x32_10_kat.txt)
 *   spline ........ partition of unity, linear-table closed form, cosine-table closed
 *                   form, periodicity, finite differences
 *   det ratio ..... brute-force det(A')/det(A) (numpy LU) on n <= 8
 *   SM / delayed .. full re-inversion (numpy) after every accepted move / flush
 *   Jastrow ....... two-electron closed form, full pair-sum difference, finite differences
 *   accept rule ... tau->0 limit, constant-orbital case, sampling of |phi|^2 (histogram)
 *   fp32 storage .. (mixed precision, R6) every stored element is its own fp32 rounding; with fp32-representable
 *                   inputs one update equals the fp64 update rounded once; the carried inverse stays within the
 *                   first-order bound r kappa_inf(A) 2^-24 of the exact one (tests/test_oracle_mixed.py)
 *   kinetic ....... central second differences of the brute-force Psi = det det exp(J) (numpy) on tiny systems;
 *                   free-particle and two-electron Jastrow closed forms
 *   whole sweep ... every logged move re-derived from brute-force determinants; the
 *                   paper prints no worked trajectory, so the *trajectory itself* is
 *                   "parity unpinned" by the paper (S8c T9) and pinned only through
 *                   the per-move invariants above.
 */
#ifndef QMC_ORACLE_H
#define QMC_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
  int32_t n_elec;      /* N (even): electrons [0,N/2) spin-up, [N/2,N) spin-down (S8c 8(a)) */
  int32_t n_orb;       /* M = N/2, one orbital set shared by both spins (S8c A5)          */
  int32_t grid[3];     /* Ng per axis                                                      */
  int32_t coef_dtype;  /* 0: coefs points to float, 1: to double (values used as fp64)     */
  double  box[3];      /* L per axis, orthorhombic periodic                                */
  const void* coefs;   /* [gx][gy][gz][n_orb], orbital index innermost (BJ), borrowed      */
  double  j2_a, j2_b;  /* u(r) = a r / (1 + b r)                                           */
  double  tau;         /* time step                                                        */
  uint64_t seed;       /* Philox key                                                       */
  int32_t delay_rank;  /* 1 = Sherman-Morrison, k > 1 = delayed rank-k                     */
  int32_t inverse_fp32;/* 0: the carried inverse is fp64 (BASELINE.json configs).  1: mixed precision (SURVEY.md 8(f)
                          item 3, reading R6): the carried inverse is STORED in fp32 -- every element is rounded
                          to the nearest fp32 value after each operation that writes it (inversion, rank-1 update,
                          flush) -- while every dot product and update is evaluated in fp64 on the stored values      */
} oracle_system;

/* one record per (walker, electron) move of a sweep; everything the acceptance needs */
typedef struct {
  double rnew[3];      /* proposed position r'                                  */
  double delta[3];     /* applied displacement (fp32-valued)                    */
  double g_old[3];     /* G_k(R)  = grad_k ln Psi at the current position       */
  double g_new[3];     /* G_k(R') = grad_k ln Psi at the proposed position      */
  double rho_d;        /* determinant ratio                                     */
  double rho_j;        /* Jastrow ratio                                         */
  double p;            /* acceptance probability (un-clamped)                   */
  double u;            /* uniform drawn for the decision                        */
  double disp_margin;  /* min over components of distance (in fp32 ulps) of the  */
                       /* unrounded displacement to an fp32 rounding boundary    */
  int32_t accepted;
  int32_t _pad;
} oracle_move_log;

/* ---- C7: counter-based random numbers (Philox4x32-10, Salmon et al. SC'11) ---- */
void   oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
void   oracle_rng_gauss3(uint64_t seed, uint32_t walker, uint32_t k, uint32_t sweep, double chi[3]);
double oracle_rng_uniform(uint64_t seed, uint32_t walker, uint32_t k, uint32_t sweep);

/* ---- C1: uniform tricubic B-spline orbitals ---- */
void oracle_bspline_weights(double t, double a[4], double da[4], double d2a[4]);
void oracle_spo_vgl(const oracle_system* sys, const double r[3],
                    double* phi /*[M]*/, double* dphi /*[3][M]*/, double* d2phi /*[M]*/);

/* ---- C3: two-body Jastrow ---- */
double oracle_j2_logpsi(const oracle_system* sys, const double* R /*[N][3]*/);
void   oracle_j2_usum_grad(const oracle_system* sys, const double* R, int k, const double rk[3],
                           double* usum, double grad[3]);

/* ---- kinetic part of the local energy (Alg. 1 L11; definition: lap ln Psi + |grad ln Psi|^2) ---- */
double oracle_kinetic_energy(const oracle_system* sys, const double* R /*[N][3]*/, const double* B_up /*[n][n]*/,
                             const double* B_dn, double* e_elec /*[N] or NULL*/);

/* ---- C2/C5/C6: determinants ---- */
int  oracle_lu_inverse_transpose(int n, const double* A, double* B, double* logabsdet, int* sign);
void oracle_sm_update(int n, double* B, int k, const double* phi, double rho_d);
int  oracle_delayed_row(int n, const double* B0, int m, const int32_t* rows, const double* V,
                        const double* C, int k, double* b);
int  oracle_delayed_flush(int n, double* B0, int m, const int32_t* rows, const double* V,
                          const double* C);

/* ---- C4: one move, split so tests can teacher-force each half ---- */
void oracle_move_propose(double tau, const double rk[3], const double g_old[3], const double chi[3],
                         double delta[3], double rnew[3], double* disp_margin);
int  oracle_move_accept(double tau, const double delta[3], const double g_old[3],
                        const double g_new[3], double rho_d, double rho_j, double u, double* p);

/* ---- the crowd: Alg. 1 L4-L9 over all walkers, lock-step in k ---- */
typedef struct oracle_crowd oracle_crowd;
oracle_crowd* oracle_crowd_create(const oracle_system* sys, int n_walkers, int walker_id0,
                                  const double* pos /*[W][N][3]*/, int* status);
void oracle_crowd_destroy(oracle_crowd* c);
/* runs n_sweeps full sweeps starting at sweep index *c->sweep; log may be NULL or
 * [n_sweeps][W][N] records. Returns number of accepted moves. Threads over walkers. */
int64_t oracle_crowd_sweep(oracle_crowd* c, int n_sweeps, oracle_move_log* log);
void oracle_crowd_set_sweep_index(oracle_crowd* c, uint32_t s);
/* periodic recompute: rebuilds both Slater matrices from the carried positions, inverts
 * them by LU in fp64 (then rounds to fp32 in the mixed-precision mode) and refreshes the caches; needs an empty
 * window.  Returns the LU status (0 = ok), -1 on an open window. */
int  oracle_crowd_recompute(oracle_crowd* c);
/* R6: x <- fl32(x) for the n x n carried inverse (round to nearest even, the C cast) */
void oracle_round_to_fp32(int n, double* B);
/* branching data movement: slot w <- state of slot src[w]; -1 on a bad entry / open window */
int  oracle_crowd_branch(oracle_crowd* c, const int32_t* src /*[W]*/);
void oracle_crowd_get_positions(const oracle_crowd* c, double* pos /*[W][N][3]*/);
void oracle_crowd_get_inverse(const oracle_crowd* c, int spin, double* B /*[W][n][n]*/);
int  oracle_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
