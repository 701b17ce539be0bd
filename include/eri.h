/* eri.h -- C ABI of liberi_b200.so: integral-direct J/K build and J/K nuclear gradient on one B200 (sm_100a).
 *
 * What is computed (citations are lines of the paper text, PAPER.md, of arxiv 2407.09700):
 *   contracted four-centre electron-repulsion integrals over Gaussian shells with l <= 6 by Rys quadrature
 *   (Eq. 1-5), digested on the fly with a density matrix into the Coulomb and exchange matrices
 *   by the six updates of Algorithm 2 lines 8-13, read as full sums:
 *       J_ij = sum_kl (ij|kl) D_kl,     K_ik = sum_jl (ij|kl) D_jl,
 *   and the first-derivative contraction of Eq. 12-15 / Algorithm 4:
 *       grad_J[A] = d/dR_A ( 1/2 sum_ijkl D_ij D_kl (ij|kl) ),   grad_K[A] = d/dR_A ( 1/2 sum_ijkl D_ik D_jl (ij|kl) )
 *   at fixed D, basis functions moving with their atoms.  Screening is the Schwarz rule of Eq. 7:
 *   a unique shell quartet is skipped iff Q_ij * Q_kl < schwarz_thr, Q_ij = max |(ab|ab)|^(1/2) over the spherical
 *   components of the two shells; schwarz_thr = 0 skips nothing.
 *
 * Conventions (DESIGN.md "Readings" R1-R3):
 *   - a primitive is the raw Cartesian Gaussian of Eq. 2; `coef` multiplies the raw primitive, the
 *     library never normalises;
 *   - atomic orbitals are real solid harmonics, unit-normalised on the sphere, m = -l..+l for every l; shells appear
 *     in input order, `ao_off` is the index of the shell's m = -l function and must equal the running sum of (2l+1);
 *   - matrices are nao x nao, row-major, FP64; units Bohr and Hartree;
 *   - D is assumed symmetric by the J/K build, the list digest and the gradient (the eight-fold list uses it, PAPER.md:68;
 *     the cooperative kernels also read density blocks through their transposes).
 *
 * Memory: every pointer says HOST or DEVICE.  The caller owns every buffer it passes; the library copies what it
 * needs and owns the plan and its workspaces.  Outputs are overwritten, not accumulated.  Device work is enqueued on
 * `cuda_stream` (a cudaStream_t passed as void*, e.g. torch.cuda.current_stream().cuda_stream); plan construction
 * also blocks the host until its own device work is done.  The *_host entry points synchronise the stream before
 * returning.
 *
 * Devices: the library binds to the CUDA device that is current at its first compute call (its Rys tables, the
 * constant-memory transform table and the kernels' shared-memory attributes live there).  Calling any compute entry point
 * while another device is current returns ERI_ERR_BAD_ARG; one process drives one GPU (multi-GPU: one process per GPU,
 * eri_plan_set_shard).  eri_plan_set_kernel_mode and eri_plan_set_tuning wait for the device, re-upload the plan's row
 * tables and block the host until that is done (rare calls, like plan creation).
 *
 * Errors: every int-returning function returns ERI_OK (0) or a negative code and never throws; the message of the
 * last failure in the calling thread is available through eri_last_error().  There is no CPU fallback: without a
 * CUDA device every compute entry point returns ERI_ERR_CUDA.
 */
#ifndef ERI_B200_H
#define ERI_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ERI_OK 0
#define ERI_ERR_BAD_ARG (-1)       /* null pointer, nprim <= 0, exponent <= 0, inconsistent ao_off / prim_off / atom */
#define ERI_ERR_UNSUPPORTED_L (-2) /* l < 0 or l > ERI_LMAX */
#define ERI_ERR_CUDA (-3)          /* any CUDA runtime failure, including "no device" */
#define ERI_ERR_NOMEM (-4)         /* host or device allocation failed */
#define ERI_LMAX 6   /* s, p, d, f, g with tuned kernels; h and i (the paper stops at g) on the generic kernels */

typedef struct { int32_t atom; int32_t l; int32_t nprim; int32_t prim_off; int32_t ao_off; } eri_shell_t;
typedef struct { double exp; double coef; } eri_prim_t;
typedef struct eri_plan eri_plan_t; /* opaque: pair data, Schwarz bounds, task lists, workspaces */

/* Totals of a plan (shell grouping, pair sets, Schwarz prescreen). */
typedef struct {
  int32_t nshell, nao, nao_cart, natm;
  int32_t n_shell_groups;     /* distinct (l, K)                                              */
  int32_t n_pair_classes;     /* pair sets |ab, KaKb} with at least one surviving pair        */
  int32_t n_quartet_classes;  /* (bra pair class, ket pair class) combinations with work      */
  int32_t launches_per_call;  /* kernels launched by one eri_plan_build_jk call               */
  int64_t pairs_total, pairs_kept;
  int64_t quartets_total;     /* unique shell quartets, nshell-pair*(nshell-pair+1)/2         */
  int64_t quartets_kept;      /* unique shell quartets with Q_ij*Q_kl >= schwarz_thr          */
  double canonical_flops;     /* DESIGN.md "FLOP model" summed over kept quartets (energy)    */
  double canonical_flops_grad;
  double plan_ms;             /* host wall time of eri_plan_create                            */
  double plan_ms_init, plan_ms_schwarz, plan_ms_pairs, plan_ms_units;   /* its parts: basis + tables; pair sets + Schwarz factors;
                                                                           prescreen, sort, grouped twins; work units + kernel selection */
} eri_stats_t;

/* One (bra pair class, ket pair class) work unit = one kernel launch. */
typedef struct {
  int32_t la, lb, lc, ld;     /* la >= lb, lc >= ld                                            */
  int32_t ka, kb, kc, kd;     /* contraction degrees                                           */
  int32_t nroots;             /* Eq. 3                                            */
  int32_t kernel;             /* 0 generic thread-per-quartet, 1 register-unrolled, 2 cooperative shared-memory, 3 tile */
  int64_t quartets;           /* kept unique quartets in this unit                             */
  int64_t slots;              /* quartet slots the unit's J/K launch covers (tile shape x blocks) >= quartets: lane efficiency */
  double canonical_flops;     /* per call                                                      */
  float last_ms;              /* device time of the unit's last launch; needs eri_plan_set_timing(plan,1)      */
  float last_ms_grad;
  int32_t kernel_grad;        /* gradient kernel of the unit: 0 generic, 2 cooperative shared-memory, 3 tile, 4 primitive-parallel */
  int32_t tile_fill_pm;       /* lane fill of the unit's tile decomposition in permille (quartets / swept lane slots; 0: no tiles) */
  double canonical_flops_grad;
} eri_class_stat_t;

/* ---- one-shot calls (north-star signatures).  shells/prims/coords HOST; D, J, K, grad_* DEVICE. ---------------- */
int eri_build_jk(const eri_shell_t* shells, int nshell, const eri_prim_t* prims, int nprim,
                 const double* coords /*HOST natm*3*/, int natm, const double* D /*DEVICE nao*nao*/,
                 double schwarz_thr, double* J /*DEVICE out*/, double* K /*DEVICE out*/, void* cuda_stream);
int eri_jk_grad(const eri_shell_t* shells, int nshell, const eri_prim_t* prims, int nprim,
                const double* coords, int natm, const double* D /*DEVICE*/, double schwarz_thr,
                double* grad_J /*DEVICE out natm*3*/, double* grad_K /*DEVICE out natm*3*/, void* cuda_stream);

/* ---- two-phase form: the plan depends on geometry, basis and threshold, not on the density. ------------------- */
int eri_plan_create(const eri_shell_t* shells, int nshell, const eri_prim_t* prims, int nprim,
                    const double* coords, int natm, double schwarz_thr, int want_grad, void* cuda_stream,
                    eri_plan_t** out);
int eri_plan_build_jk(eri_plan_t* plan, const double* D /*DEVICE*/, double* J /*DEVICE*/, double* K /*DEVICE*/,
                      void* cuda_stream);
int eri_plan_jk_grad(eri_plan_t* plan, const double* D /*DEVICE*/, double* grad_J /*DEVICE*/, double* grad_K /*DEVICE*/,
                     void* cuda_stream);
/* Density-weighted batch screening of the paper (Eq. 8-9 and Algorithm 1 lines 12-16), the step that makes
 * repeated SCF iterations cheap: J and K of D as eri_plan_build_jk, but a unique quartet of the unit
 * {ab|cd} (shell groups a, b, c, d: equal angular momentum and contraction degree) is evaluated iff
 *     Q_ij * Q_kl * min(1, P_{ab|cd}) >= schwarz_thr,   P_{ab|cd} = max |D| over the six sub-blocks of D between the groups,
 * computed per call from D on the device (no host synchronisation).  The cap at 1 keeps the kept set inside the plan's
 * Schwarz-only list.  Linear in D like the plain build, so an incremental Fock build calls it with D_new - D_old, whose
 * small elements remove most of the list.  The error against the unscreened result is bounded like the Schwarz rule's:
 * each skipped quartet contributes less than schwarz_thr per matrix element.  D, J, K DEVICE.  schwarz_thr = 0: same as
 * eri_plan_build_jk.  eri_plan_dscreen_quartets: unique quartets evaluated by the last such call (waits for it). */
int eri_plan_build_jk_dscreen(eri_plan_t* plan, const double* D /*DEVICE*/, double* J /*DEVICE*/, double* K /*DEVICE*/,
                              void* cuda_stream);
int eri_plan_dscreen_quartets(eri_plan_t* plan, int64_t* out /*HOST*/);
/* The shell-group maxima of the last eri_plan_build_jk_dscreen call (waits for it): ao_group[i] = shell group (equal l and K,
 * PAPER.md:68) of AO i, P[g * n_shell_groups + h] = max |D| over the sub-block between groups g and h (the P_{a|b} of Eq. 9).
 * ao_group HOST out nao, P HOST out n_shell_groups^2 (eri_plan_stats); either may be NULL.  ERI_ERR_BAD_ARG before the first
 * density-weighted call. */
int eri_plan_dscreen_group_max(eri_plan_t* plan, int32_t* ao_group /*HOST out*/, double* P /*HOST out*/);
/* Allocation-free form of that pass over the density (Eq. 9), for callers that cannot call cudaMalloc (CUDA
 * graph capture, serving loops, harnesses that forbid it):  P[g * ngroups + h] = max |D_ij| over AOs i of group g, j of group h.
 * D DEVICE nao*nao, ao_group DEVICE nao (entries outside 0..ngroups-1 are ignored), P DEVICE out ngroups^2; nothing else is
 * touched: the accumulators live in a static device array of ERI_NOALLOC_MAX_GROUPS^2 64-bit words (32 KB per GPU, held
 * until the process exits).  The call makes no cudaMalloc, cudaFree or other allocating call and no host synchronisation; it
 * enqueues a clear of the accumulators, the pass and the copy to P on `cuda_stream`.  ngroups > ERI_NOALLOC_MAX_GROUPS (or
 * < 0, nao < 0, a null pointer) returns ERI_ERR_BAD_ARG.  EVERY call on a device shares the one array: calls whose device
 * work may overlap (different streams, several host threads) race and give wrong maxima -- order them.  Works on whichever
 * device is current (the array exists once per device); it does not bind the library to a device. */
#define ERI_NOALLOC_MAX_GROUPS 64
int eri_density_group_max_noalloc(const double* D /*DEVICE*/, int nao, const int32_t* ao_group /*DEVICE*/, int ngroups,
                                  double* P /*DEVICE out*/, void* cuda_stream);
/* Same work with HOST buffers: H2D copy of D, build, D2H copy of the results, stream synchronised on return. */
int eri_plan_build_jk_host(eri_plan_t* plan, const double* D /*HOST*/, double* J /*HOST*/, double* K /*HOST*/,
                           void* cuda_stream);
int eri_plan_jk_grad_host(eri_plan_t* plan, const double* D /*HOST*/, double* grad_J /*HOST*/, double* grad_K /*HOST*/,
                          void* cuda_stream);
int eri_plan_stats(const eri_plan_t* plan, eri_stats_t* out);
int eri_plan_num_classes(const eri_plan_t* plan);
int eri_plan_class_stats(const eri_plan_t* plan, eri_class_stat_t* out /*HOST*/, int max_entries);
/* timing mode: a CUDA event is recorded on the stream between class launches (no host synchronisation); the per-class
 * device times of the last call are collected by the next eri_plan_class_stats, which waits for that call to end. */
int eri_plan_set_timing(eri_plan_t* plan, int on);
/* kernel selection: 0 = tuned kernels where one exists, tile family preferred (default), 1 = generic kernel everywhere
 * (reference path), 2 = tuned kernels without the tile family (register and cooperative families only) */
int eri_plan_set_kernel_mode(eri_plan_t* plan, int mode);
/* Tuning knobs of the kernel selection (measured defaults); the kernels are re-selected like
 * eri_plan_set_kernel_mode does.  The results do not depend on them beyond rounding (the test-suite uses them to run every
 * kernel family on small inputs):
 *   ERI_TUNE_TILE_FILL_SCALE  multiplies the lane-fill thresholds below which a unit is NOT given to the tile family
 *                             (default 1; 0 = tile family wherever the class is served and the HRR guard passes)
 *   ERI_TUNE_GRAD_MIN_TASKS   cooperative gradient kernel: the run of bra pairs per task (16) is halved while a unit has
 *                             fewer tasks than this (default 32768; 0 = always runs of 16)
 *   ERI_TUNE_PGRAD_MIN_NPP    primitive quartets per shell quartet (Ka Kb Kc Kd) from which a unit of a low-l class that the tile gradient
 *                             kernel does not take (or fills badly) runs on the primitive-parallel gradient kernel (default 3; 1 = wherever the class is served) */
#define ERI_TUNE_TILE_FILL_SCALE 0
#define ERI_TUNE_GRAD_MIN_TASKS 1
#define ERI_TUNE_PGRAD_MIN_NPP 2
int eri_plan_set_tuning(eri_plan_t* plan, int key, double value);
/* Multi-GPU sharding: this process evaluates only the thread blocks b with b % nranks == rank of every
 * class launch (quartets are independent units).  The outputs are then PARTIAL sums; J, K and the gradient
 * are linear in them, so the caller sums the outputs over ranks (one all-reduce).  Default rank 0 of 1. */
int eri_plan_set_shard(eri_plan_t* plan, int rank, int nranks);
void eri_plan_destroy(eri_plan_t* plan);   /* waits for the device to finish, then releases the plan's buffers */

/* ---- diagnostics / benchmark entry points -------------------------------------------------------------------- */
/* Spherical ERI blocks (ij|kl) for an explicit list of shell quartets (any order of shells).  Block n is written
 * row-major [ns_i][ns_j][ns_k][ns_l] at out + out_off[n].  quartets, out_off HOST; out DEVICE. */
int eri_compute_quartets(const eri_shell_t* shells, int nshell, const eri_prim_t* prims, int nprim,
                         const double* coords, int natm, const int32_t* quartets /*HOST n*4*/, int n,
                         double* out /*DEVICE*/, const int64_t* out_off /*HOST n*/, void* cuda_stream);
/* cfg1 micro-benchmark: every listed quartet (i,j,k,l) adds its six updates once, no symmetry
 * factor, no final symmetrisation:  Jt_ij += g D_kl, Jt_kl += g D_ij, Kt_ik += g D_jl, Kt_jl += g D_ik,
 * Kt_il += g D_jk, Kt_jk += g D_il.  A list whose quartets all belong to one canonical class (la>=lb, lc>=ld,
 * equal contraction pattern) runs on that class's tuned kernel, anything else on the generic kernel. */
int eri_digest_quartet_list(const eri_shell_t* shells, int nshell, const eri_prim_t* prims, int nprim,
                            const double* coords, int natm, const int32_t* quartets /*HOST n*4*/, int n,
                            const double* D /*DEVICE*/, double* Jt /*DEVICE out*/, double* Kt /*DEVICE out*/,
                            void* cuda_stream);
/* Two-phase form of the list digest for timing: the list plan holds pair data and the work list. */
int eri_list_plan_create(const eri_shell_t* shells, int nshell, const eri_prim_t* prims, int nprim,
                         const double* coords, int natm, const int32_t* quartets /*HOST n*4*/, int n,
                         void* cuda_stream, eri_plan_t** out);
int eri_list_plan_digest(eri_plan_t* plan, const double* D /*DEVICE*/, double* Jt /*DEVICE*/, double* Kt /*DEVICE*/,
                         void* cuda_stream);
/* Schwarz factors Q_ij (Eq. 7) for all shell pairs; Q HOST out nshell*nshell. */
int eri_schwarz(const eri_shell_t* shells, int nshell, const eri_prim_t* prims, int nprim,
                const double* coords, int natm, double* Q /*HOST out*/, void* cuda_stream);
/* Rys roots u_n = t_n^2 and weights w_n of Eq. 1 for n points x; x, u, w HOST; u, w are n*N. */
int eri_rys_roots(int nroots, const double* x /*HOST*/, int n, double* u /*HOST out*/, double* w /*HOST out*/);
/* The library's Cartesian -> real-solid-harmonic table for angular momentum l: T HOST out, ns(l) x nc(l) row-major,
 * rows m = -l..l, columns in the order lx descending then ly descending (reading R3). */
int eri_c2s_matrix(int l, double* T /*HOST out*/);
/* Sustained FP64 FMA rate of the device in TFLOP/s (denominator of "% of FP64 peak"; dependent-chain-free DFMA loop). */
int eri_measure_fp64_peak(double* tflops /*HOST out*/, void* cuda_stream);
/* Canonical FLOP count of one contracted quartet; deriv != 0: gradient count. */
double eri_canonical_flops(int la, int lb, int lc, int ld, int ka, int kb, int kc, int kd, int deriv);

/* Test diagnostics: the tuned kernel instantiations the library holds and those this process has launched so far, as
 * newline-separated "family la lb lc ld" (family: reg, coop, tile, tgrad, cgrad, pgrad; launched also: generic, generic_grad).
 * Writes at most n bytes (NUL-terminated) to buf (HOST, may be NULL) and returns the size needed. */
int eri_kernel_catalog(char* buf, int n);
int eri_kernel_launched(char* buf, int n);

const char* eri_strerror(int code);
const char* eri_last_error(void);
const char* eri_version(void);

#ifdef __cplusplus
}
#endif
#endif /* ERI_B200_H */
