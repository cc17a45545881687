/* kldi.h — C ABI of the block-filtered Kohn-Sham EXC contraction library (B200 / sm_100a, FP64).
 *
 * Method: KerneLDI, arxiv/paper_2605_10363 (cited below as PAPER.md:<line>).  The library
 * computes, on ONE GPU, the hot path of exchange-correlation (EXC) grid integration written as
 * block-structured matrix products (Eq. 1-6):
 *
 *     Phi(g,mu) = chi_mu(r_g)                                  (Eq. 2)
 *     X = Phi D,   rho(g) = sum_mu Phi(g,mu) X(g,mu)           (Eq. 4)
 *     V = Phi^T diag(w v_xc) Phi                               (Eq. 3/5; b = 1)
 *
 * restricted to the block pairs that survive the block-level filter max|Phi_pq| >= eps
 * (Eq. 11-14) and the executable-pair test a_pq*b_qr >= eps (Eq. 17-19,
 * PAPER.md:195-216), stored in row- and column-oriented block-compressed layouts (BCS(R)/BCS(C),
 * PAPER.md:176-191, 459-471).  A "grid block" p is 128 consecutive points of the grid sorted along a
 * space-filling curve (the Hilbert index of Eq. 20's lattice coordinates; kldi_grid_key); an "AO
 * block" q is one shell (AO-shell partition).
 *
 * Conventions (all calls):
 *   - "host" pointers are ordinary CPU memory; "dev" pointers are CUDA device memory on the
 *     device that was current when the plan was created.  The caller owns every buffer it
 *     passes; the library neither frees nor keeps caller pointers after a call returns.
 *   - AO order at the boundary: shells in the order given, Cartesian components in the order
 *     s | x,y,z | xx,xy,xz,yy,yz,zz; every component is individually normalised (<chi|chi> = 1
 *     for an uncontracted shell with coef = 1).  Grid order: the caller's.  Every internal
 *     permutation (curve order of points, spatial order of atoms/shells) is undone before
 *     results are written.
 *   - Matrices are row-major, FP64.  D must be symmetric.
 *   - All work is enqueued on the CUDA stream given to kldi_plan_create.  Calls are
 *     asynchronous on that stream unless stated otherwise.
 *   - Every function returns a kldi_status; on failure kldi_last_error() (thread-local) holds a
 *     message, outputs are unspecified and the plan remains usable.  No exceptions, no aborts,
 *     no CPU fallback: without a CUDA device every compute call returns KLDI_ECUDA.
 */
#ifndef KLDI_H_
#define KLDI_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct kldi_plan kldi_plan; /* opaque; owns all of its device memory */

typedef enum { KLDI_OK = 0, KLDI_EINVAL = -1, KLDI_ENOMEM = -2, KLDI_ECUDA = -3, KLDI_ESTATE = -4 } kldi_status;

/* Exchange functionals, spin-restricted (b = 1):
 *   KLDI_LDA_SLATER: e = -C_x rho^{4/3}, C_x = (3/4)(3/pi)^{1/3}
 *   KLDI_GGA_PBEX  : e = -C_x rho^{4/3} F(s), F = 1 + kappa - kappa/(1 + mu s^2/kappa),
 *                    s^2 = |grad rho|^2 / (4 (3 pi^2)^{2/3} rho^{8/3}), kappa = 0.804, mu = 0.21951
 * Points with rho < 1e-20 contribute nothing (e = v = 0). */
typedef enum { KLDI_LDA_SLATER = 0, KLDI_GGA_PBEX = 1 } kldi_functional;

typedef struct {
  int32_t n_atoms;
  const double* xyz; /* host, [n_atoms][3], bohr */
} kldi_atoms;

/* Contracted Cartesian Gaussian shells:
 *   chi(r) = sum_i coef[i] N_i (x-Ax)^a (y-Ay)^b (z-Az)^c exp(-alpha[i] |r-A|^2),  a+b+c = l,
 *   N_i = (2 alpha_i/pi)^{3/4} (4 alpha_i)^{l/2} / sqrt((2a-1)!!(2b-1)!!(2c-1)!!).            */
typedef struct {
  int32_t n_shells;
  const int32_t* atom;      /* host, [n_shells] index into kldi_atoms */
  const int32_t* l;         /* host, [n_shells] 0, 1 or 2 (1, 3, 6 Cartesian components) */
  const int32_t* nprim_off; /* host, [n_shells+1] offsets into alpha / coef */
  const double* alpha;      /* host, exponents > 0 */
  const double* coef;       /* host, coefficients of the NORMALISED primitives */
} kldi_shells;

typedef struct {
  int64_t n_pts;
  const double* xyz; /* host, [n_pts][3], bohr */
  const double* w;   /* host, [n_pts] quadrature weights (may contain zeros) */
} kldi_grid;

/* Counters of a plan and of its most recent contraction calls. */
typedef struct {
  int64_t n_pts;            /* grid points given */
  int64_t n_blocks;         /* grid blocks of 128 (last one padded with zero-weight points) */
  int64_t n_blocks_nonempty;/* grid blocks that retain at least one AO block */
  int32_t n_ao;
  int32_t n_shells;         /* = number of AO blocks per grid block before filtering */
  int32_t n_atoms;
  int32_t want_gradients;
  int64_t retained_blocks;  /* |S_A|: retained (grid block, AO block) pairs (Eq. 13) */
  int64_t candidate_blocks; /* n_blocks * n_shells */
  int64_t sum_k;            /* sum_p K_p, K_p = retained AO columns of grid block p (unpadded) */
  int64_t sum_k_pad;        /* same with each K_p padded to a multiple of 8 */
  int64_t max_k;            /* max_p K_p */
  int64_t phi_bytes;        /* device bytes of the stored Phi (and gradient) tiles */
  int64_t workspace_bytes;  /* other device bytes owned by the plan */
  double flops_rho_useful;  /* sum_p 2*128*K_p^2: retained-block FLOPs of one rho build without symmetry (GGA form) */
  double flops_rho_exec;    /* FLOPs the GGA-form rho kernel issues (K_p padded to 8) */
  double flops_v_useful;    /* LDA: sum_p 128*K_p*(K_p+1) (q<=r only); GGA: sum_p 2*128*K_p^2 */
  double flops_v_exec;      /* FLOPs the V kernel issues (the 8 x 8 blocks of its schedule, K_p padded to 8) */
  double flops_dense;       /* 2*n_pts*n_ao^2 : one dense product */
  double plan_seconds;      /* wall time of kldi_plan_create */
  double eps;
  double flops_rho_useful_sym; /* sum_p 128*K_p*(K_p+1): the LDA rho build, which uses D = D^T */
  double flops_rho_exec_sym;   /* FLOPs the LDA-form (triangular D) rho kernel issues */
  double flops_v_crit;         /* V kernel: 4 scheduler partitions x the busiest partition's units per pass, summed (schedule imbalance) */
  int64_t pair_stages_total;   /* KLDI_OPT_PAIR_TEST, last rho call: (K chunk, N tile) stages before the test; -1 = off */
  int64_t pair_stages_executed;/* ... and stages that contain an executable pair a_pq*b_qr >= eps (Eq. 17-19) */
  int64_t kernel_launches;     /* kernels of this library launched by the most recent compute call on the plan */
  double ops_rho_tc;           /* KLDI_OPT_RHO_TC: int8 operations (2 per multiply-add) one rho build issues on the tensor cores */
} kldi_stats;

/* Once per geometry: space-filling-curve reorder of the grid into blocks of 128 (Eq. 20's lattice), spatial
 * order of atoms and the AO-shell partition, AO evaluation on candidate (grid block, shell) tiles,
 * block-max filter (keep iff max|chi| >= eps, Eq. 12; with want_gradients the max also runs over the
 * three gradient components), BCS(R)/BCS(C) layouts, task lists.  eps <= 0 retains every block
 * (dense; for tests).  want_gradients: 0 = values only (LDA), 1 = values + gradients (GGA).
 * cuda_stream: a cudaStream_t (NULL = default stream) used by every later call on this plan.
 * Synchronises the stream before returning.  *out is NULL on failure. */
kldi_status kldi_plan_create(const kldi_atoms* atoms, const kldi_shells* shells, const kldi_grid* grid,
                             double eps, int want_gradients, void* cuda_stream, kldi_plan** out);
kldi_status kldi_plan_destroy(kldi_plan* plan);
kldi_status kldi_plan_stats(const kldi_plan* plan, kldi_stats* out);

/* rho[g] = sum_{mu,nu} D[mu][nu] chi_mu(r_g) chi_nu(r_g) over executable block pairs
 * (Eq. 4/18); if drho != NULL (plan needs want_gradients) also drho[c][g] = d rho / d r_c.
 *   D    dev [n_ao][n_ao]   rho  dev [n_pts]   drho  dev [3][n_pts] or NULL                        */
kldi_status kldi_eval_rho(kldi_plan* plan, const double* D, double* rho, double* drho);

/* V = Phi^T diag(wv) Phi over retained block pairs (Eq. 5/16), wv = w*v_xc supplied by the caller.
 * With gga != 0 (plan needs want_gradients): wv is [4][n_pts] with wv[0] = w v_rho,
 * wv[1+c] = 2 w v_sigma d_c rho, and V = B + B^T, B = Phi^T (1/2 wv0 Phi + sum_c wv_c d_c Phi).
 *   wv  dev [n_pts] or [4][n_pts]     V  dev [n_ao][n_ao], overwritten, exactly symmetric          */
kldi_status kldi_build_vxc(kldi_plan* plan, const double* wv, int gga, double* V);

/* The LDA/GGA driver: rho (and grad rho) -> functional -> E_xc = sum_g w_g e_g and V.
 *   D dev [n_ao][n_ao];  Exc HOST, one value, valid on return (the call synchronises the stream);
 *   V dev [n_ao][n_ao] or NULL (energy only).                                                    */
kldi_status kldi_exc(kldi_plan* plan, const double* D, kldi_functional f, double* Exc, double* V);

/* Same as kldi_exc with HOST buffers: copies D to the device, runs, copies V back (end-to-end
 * timing; D_host/V_host should be page-locked for full PCIe speed but need not be).  D is symmetric and only its
 * lower triangle (row >= column) is read, here and in every other call: kldi_exc_host uploads just that half. */
kldi_status kldi_exc_host(kldi_plan* plan, const double* D_host, kldi_functional f, double* Exc,
                          double* V_host);

/* Device times (ms) of the stages of the most recent kldi_exc / kldi_eval_rho / kldi_build_vxc on
 * this plan, measured with CUDA events on the plan's stream.  Synchronises.  out[8] HOST:
 *   [0] D permute + block maxima  [1] rho contraction  [2] functional + energy  [3] wv gather / Z build
 *   [4] V contraction  [5] V finalise  [6] total  [7] reserved                                   */
kldi_status kldi_last_timings(kldi_plan* plan, double* out);

/* Inspection of the plan's index structures (tests of Eq. 20 / BCS invariants).  Copies array
 * `which` to host memory `buf` (capacity cap_bytes), writes the byte size to *need_bytes; with
 * buf == NULL only the size is returned.  Arrays (int32 unless noted):
 *   0 perm_g       [n_blocks*128] caller index of sorted point i, -1 for padding
 *   1 row_ptr      [n_blocks+1]   BCS(R): retained AO blocks of grid block p are col_idx[row_ptr[p]..)
 *   2 col_idx      [retained]     AO block (shell, in the plan's spatial shell order), increasing
 *   3 col_ptr      [n_shells+1]   BCS(C): grid blocks retaining AO block q are row_idx[col_ptr[q]..)
 *   4 row_idx      [retained]     grid block, increasing
 *   5 pos          [retained]     BCS(C) -> BCS(R) position of the same block
 *   6 shell_perm   [n_shells]     caller shell index of plan shell q
 *   7 ao_perm      [n_ao]         caller AO index of plan AO i
 *   8 grid_keys    [n_blocks*128] uint64, sorted kldi_grid_key values (padding = 2^63)
 *   9 block_amax   [retained]     float64, a_pq = max|Phi_pq| in BCS(R) order (with want_gradients the max also runs
 *                                 over the three gradient tiles, the filter's quantity)
 *  10 panel_off    [n_blocks+1]   int64, first packed column of grid block p in the Phi store
 *  11 blk_col0     [retained]     packed column (within its panel) where the block starts       */
kldi_status kldi_plan_export(const kldi_plan* plan, int which, void* buf, int64_t cap_bytes,
                             int64_t* need_bytes);

/* Copies the stored Phi tile (c = 0) or gradient tile (c = 1..3) of BCS(R) entry `entry` to host
 * memory: out[k][128] for the block's columns k (column-major tile, 128 sorted points each). */
kldi_status kldi_plan_export_tile(const kldi_plan* plan, int64_t entry, int c, double* out,
                                  int64_t cap_bytes, int32_t* width);

/* Meta-GGA contractions (the paper's functional class, PAPER.md:270 — the functional itself is not
 * part of the library): the density build and the V accumulation (Eq. 4 / Eq. 5) with the stored AO
 * gradients in place of Phi, over the same retained block pairs.  Both need want_gradients = 1 (else KLDI_ESTATE).
 *   kldi_eval_tau  : tau[g] = 1/2 sum_{mu,nu} D_{mu,nu} grad chi_mu(r_g) . grad chi_nu(r_g);  D dev [n_ao][n_ao]
 *                    symmetric, tau dev [n_pts], caller grid order, overwritten.
 *   kldi_build_vtau: V = 1/2 sum_c (d_c Phi)^T diag(wv_tau) (d_c Phi), wv_tau = w * v_tau dev [n_pts];  V dev
 *                    [n_ao][n_ao], overwritten, exactly symmetric (add it to the V of kldi_build_vxc).  Accumulation
 *                    follows KLDI_OPT_DETERMINISTIC_V (1 runs as 2).
 * Asynchronous on the plan's stream. */
kldi_status kldi_eval_tau(kldi_plan* plan, const double* D, double* tau);
kldi_status kldi_build_vtau(kldi_plan* plan, const double* wv_tau, double* V);

/* EXC nuclear-gradient contraction (the paper's second workload; it prints no formula, so this is
 * the chain rule on E_xc = sum_g w_g e(rho_g, |grad rho_g|^2), DESIGN.md §3 reading G1): at fixed D and FIXED quadrature
 * (points and weights do not follow the atoms, no grid response), with X = Phi D and X^d = d_d Phi D,
 *   KLDI_LDA_SLATER: grad[A][c] = -2 sum_g w_g v_rho sum_{mu on A} d_c Phi_{g,mu} X_{g,mu}
 *   KLDI_GGA_PBEX  : grad[A][c] = -2 sum_g sum_{mu on A} { wv0 d_c Phi X + sum_d wv_d [ d_c d_d Phi X + d_c Phi X^d ] },
 *                    wv0 = w v_rho, wv_d = 2 w v_sigma d_d rho (AO second derivatives are evaluated on the fly)
 * over the retained (grid-block, AO-shell) pairs.  Other functionals -> KLDI_EINVAL; the plan must hold the gradient
 * stores (want_gradients = 1, else KLDI_ESTATE).  D: DEVICE [n_ao][n_ao] row-major, symmetric.  grad: DEVICE
 * [n_atoms][3], caller atom order, overwritten.  Exc: HOST, may be NULL.  The first call allocates an X store of the size
 * of one Phi store (GGA: four), owned by the plan.  Synchronises before it returns.
 * kldi_last_timings: rho = the X / rho builds, vxc = the gradient contraction. */
kldi_status kldi_exc_grad(kldi_plan* plan, const double* D, kldi_functional f, double* Exc, double* grad);

/* Options of a plan (kldi_plan_set_option returns KLDI_EINVAL for an unknown option).
 * KLDI_OPT_DETERMINISTIC_V: how the V contraction adds each grid block's Gram tile into V.  2 (default) = every
 * contribution is added as a 64-bit fixed-point integer (red.global.add.u64): integer addition is associative, so V is
 * bitwise reproducible and no FP64 atomic is used; the scale is the power of two that keeps every partial sum below
 * 2^61, from a per-call bound max_q sum_p (sum_{g in p} |wv_g|) a_pq^2 >= |V_ij| (Eq. 11 block maxima a_pq;
 * Cauchy-Schwarz); a contribution is rounded once, to 2^-61 of that bound, and the sum itself is exact.  0 =
 * red.global.add.f64 (order-dependent rounding, ~1e-16 relative; 2 % faster).  1 = the tiles go to a workspace
 * (allocated on first use, about 4 n_blocks K_p^2 bytes) and are summed per AO row in a fixed order, the per-AO-block
 * reduction of PAPER.md:222 (bitwise reproducible, several times slower).  Other values -> KLDI_EINVAL.
 * KLDI_OPT_PAIR_TEST: 0 (default) = the rho contraction executes every retained pair (E = I, the conservative
 * superset); 1 = per call, b_qr = max|D_qr| is formed for every AO-shell pair and a (32-column K chunk, N tile)
 * stage of the rho kernel runs only if it contains a pair with a_pq * b_qr >= eps (Eq. 17-19, t_d = eps); costs
 * one pass over D and one over the retained-pair lists per call, pays off for a localised D.
 * KLDI_OPT_RHO_DFMA: 0 (default) = the LDA rho contraction runs on FP64 tensor-core DMMA tiles; 1 = on the vector FP64
 * pipe with register tiles (experimental and currently SLOWER, 6.1 vs 3.8 ms on cfg3: DMMA.8x8x4 tops out at 80 % of
 * the FP64 unit rate on B200 and DFMA does not, but register tiles that fit the register file are bound by the
 * shared-memory wavefront rate);
 * same result to rounding, rho still bitwise reproducible; ignored while KLDI_OPT_PAIR_TEST is on and for GGA.
 * KLDI_OPT_RHO_TC: 0 (default) = FP64 DMMA tiles; 1 = the LDA rho contraction runs as int8 slice products on the
 * 5th-generation tensor cores (tcgen05.mma kind::i8, int32 accumulators in tensor memory, the paper's
 * low-precision Tensor-Core multiplier, with error compensation): Phi (row scale, at first
 * use) and D' (column scale, per call) are split into five signed base-256 digits, the 15 digit products of weight
 * >= 256^-6 are accumulated exactly, and rho is recombined in FP64.  Error ~1e-10 absolute on rho (same parity bar,
 * 1e-9); rho stays bitwise reproducible.  Costs a second store of 5 bytes per retained Phi value and n_ao^2 64-bit
 * words.  kldi_eval_tau follows the option too (its three builds on the gradient stores; three more digit stores).
 * kldi_exc_grad runs its X-only builds (LDA: X = Phi D; GGA: the three X^d = d_d Phi D; full D) the same way.  Ignored by
 * the GGA rho contraction of kldi_exc / kldi_eval_rho and while KLDI_OPT_PAIR_TEST is on; KLDI_ESTATE from the compute
 * call if a grid block retains more than 16384 AO columns.
 * KLDI_OPT_HOST_V_TRIANGLE: 0 (default) = kldi_exc_host fills all of V_host; 1 = only its lower triangle (row >= column,
 * the convention D is read in), in row bands: V is exactly symmetric, so the other half is redundant and the
 * device-to-host copy halves. */
typedef enum { KLDI_OPT_DETERMINISTIC_V = 1, KLDI_OPT_PAIR_TEST = 2, KLDI_OPT_RHO_DFMA = 3, KLDI_OPT_RHO_TC = 4,
               KLDI_OPT_HOST_V_TRIANGLE = 5 } kldi_option;
kldi_status kldi_plan_set_option(kldi_plan* plan, kldi_option option, int value);

/* FP64 tensor-pipe microbenchmark: every SM issues dependent-free DMMA.8x8x4 for `iters`
 * iterations; returns achieved TFLOP/s (device-timed) in *tflops.  kind 0 = DMMA, 1 = DFMA,
 * 2 = 16 DMMA + 64 DFMA per iteration (do the tensor and the vector FP64 instructions share a pipe?). */
kldi_status kldi_fp64_peak(int kind, int iters, double* tflops);

/* Eq. 20 as the plan applies it, on the host, no GPU needed: the 60-bit key
 * m = sum_k z_k 2^{3k} + y_k 2^{3k+1} + x_k 2^{3k+2} of trunc(128*(xyz - origin)) per axis, each clamped
 * to [0, 2^20-1].  xyz, origin: HOST [3]. */
uint64_t kldi_morton_key(const double* xyz, const double* origin);

/* The key the plan sorts the grid points (and the atoms) by, on the host, no GPU needed: the Hilbert-curve index of the
 * same three 20-bit lattice coordinates as Eq. 20 (Skilling's transform, then Eq. 20's bit interleave) — SURVEY.md
 * §8(f1): no jumps along the curve, so blocks of 128 consecutive points are more compact than with the Z-order and
 * retain fewer AO shells.  The order is internal; results do not depend on it.  xyz, origin: HOST [3]. */
uint64_t kldi_grid_key(const double* xyz, const double* origin);
/* The same key for n points at once (host only): xyz HOST [n][3], keys HOST [n].  Used by the multi-GPU partition
 * (contiguous ranges of the plan's curve order). */
kldi_status kldi_grid_keys(const double* xyz, int64_t n, const double* origin, uint64_t* keys);

/* Host only, no GPU needed: the V-contraction schedule the plan builds for a packed panel of nb column blocks
 * of 8 (square = 0: LDA, strips on and above the diagonal; 1: GGA, full square).  passes: [cap][8] int32
 * {c1_lo, c1_n, c2_lo, c2_n, max_load (of a warp), units, smsp_load (max over the 4 scheduler partitions w % 4), n_warps | n_slots << 8}; items: [cap][32][2] int32 (item
 * warp * n_slots + slot of the pass, the rest zero: a = a_slot | b_slot << 10 | nj << 20 | diag << 24, b = arow | bcol << 16; loads and units count 8x8 blocks).  *n_passes is always set; nothing is written
 * if cap < *n_passes.  For tests of the host logic. */
kldi_status kldi_vsched_export(int nb, int square, int32_t* passes, int32_t* items, int64_t cap, int64_t* n_passes);

/* Host only: element offset (in doubles) of (column col, grid row row) of a K8-column panel that starts at packed
 * column panel_off in the V layout (4 slabs of 32 rows, [col][32] each, 16-byte chunks XOR-swizzled by col & 7). */
int64_t kldi_vlayout_offset(int64_t panel_off, int32_t K8, int32_t col, int32_t row);

/* Overlap-signature ordering of the AO blocks (Eq. 8-10, Eq. 21),
 * host only, no GPU needed: the overlap matrix S in closed form, signatures = rows of the atom-block norms
 * T_AB = ||S_AB||_F (the clustered unit is the centre: its shells are the AO blocks and stay together), cosine distance
 * d(A,B) = 1 - s_A.s_B/(|s_A||s_B|), agglomerative clustering with average linkage, the two sub-trees of every merge
 * oriented so that the closest of their end leaves become adjacent; order[r] = caller atom at position r.  mode must be
 * 1.  dist: HOST [n_atoms][n_atoms] cosine distances or NULL.  At most 4096 centres (KLDI_EINVAL beyond). */
kldi_status kldi_ao_order(const kldi_atoms* atoms, const kldi_shells* shells, int mode, int32_t* order, double* dist);

/* Process-wide defaults of plans created afterwards.  KLDI_DEFAULT_AO_ORDER: order of the atoms (and so of the AO
 * blocks) inside the plan: 0 (default) = along the same space-filling curve as the grid; 1 = kldi_ao_order's
 * overlap-signature clustering (falls back to 0 beyond 4096 centres); 2 = the caller's order.  The order is internal:
 * results do not depend on it (tested); with per-shell filtering and packed panels it does not change K_p either, only
 * the locality of the D gather and of the V scatter. */
typedef enum { KLDI_DEFAULT_AO_ORDER = 1 } kldi_plan_default;
kldi_status kldi_set_plan_default(kldi_plan_default what, int value);

/* The functional + energy step without any allocation, for callers that cannot call cudaMalloc (CUDA graph capture,
 * serving loops, harnesses that forbid it): Slater exchange per point, spin-restricted (Eq. 1, 71 Eq. 3),
 *     wv[g] = w[g] v_rho(rho[g]),   *Exc_dev = sum_g w[g] e(rho[g]),   e = v = 0 where rho < 1e-20,
 * the same arithmetic as the functional stage of kldi_exc (a fixed reduction tree: bitwise reproducible).  No plan:
 * rho, w, wv DEVICE [n_pts] in one common point order, Exc_dev DEVICE one value; asynchronous on cuda_stream (a
 * cudaStream_t, NULL = default stream) of the CURRENT device.  The per-block partial sums live in a static device array
 * of the library (256 KB, held by every GPU that loads the library until exit), hence the limit
 * n_pts <= kldi_xc_lda_noalloc_max_pts() = 8,388,608: larger -> KLDI_EINVAL.  Calls no cudaMalloc / cudaFree.  Every call
 * on a device shares that array: it keeps the last call's contents (each call overwrites what it then reads), and calls
 * that overlap on the GPU (different streams, or graphs replayed concurrently) race on it. */
kldi_status kldi_xc_lda_noalloc(const double* rho, const double* w, int64_t n_pts, double* wv, double* Exc_dev,
                                void* cuda_stream);
int64_t kldi_xc_lda_noalloc_max_pts(void);

const char* kldi_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* KLDI_H_ */
