/*
 * b200md.h -- C-ABI of the B200-native single-GPU molecular-dynamics hot path.
 *
 * Implements the single-GPU engine that runs on every rank of HOOMD-blue 1.0 as described in
 * Glaser et al., "Strong scaling of general-purpose molecular dynamics simulations on GPUs"
 * (arXiv:1412.3387).  Citations "PAPER.md:<line>" refer to /root/reference/PAPER.md; "R<n>" to the
 * numbered readings in DESIGN.md (the paper prints no formulas, so each operation also names the
 * textbook definition it uses).
 *
 * Conventions
 *  - Every function returns 0 (MD_OK) or a negative md_status; md_last_error(ctx) gives the text.
 *  - Box: orthorhombic, periodic, edge lengths box[3], coordinates in [-L/2, L/2) per axis (R4).
 *  - Particles are identified by TAG = index into the caller's arrays (0..N-1).  Every array crossing
 *    this boundary is in TAG ORDER, row-major (N x 3 for vectors).  Internally particles are kept
 *    sorted by cell along a space-filling curve ("reordering of the GPU arrays").
 *  - POINTERS: every array pointer may be a HOST pointer or a CUDA DEVICE pointer; the library asks
 *    the driver (cudaPointerGetAttributes) and copies accordingly.  The caller owns every pointer it
 *    passes; the library never keeps one past the call.  Calls with device pointers only enqueue work
 *    on the context's stream; calls with a host OUTPUT pointer synchronise that stream before
 *    returning.  No torch types appear here; the Python binding passes tensor.data_ptr().
 *  - All device work runs on the stream given to md_configure (default: the legacy default stream).
 *  - Internal device memory: carved from a caller-provided workspace (md_workspace_bytes, md_set_workspace) or, without
 *    one, allocated with cudaMalloc at configure time (the neighbour list grows on demand at a rebuild).  One context
 *    per host thread; no global state.
 *  - There is NO CPU fallback: every entry point needs a CUDA device and fails with MD_ECUDA otherwise.
 */
#ifndef B200MD_H
#define B200MD_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct md_ctx md_ctx;

typedef enum {
    MD_OK = 0,
    MD_EINVAL = -1,  /* bad argument; box too small (needs floor(L/r_list) >= 3 per axis so that the 27-cell
                        stencil has no duplicate cells and r_list < L/2 for the minimum image) */
    MD_ESTATE = -2,  /* call out of order (e.g. md_build_nlist before md_set_state) */
    MD_ENOMEM = -3,  /* device allocation failed */
    MD_ECUDA = -4    /* CUDA runtime error, text in md_last_error */
} md_status;

/* arithmetic of the pair-force evaluation ("full double precision is available per compile-time
   option"; here a run-time mode, R25) */
#define MD_FP64 0   /* everything fp64 */
#define MD_MIXED 1  /* LJ pair polynomial in fp32 on fp32 separations, r<rc decision as fp64 would take it,
                       contributions accumulated in fp64 (fp32 sums of 8 consecutive list entries are widened,
                       MD_OPT_ACC_BLOCK); pairs of the first neighbour shell (every pair that can be closer than 1.5 sigma
                       before the next rebuild) are evaluated in fp64 -- fp32 cannot hold the 1e-4 force bar there (DESIGN.md
                       R25); positions, velocities, integration, cell ids, neighbour-list decisions, displacement check
                       stay fp64.  The other pair potentials, bonds and angles are fp64 in both modes */

/* internal storage order of the cells (particles are always sorted by cell; inside a cell by tag, with
   MD_ORDER_MORTON by (3-bit-per-axis sub-cell Morton key, tag): a pure function of the positions either way) */
#define MD_ORDER_LEX 0     /* x fastest, then y, then z; general list kernels (32-bit indices, L1/L2 gathers) */
#define MD_ORDER_MORTON 1  /* Z-order curve over (cx, cy, cz); enables the tile kernels: one CTA per brick of cells,
                              stencil staged in shared memory, 16-bit list entries (the fast path, default of the
                              Python binding); falls back to the general kernels if a tile exceeds shared memory */
#define MD_ORDER_HILBERT 2 /* 3-D Hilbert curve over (cx, cy, cz); general list kernels */

/* which terms md_step evaluates */
#define MD_F_LJ 1u
#define MD_F_DPD 2u
#define MD_F_BONDS 4u
#define MD_F_NVT 8u /* md_step integrates with the Nose-Hoover thermostat (md_integrate_nvt) instead of NVE */
#define MD_F_PAIR 16u   /* a pair potential of SURVEY.md 8(f) row 3 (pair_kind, pair_p) instead of LJ / DPD */
#define MD_F_ANGLES 32u /* harmonic angles (md_set_angles; angle_k, angle_theta0) */
#define MD_F_DIHEDRALS 64u /* periodic dihedrals (md_set_dihedrals; dihedral_k, dihedral_sign, dihedral_n) */
#define MD_F_LANGEVIN 128u /* Langevin thermostat as a one-body force (langevin_gamma, langevin_kT, langevin_seed; R36) */
#define MD_F_MTK 256u /* md_step integrates NVT with the Martyna-Tobias-Klein update (nvt_kT, nvt_tau; R39) instead of NVE */

/* pair potentials of md_forces_pair / MD_F_PAIR (PAPER.md:63 lists them, R31); parameters p[0..2] */
enum { MD_PAIR_LJ = 0,       /* U = 4 p0 ((p1/r)^12 - (p1/r)^6)                        p0 = epsilon, p1 = sigma     */
       MD_PAIR_YUKAWA = 1,   /* U = p0 exp(-p1 r) / r                                  p0 = epsilon, p1 = kappa     */
       MD_PAIR_GAUSSIAN = 2, /* U = p0 exp(-r^2 / (2 p1^2))                            p0 = epsilon, p1 = sigma     */
       MD_PAIR_MORSE = 3,    /* U = p0 (exp(-2 p1 (r - p2)) - 2 exp(-p1 (r - p2)))     p0 = D0, p1 = alpha, p2 = r0 */
       MD_PAIR_TABLE = 4 };  /* the table of md_set_pair_table, linear interpolation (R37); p unused, no energy shift */
/* bond potentials (R19, R33) */
enum { MD_BOND_HARMONIC = 0, /* U = k/2 (r - r0)^2 */
       MD_BOND_FENE = 1,     /* U = -1/2 k r0^2 ln(1 - (r/r0)^2), r < r0 (r >= r0: NaN, the bond is broken) */
       MD_BOND_TABLE = 2 };  /* the table of md_set_bond_table, linear interpolation (R38); bond_k, bond_r0 unused */

/* scheduling of md_step */
#define MD_SCHED_SYNC 0        /* the host waits for the rebuild flag of half 1 before it enqueues the forces */
#define MD_SCHED_SPECULATIVE 1 /* default: forces are enqueued before the flag arrives whenever no rebuild is predicted
                                  (PAPER.md:122); if the flag says "rebuild" they are discarded and evaluated again on
                                  the new list.  Results are identical in both modes */
#define MD_SCHED_BATCH 2       /* no host round trip per step (launch overhead at small N): the kernels of
                                  a batch of steps are enqueued ahead, each gated on a device-side flag; when half 1 of a
                                  step fires the criterion, everything enqueued after it returns at once and the host,
                                  which reads the flag once per batch, rebuilds and resumes from that step.  Same kernels
                                  on the same data: results identical to the other two modes */

typedef struct {
    uint32_t flags;      /* MD_F_* */
    int32_t lj_energy_shift;
    double dt;
    double lj_epsilon, lj_sigma;
    double dpd_A, dpd_gamma, dpd_kT;
    uint64_t dpd_seed;
    double bond_k, bond_r0;
    double nvt_kT, nvt_tau; /* MD_F_NVT: target temperature (k_B T0) and thermostat period tau */
    int32_t pair_kind;      /* MD_F_PAIR: MD_PAIR_*; the energy shift is lj_energy_shift */
    int32_t bond_kind;      /* MD_F_BONDS: MD_BOND_* (0 = harmonic) */
    double pair_p[4];       /* MD_F_PAIR: parameters of the pair potential */
    double angle_k, angle_theta0; /* MD_F_ANGLES: U = k/2 (theta - theta0)^2, theta0 in radians */
    double dihedral_k;            /* MD_F_DIHEDRALS: U = k/2 (1 + sign cos(n phi)) */
    int32_t dihedral_sign, dihedral_n; /* sign = +1 or -1, n = 1, 2, 3, ... */
    double langevin_gamma, langevin_kT; /* MD_F_LANGEVIN: friction coefficient and k_B T of the bath */
    uint64_t langevin_seed;
} md_step_desc;

#define MD_N_KERNELS 8
enum { MD_K_NLIST = 0, MD_K_LJ = 1, MD_K_DPD = 2, MD_K_BONDS = 3, MD_K_INTEGRATE = 4, MD_K_CELLS = 5 };

typedef struct {
    uint64_t steps;             /* time steps taken by md_step since create */
    uint64_t rebuilds;          /* neighbour-list builds (md_build_nlist calls + rebuilds inside md_step) */
    uint64_t dangerous_builds;  /* rebuilds at which some particle had moved more than r_buff (not r_buff/2)
                                   since the last build: with a check every step this must stay 0 */
    uint64_t nlist_entries;     /* entries of the current full (double-sided) list */
    uint64_t nlist_capacity;    /* entries allocated */
    uint64_t device_bytes;      /* device memory owned by the context */
    double mean_neighbors;      /* nlist_entries / N */
    uint32_t dims[3];           /* cell grid */
    uint32_t max_cell_count;    /* most populated cell at the last build */
    int32_t block[MD_N_KERNELS];    /* launch parameters chosen by the tuner, per kernel */
    int32_t w[MD_N_KERNELS];        /* threads per particle, per kernel */
    float tuned_us[MD_N_KERNELS];   /* median time of the chosen setting when it was tuned */
    uint32_t tuner_runs;        /* number of tuning sweeps performed */
    uint32_t launches;          /* kernel launches issued by this context since create (all entry points) */
    double stage_ms[MD_N_KERNELS];          /* with md_set_profiling(ctx,1): device time per stage (CUDA events on */
    uint64_t stage_launches[MD_N_KERNELS];  /* the context's stream), accumulated since profiling was switched on  */
    uint64_t speculative_forces;            /* force evaluations enqueued before the rebuild flag was known ...     */
    uint64_t wasted_forces;                 /* ... and how many of them were discarded because a rebuild was due    */
    double r_buff;                          /* the skin in use (md_create's, or the one md_tune_rbuff chose)         */
    double rbuff_tuned_tps;                 /* time steps per second of that skin in md_tune_rbuff's burst (0: never tuned) */
} md_stats;

/* ---- lifetime ------------------------------------------------------------------------------------------ */

/* Neighbour problem of PAPER.md:79 / Fig. 1: N particles in a periodic box, pair cut-off rc
   and buffer ("skin") r_buff; the list radius is r_list = rc + r_buff.  box: HOST pointer to 3 doubles.
   Fails with MD_EINVAL unless floor(box[a]/r_list) >= 3 on every axis. */
int md_create(md_ctx **out, const double box[3], uint64_t N, double rc, double r_buff);

/* Device memory from the caller (north_star: "PyTorch used only for device memory and streams").
   md_workspace_bytes: an upper estimate of everything a context of this problem allocates -- state and its reorder twins,
   cell and tile tables, the neighbour list at 1.5x the stride its density suggests, the exact 32-bit copy that the list
   exports build, staging for host-pointer arguments, a bond table of up to 2 bonds per particle.  box, bytes: HOST.
   md_set_workspace: right after md_create (MD_ESTATE once anything is allocated); `workspace` is a DEVICE pointer the caller
   owns and keeps alive until md_destroy.  Every internal buffer is then carved from it (first fit, 256-byte blocks;
   buffers that grow -- a longer row stride at a rebuild, a larger export -- are re-carved); a request that does not fit
   returns MD_ENOMEM with the missing bytes in md_last_error, nothing is allocated behind the caller's back.  Without
   this call the context allocates with cudaMalloc.  Results are bit-identical either way. */
int md_workspace_bytes(const double box[3], uint64_t N, double rc, double r_buff, int precision, uint64_t *bytes);
int md_set_workspace(md_ctx *ctx, void *workspace, uint64_t bytes);

/* precision: MD_FP64 | MD_MIXED.  stream: a cudaStream_t (as void*), NULL = default stream.
   order: MD_ORDER_*.  sched: MD_SCHED_*.  May be called again before md_set_state. */
int md_configure(md_ctx *ctx, int precision, void *stream, int order, int sched);

/* Releases every device buffer.  ctx is invalid afterwards. */
int md_destroy(md_ctx *ctx);

const char *md_last_error(md_ctx *ctx); /* static/ctx-owned string; valid until the next call on ctx */

/* ---- state (tag order) --------------------------------------------------------------------------------- */

/* pos, vel: N x 3 doubles.  mass: N doubles or NULL (= 1).  Positions are wrapped into the box once and the
   periodic image counters reset to 0 (R4).  step0 is the time-step counter of this state (enters the DPD hash).
   Invalidates cells, neighbour list and forces. */
int md_set_state(md_ctx *ctx, const double *pos, const double *vel, const double *mass, uint64_t step0);

/* Bonds as unordered tag pairs.  Stored per particle so that each particle sums its own bonds
   without atomics.  n_bonds = 0 clears.  A particle may have any number of bonds. */
int md_set_bonds(md_ctx *ctx, const uint32_t *tag_a, const uint32_t *tag_b, uint64_t n_bonds);

/* pos, vel: N x 3 doubles (wrapped positions); image: N x 3 int32 or NULL.  Any of the three may be NULL. */
int md_get_state(md_ctx *ctx, double *pos, double *vel, int32_t *image);

/* force: N x 3 doubles, energy: N doubles (per-particle potential energy, half of each pair / bond energy) or
   NULL.  MD_ESTATE if no force has been computed for the current positions. */
int md_get_forces(md_ctx *ctx, double *force, double *energy);

/* ---- S1 cell binning (PAPER.md:126 cell list; Fig. 4 step 1) ------------------------------- */

/* Cell of every particle: n_c = floor(L/r_list) per axis, f = (x + L/2)/L, c = (int)(f n_c) clamped to n_c-1
   (R5, bit-exact IEEE double, no FMA); then a deterministic counting sort of ALL per-particle arrays into cell
   order (cells along the configured curve, particles of one cell by ascending tag), and a snapshot of the
   positions for the displacement check (S3).  Invalidates the neighbour list. */
int md_build_cells(md_ctx *ctx);

/* cell_of: N uint32 in tag order, linear id cx + n_cx (cy + n_cy cz); dims: 3 uint32 (HOST pointer). */
int md_get_cells(md_ctx *ctx, uint32_t *cell_of, uint32_t dims[3]);

/* ---- S2 neighbour list (Fig. 4; list radius PAPER.md:79) -------------------------------- */

/* Full (double-sided) Verlet list: row i holds every j != i with |minimg(x_i - x_j)|^2 < r_list^2 (strict;
   (dx^2 + dy^2) + dz^2 in IEEE double without FMA, R2).  w cooperative threads per particle stride over the 27
   stencil cells and compact with a w-wide prefix sum (no atomics).  Requires md_build_cells on the current
   positions (it is run automatically if missing). */
int md_build_nlist(md_ctx *ctx);

/* Unordered export: each listed pair once as (tag_i < tag_j).  pairs = NULL: only *n_pairs is written
   (HOST pointer).  Otherwise pairs must hold 2 * cap uint32; MD_EINVAL if cap is too small.
   The ORDER of the pairs is unspecified (sort to compare). */
int md_get_nlist(md_ctx *ctx, uint64_t *n_pairs, uint32_t *pairs, uint64_t cap);

/* Rows of selected particles: counts[n_probe] = row length, nbr_tags[p * row_stride + k] = tag of the k-th
   neighbour (k < min(count, row_stride)), order within a row unspecified. */
int md_get_nlist_rows(md_ctx *ctx, const uint32_t *probe_tags, uint32_t n_probe, uint32_t *counts,
                      uint32_t *nbr_tags, uint32_t row_stride);

/* ---- S4/S5 forces (w threads per particle, shuffle reduction, one write per particle) ------ */

/* Truncated LJ 12-6 (R1): F_i = sum_j 24 eps (2 s^12 - s^6)/r^2 d_ij over list neighbours with
   r^2 < rc^2, s = sigma/r; per-particle energy = 1/2 sum_j [4 eps (s^12 - s^6) - shift U(rc)].  OVERWRITES the
   force/energy arrays.  Needs a valid neighbour list (MD_ESTATE otherwise). */
int md_forces_lj(md_ctx *ctx, double epsilon, double sigma, int energy_shift);

/* DPD (Groot-Warren form, R9): for 0 < r < rc, w = 1 - r/rc,
   F_ij = [A w - gamma w^2 (rhat . v_ij) + sqrt(2 gamma kT) w theta_ij / sqrt(dt)] rhat,
   theta_ij = sqrt(3) (2u - 1), u = (X + 1/2) 2^-32, X = word 0 of Philox4x32-10 with
   counter (min tag, max tag, step lo, step hi) and key (seed lo, seed hi) (R13, R14).
   Uses the velocities as stored at the time of the call.  OVERWRITES force (energy lane = conservative energy). */
int md_forces_dpd(md_ctx *ctx, double A, double gamma, double kT, double dt, uint64_t step, uint64_t seed);

/* Harmonic bonds U = k/2 (r - r0)^2 (R19).  ACCUMULATES into force/energy. */
int md_forces_bonds(md_ctx *ctx, double k, double r0);

/* ---- further short-range force fields (PAPER.md:63 feature list; fp64) ---------------------- */

/* Pair potential `kind` (MD_PAIR_*) with parameters p[4] (HOST pointer), pairs with r^2 < rc^2 (strict), energies shifted
   by U(rc) if energy_shift.  Same kernel structure as md_forces_lj (w threads per particle over the row, shuffle
   reduction, one write), on the exact 32-bit list.  OVERWRITES force/energy.  fp64 in both precision modes. */
int md_forces_pair(md_ctx *ctx, int kind, const double p[4], int energy_shift);

/* Tabulated pair potential (R37; "tabulated potentials"): U[k] and F[k] = -dU/dr at r_k = r_min + k h,
   k = 0 .. m-1, h = (r_max - r_min) / (m - 1); 0 <= r_min < r_max <= r_cut, 2 <= m < 2^31.  U and F are interpolated
   linearly in r (k = floor((r - r_min) / h), clamped to m - 2); a pair contributes if r_min <= r and r^2 < r_max^2
   (strict), F(r) d / r to the first particle and half of U(r) to each energy.  U, F: HOST or DEVICE arrays of m
   doubles, copied.  m = 0 clears.  Used by md_forces_pair(kind = MD_PAIR_TABLE) and MD_F_PAIR with pair_kind =
   MD_PAIR_TABLE (MD_ESTATE if no table is set); the virial of md_pressure follows the same interpolation. */
int md_set_pair_table(md_ctx *ctx, double r_min, double r_max, const double *U, const double *F, uint64_t m);

/* Tabulated bonds (R38; "harmonic, FENE and tabulated bonds") on the bonds of md_set_bonds: U[k] and
   F[k] = -dU/dr at r_k = r_min + k h, k = 0 .. m-1, h = (r_max - r_min) / (m - 1), 0 <= r_min < r_max, 2 <= m < 2^31,
   interpolated linearly in r exactly like md_set_pair_table's; one table for all bonds (R27).  A bond with r < r_min or
   r >= r_max has left its table: NaN in the forces and energies of both ends (like the FENE bond beyond r0).
   U, F: HOST or DEVICE arrays of m doubles, copied; m = 0 clears.  md_forces_bond_table ACCUMULATES like md_forces_bonds
   (MD_ESTATE if no table is set); md_step / md_pressure take it with bond_kind = MD_BOND_TABLE. */
int md_set_bond_table(md_ctx *ctx, double r_min, double r_max, const double *U, const double *F, uint64_t m);
int md_forces_bond_table(md_ctx *ctx);

/* FENE bonds on the bond table of md_set_bonds (R33).  ACCUMULATES, like md_forces_bonds. */
int md_forces_fene(md_ctx *ctx, double k, double r0);

/* Harmonic angles (R34): triplets of tags (a, b, c), b the vertex; theta = angle between x_a - x_b and x_c - x_b
   (minimum image), U = k/2 (theta - theta0)^2, one third of it to each particle's energy; collinear triplets
   (sin theta < 1e-12) are skipped.  Stored per particle (every particle sums the terms it takes part in: no atomics).
   n_angles = 0 clears.  md_forces_angles ACCUMULATES. */
int md_set_angles(md_ctx *ctx, const uint32_t *tag_a, const uint32_t *tag_b, const uint32_t *tag_c, uint64_t n_angles);
int md_forces_angles(md_ctx *ctx, double k, double theta0);

/* Periodic dihedrals (R35; PAPER.md:63 names "dihedral"): quadruplets of tags (a, b, c, d) around the bond b-c.
   F = x_a - x_b, G = x_b - x_c, H = x_d - x_c (minimum image), A = F x G, B = H x G,
   phi = atan2((B x A).G / |G|, A.B) in (-pi, pi] (0 = cis, pi = trans); U = k/2 (1 + sign cos(n phi)), sign = +-1,
   n >= 1; one quarter of U to each particle's energy; degenerate quadruplets (|A|^2 or |B|^2 < 1e-24 |G|^4: three
   collinear particles) are skipped.  tag arrays: HOST or DEVICE, n_dihedrals entries each, copied; a tag out of range or
   repeated within a quadruplet is MD_EINVAL (host arrays only).  Stored per particle like the angles (no atomics).
   n_dihedrals = 0 clears.  md_forces_dihedrals ACCUMULATES into force/energy; MD_EINVAL for sign not +-1 or n < 1. */
int md_set_dihedrals(md_ctx *ctx, const uint32_t *tag_a, const uint32_t *tag_b, const uint32_t *tag_c, const uint32_t *tag_d,
                     uint64_t n_dihedrals);
int md_forces_dihedrals(md_ctx *ctx, double k, int sign, int n);

/* Langevin thermostat (R36; "Brownian (or Langevin) dynamics"; SURVEY.md 8(f) row 3 "from the same
   counter-based hash"): the one-body force F_i += -gamma v_i + sqrt(6 gamma kT / dt) (u_x, u_y, u_z) at the CURRENT
   velocities, u uniform on (-1, 1): u_k = 2 (X_k + 0.5) 2^-32 - 1, X = Philox4x32-10(counter = (tag, 0xffffffff, step lo,
   step hi), key = (seed lo, seed hi)).  ACCUMULATES into the force; no energy, no virial.  Inside md_step (MD_F_LANGEVIN)
   it is evaluated with the other forces, after half 1, with step = the step being completed (like the DPD terms), and the
   velocity-Verlet halves integrate it; mutually exclusive with MD_F_NVT.  gamma < 0, kT < 0 or dt <= 0: MD_EINVAL. */
int md_forces_langevin(md_ctx *ctx, double gamma, double kT, double dt, uint64_t step, uint64_t seed);

/* ---- virial and pressure (PAPER.md:63 NPT / NPH, :208, :214; R32) ----------------------------- */

/* W = sum over the pairs of `what`'s pair term of d (x) F (d = minimum-image separation, F the pair force on the first
   particle; for MD_F_DPD all three terms with hash counter = the context's current step), plus bonds, angles and dihedrals (arm (x) F
   per end) if flagged; order xx, yy, zz, xy, xz, yz.  kinetic = sum 1/2 m v^2, volume = box volume,
   pressure = (2 kinetic + W_xx + W_yy + W_zz) / (3 volume).  Evaluated on demand at the current positions with the
   neighbour list rebuilt if stale; device reductions in a fixed order.  out: HOST pointer.  Synchronises. */
typedef struct md_pressure_t {
    double virial[6], kinetic, volume, pressure;
} md_pressure_t;
int md_pressure(md_ctx *ctx, const md_step_desc *what, md_pressure_t *out);

/* ---- S6 velocity-Verlet, NVE (R7) ---------------------------------------------------------- */

/* half = 1: v += (dt/2) F/m; x += dt v; wrap into the box (image counters updated); evaluates the displacement
   criterion of PAPER.md:79 (some particle moved more than r_buff/2 since the last md_build_cells, strict >) into a
   device flag; invalidates forces.   half = 2: v += (dt/2) F/m. */
int md_integrate_nve(md_ctx *ctx, double dt, int half);

/* Host read of the displacement flag set by the last half-1 (synchronises).  *flag = 1: a rebuild is due. */
int md_needs_rebuild(md_ctx *ctx, int *flag);

/* ---- S7 step scheduler ---------------------------------------------------------------------------------- */

/* n_steps of { half 1 -> displacement check -> [cells + neighbour list] -> forces -> half 2 }.  If no force is
   current, forces are first evaluated at the current step index (R16).  The force evaluated during the step that
   advances t -> t+1 uses hash counter t+1 (R15). */
int md_step(md_ctx *ctx, const md_step_desc *what, uint64_t n_steps);

/* ---- S8 runtime tuner ------------------------------------------------------------------ */

/* Sweeps, for EVERY kernel family of the step `what` describes (binning, neighbour list, pair force, bonds,
   integrator), the block size (multiples of 32 up to the kernel's compiled limit; `full` = all of them, else a pruned
   set) and, where the kernel has it, the threads per particle w in {1,2,4,8,16,32}, on the live state (the kernels are
   pure functions of it; half 1 is replayed with dt = 0, the binning only while no step has been taken since the last
   one), median of 5 timed launches each, and fixes the fastest.  md_get_stats reports the LAUNCHED (block, w) per
   kernel; with the environment variable B200MD_LOG set every timing is printed to stderr.  MD_OPT_RETUNE_PERIOD = M
   makes md_step repeat a local re-scan (neighbouring block sizes, w/2 .. 2w) after every M rebuilds. */
int md_tune(md_ctx *ctx, const md_step_desc *what, int full);

/* SURVEY.md 8(f) row 2.  The paper determines r_buff per benchmark "as the value that yields the highest number of time
   steps per second".  For each candidate skin (candidates[n_candidates], HOST; NULL = 0.5 ... 2 times the
   current one in steps of 0.25; values the box cannot hold -- fewer than 3 cells per axis -- are skipped) the context is
   re-gridded, `what` is run for burst_steps / 10 untimed and burst_steps (0 = 200) timed steps from the SAME saved state, and
   the fastest skin is kept: the state, the step counter and the statistics are those from before the call, the cell grid
   and the neighbour list are those of the chosen skin (rebuilt at the next call).  *chosen (HOST, may be NULL) and
   md_get_stats().r_buff report it; B200MD_LOG prints every burst.  Trajectories do not depend on the skin beyond
   floating-point summation order; bench.py reports the configured r_buff = 0.4 unless asked (--auto-rbuff). */
int md_tune_rbuff(md_ctx *ctx, const md_step_desc *what, const double *candidates, uint32_t n_candidates,
                  uint64_t burst_steps, double *chosen);

/* Options of the tile path (MD_ORDER_MORTON).  MD_OPT_TILE_BRICK: edge of the cell brick one CTA owns, 1, 2 or 4
   (0 = choose from the density); invalidates cells and list.  MD_OPT_ACC_BLOCK (MD_MIXED only): 1 = every pair's
   fp32 contribution is widened and added in fp64; 8 (default) = contributions of 8 consecutive list entries are summed
   in fp32, the block sum is widened and added in fp64 (R25). */
#define MD_OPT_TILE_BRICK 1
#define MD_OPT_ACC_BLOCK 2
#define MD_OPT_RETUNE_PERIOD 4 /* rebuilds between periodic local re-scans of the tuner inside md_step; 0 (default) = never */
#define MD_OPT_PROFILE_STRIDE 8 /* md_set_profiling(ctx, 2) brackets every S-th pair-force launch with events (default 1 = every one);
                                  stage_ms / stage_launches then hold the sampled launches only */
int md_set_option(md_ctx *ctx, int option, int64_t value);

/* Fix launch parameters by hand (block multiple of 32 in [32,1024]; w power of two <= 32); kernel = MD_K_*. */
int md_set_launch(md_ctx *ctx, int kernel, int block, int w);

/* NVT, Nose-Hoover thermostat (named by the paper, which prints no
   equations: DESIGN.md R30).  dv/dt = F/m - xi v, dxi/dt = (T_inst/T0 - 1)/tau^2, deta/dt = xi, T_inst = 2K/(3N-3).
   half = 1: v <- (v + (dt/2) F/m) / (1 + (dt/2) xi); x <- x + dt v; wrap; displacement check (as md_integrate_nve);
             then K' = sum 1/2 m v^2 is reduced on the device (fixed order) and xi <- xi + (dt/tau^2)(2K'/((3N-3) kT) - 1),
             eta <- eta + (dt/2)(xi + xi_old): no host round trip.
   half = 2: v <- v + (dt/2)(F/m - xi v).
   The thermostat variables live in the context: md_set_state resets them to 0. */
int md_integrate_nvt(md_ctx *ctx, double dt, int half, double kT, double tau);
/* Martyna-Tobias-Klein update for NVT (R39; "the symplectic Martyna-Tobias-Klein update equations"; SURVEY.md
   8(f) row 1): the equations of motion of md_integrate_nvt with one thermostat, Q = (3N - 3) kT tau^2, as the symmetric
   factorisation  step = T(dt/2) half1 [forces] half2 T(dt/2)  with the NVE halves of md_integrate_nve and
     T(dt/2): xi += (dt/4)(2K - (3N-3) kT)/Q; s = exp(-xi dt/2); v <- s v; K <- s^2 K; eta += xi dt/2; xi += (dt/4)(2K - (3N-3) kT)/Q.
   md_mtk_thermostat_half applies one T(dt/2) on the device (K reduction in md_thermo's fixed order, one-thread update of
   xi and eta, one scaling pass); xi and eta are the ones of md_set_thermostat / md_get_thermostat.  md_step with MD_F_MTK
   (excludes MD_F_NVT and MD_F_LANGEVIN) runs the whole step and merges the trailing factor of a step with the leading one
   of the next into one reduction and one scaling pass; every scheduler gives identical results.  Time-reversible. */
int md_mtk_thermostat_half(md_ctx *ctx, double dt, double kT, double tau);
int md_set_thermostat(md_ctx *ctx, double xi, double eta);
int md_get_thermostat(md_ctx *ctx, double *xi, double *eta); /* HOST pointers; synchronises */

int md_get_stats(md_ctx *ctx, md_stats *out); /* synchronises */

/* Device-side thermodynamic reductions (the paper reduces kinetic energy every NVT step,
   PAPER.md:208, :214): kinetic = sum 1/2 m v^2, potential = sum of the per-particle potential energies of the current
   forces (md_get_forces' energy lane; forces left by md_step are re-evaluated with energies, R16 / md_get_forces),
   momentum = sum m v, temperature = 2 kinetic / (3 N - 3) (R18).  Two kernels, fixed summation order (per-block
   partial sums in slot order, then one block over the partials): the result is bit-reproducible for a given state.
   out: HOST pointer.  Synchronises.  MD_ESTATE if no force is current (potential would be undefined). */
typedef struct md_thermo_t {
    double kinetic, potential, momentum[3], temperature;
} md_thermo_t;
int md_thermo(md_ctx *ctx, md_thermo_t *out);

/* The same kinetic-energy / momentum reduction for callers that cannot allocate device memory (code under CUDA graph
   capture, tight serving loops, harnesses that forbid cudaMalloc).  No context: the caller passes the inputs and the
   output; the per-block partial sums, which md_thermo keeps in a buffer of the context, live in a file-scope __device__
   array of the library (256 KiB, held by every GPU that loads the library until the process exits).  Calls no
   cudaMalloc / cudaFree and no allocating library routine; enqueues two kernels on `stream` and returns WITHOUT
   synchronising.
     vel    DEVICE pointer, N x 3 doubles, row-major (velocities in the caller's own order)
     mass   DEVICE pointer, N doubles, or NULL (every mass 1)
     N      number of particles, 0 <= N <= MD_NOALLOC_MAX_N; beyond it MD_EINVAL with a message that names the limit
            (use md_thermo on a context for larger systems)
     out4   DEVICE pointer, 4 doubles, overwritten when the kernels have run: sum 1/2 m v^2, sum m v_x, m v_y, m v_z
     stream cudaStream_t as a pointer; NULL = the default stream
   Fixed summation order (blocks of 4096 particles, then one block over the partials): bit-reproducible for a given
   input.  A host pointer is MD_EINVAL (nothing is staged).  The scratch array is shared by ALL calls on a device and
   keeps the last call's contents; nothing in it needs clearing (a call writes every slot it reads), but two calls that
   overlap on the GPU -- different streams, or graph branches without a dependency -- race on it: serialise them.
   md_noalloc_last_error: text of the calling thread's last failure of md_kinetic_noalloc. */
#define MD_NOALLOC_MAX_N 33554432ull /* 8192 block partials x 4096 particles */
int md_kinetic_noalloc(const double *vel, const double *mass, uint64_t N, double *out4, void *stream);
const char *md_noalloc_last_error(void);

/* on = 1: bracket every stage launched by md_step / md_build_* / md_forces_* / md_integrate_nve with CUDA events on the
   context's stream and accumulate their durations into md_stats.stage_ms (MD_K_CELLS = binning + reorder, MD_K_NLIST =
   count + scan + fill, MD_K_LJ / MD_K_DPD / MD_K_BONDS force kernels, MD_K_INTEGRATE both halves).  Resets the
   accumulators.  on = 2: only the pair-force stages (MD_K_LJ / MD_K_DPD) are bracketed -- two events per step instead of
   about eight, for timing a run while measuring its dominant kernel.  on = 0 switches the events off. */
int md_set_profiling(md_ctx *ctx, int on);

/* Test hook: Philox4x32-10 of `n` (counter, key) inputs evaluated ON THE DEVICE by the same device function the
   DPD kernel uses.  ctr: n x 4 uint32, key: n x 2 uint32, out: n x 4 uint32 (host or device pointers). */
int md_debug_philox(md_ctx *ctx, const uint32_t *ctr, const uint32_t *key, uint32_t *out, uint64_t n);

/* sizeof of the structs crossing this boundary as the library was compiled (0 md_step_desc, 1 md_stats, 2 md_thermo_t,
   3 md_pressure_t; -1 otherwise): lets a binding check its mirror of the layouts */
int md_struct_size(int which);

/* Measurement hook (measured, not nominal, peaks of the non-tensor pipes; PAPER.md:300 is the paper's
   only statement on what bounds the path): issue rate of one instruction kind on the whole GPU, every thread running 8
   independent chains, in giga lane-instructions per second (an FMA counts once; FMA2 = packed fma.rn.f32x2, counted
   once per instruction, i.e. two FMAs; CVT = cvt.f64.f32 / cvt.rn.f32.f64; LDS128 = conflict-free 16-byte shared loads).
   Best of 3 timed launches on the context's stream; synchronises.  giga_per_s: HOST pointer. */
enum { MD_PEAK_FP32_FMA = 0, MD_PEAK_FP32_FMA2 = 1, MD_PEAK_FP64_FMA = 2, MD_PEAK_INT32_MAD = 3, MD_PEAK_INT32_MULHI = 4,
       MD_PEAK_CVT_F32_F64 = 5, MD_PEAK_RCP_F32 = 6, MD_PEAK_LDS128 = 7 };
int md_debug_peak(md_ctx *ctx, int pipe, double *giga_per_s);

#ifdef __cplusplus
}
#endif
#endif /* B200MD_H */
