// md_internal.h -- context object and internal kernel-launcher prototypes of libb200md (CUDA path).
// Shares nothing with oracle/ (see DESIGN.md "Independence").
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <utility>
#include <vector>

#include "../../include/b200md.h"

#define MD_CUDA_CHECK(ctx, expr)                                                                   \
    do {                                                                                           \
        cudaError_t _e = (expr);                                                                   \
        if (_e != cudaSuccess) {                                                                   \
            (ctx)->err = std::string(#expr) + ": " + cudaGetErrorString(_e) + " (" + __FILE__ +    \
                         ":" + std::to_string(__LINE__) + ")";                                     \
            return _e == cudaErrorMemoryAllocation ? MD_ENOMEM : MD_ECUDA;                         \
        }                                                                                          \
    } while (0)

// compiled block-size limits (__launch_bounds__) of the kernel families; the tuner sweeps launchable sizes only
#define MD_TILE_MAX_BLOCK 512   // tile kernels (up to 128 registers per thread)
#define MD_LJ3_MAX_BLOCK 256    // k_tile_lj3: 4 CTAs of 256 threads per SM at 64 registers
#define MD_DPD2_MAX_BLOCK 256   // k_tile_dpd2: 4 CTAs of 256 threads per SM at 64 registers
#define MD_HALF1_MAX_BLOCK 256  // k_half1: 6 CTAs of 256 threads per SM

// nl_cnt word of a tile row: entries in the low 24 bits, blocks of the near section (the LAST K blocks of the row,
// evaluated in fp64 by the mixed-precision force kernel; R25) in the high 8
// pairs closer than MD_NEAR_SIGMAS sigma are evaluated in fp64 in MD_MIXED mode (first neighbour shell of a liquid)
#define MD_NEAR_SIGMAS 1.5
#define MD_NL_NEAR_SHIFT 24
#define MD_NL_CNT_MASK 0xffffffu

#define MD_TRY(expr)                  \
    do {                              \
        int _s = (expr);              \
        if (_s != MD_OK) return _s;   \
    } while (0)

// MD_SCHED_BATCH: the kernels of several steps are enqueued before the host looks at the rebuild
// flag.  Each carries a gate; once half 1 of enqueue index m has fired the displacement criterion (rebuild_at = m), the
// kernels with gate index >= m find the gate closed and return at once, so the state stays as that half 1 left it until
// the host has rebuilt the list.  at == nullptr: not gated.
struct Gate {
    const unsigned int *at;
    unsigned int s;
};

// geometry handed to kernels by value
struct Geom {
    double L[3];     // box edges
    double h[3];     // L/2
    double lo[3];    // -L/2
    double dn[3];    // (double) cells per axis
    double cw[3];    // cell widths L/n
    double q0, q0i;  // grid of the cell-relative fp32 records (md_rel_record): multiples of q0 = 2^-24 x the binade above
                     // the staged extent, so that record + cell offset is an EXACT fp32 sum in the tile kernels
    double qr, qri;  // quantum of the residuals carried in rel.w: q0 / 512 (fields hold -255 .. 255)
    uint32_t n[3];   // cells per axis
    uint32_t n_cells;
    uint32_t N;
};

// device-side flags / counters, mirrored to pinned host memory on demand
struct DevFlags {
    int rebuild;                  // displacement criterion fired (half 1)
    int dangerous;                // some particle moved more than r_buff since the last build
    unsigned int max_cell_count;  // most populated cell at the last binning
    unsigned int max_home;        // largest tile: home particles
    unsigned int max_staged;      // largest tile: staged (stencil) particles
    unsigned int rebuild_at;      // MD_SCHED_BATCH: enqueue index of the step whose half 1 fired the criterion (0: none); kernels
                                  // enqueued for that step's forces and everything after it return at once (md_gate_closed)
    unsigned long long nl_total;  // entries of the list being built (general path: padded rows; tile path: sum of row lengths)
    unsigned int nl_overflow;     // tile build: longest row if it exceeds the row stride (host grows the stride, rebuilds)
    unsigned int pad2;
    unsigned int max_d2[2];       // float bits of the largest squared displacement since the last binning, written by
                                  // half 1 into the slot of the step's parity (the other slot is cleared)
};

struct LaunchCfg {
    int block;
    int w;
    float us;
};

struct md_ctx {
    // problem
    double box[3];
    uint64_t N;
    double rc, r_buff, r_list;
    uint32_t dims[3];
    uint32_t n_cells;
    int precision, order, sched;
    cudaStream_t stream;
    std::string err;
    Geom g;

    // per-particle state, internal (slot) order; *_alt = reorder targets
    double4 *pos = nullptr, *pos_alt = nullptr;      // x, y, z, tag (bits)
    double4 *vel = nullptr, *vel_alt = nullptr;      // vx, vy, vz, mass
    double4 *force = nullptr, *force_alt = nullptr;  // fx, fy, fz, potential energy
    int *image = nullptr, *image_alt = nullptr;      // 3 per particle
    double *pos_ref = nullptr;                       // 3 per particle: positions at the last binning
    float4 *rel = nullptr;                           // fp32 position relative to the centre of the particle's binned cell
                                                     // (kept current by the binning and by half 1; staged by the fp32 tile kernels)
    uint32_t *tag = nullptr, *tag_alt = nullptr;     // slot -> tag
    uint32_t *rtag = nullptr;                        // tag -> slot
    uint32_t *cell_lin = nullptr;                    // slot -> linear cell id (valid after binning)

    // cell structures
    uint32_t *rank_of_lin = nullptr;  // linear cell id -> storage rank (nullptr = identity, MD_ORDER_LEX)
    uint32_t *cell_rank_tmp = nullptr;  // old slot -> rank (binning scratch)
    uint32_t *cell_count = nullptr, *cell_start = nullptr;  // per rank; cell_start has n_cells+1 entries
    uint32_t *perm = nullptr, *perm_sorted = nullptr;

    // neighbour list (CSR, rows padded to multiples of 4 entries)
    uint32_t *nl_cnt = nullptr;
    uint64_t *nl_off = nullptr;
    uint32_t *nl_idx = nullptr;
    uint64_t nl_capacity = 0, nl_entries = 0, nl_exact_entries = 0;
    uint32_t *nl_cnt_exp = nullptr;  // row lengths of the decoded / general CSR that the exports read

    // tile path (tiles.cu): bricks of tile_B^3 cells, Morton cell order, 16-bit staged indices
    bool use_tiles = false;     // configured (MD_ORDER_MORTON)
    bool nl_is_tile = false;    // the current list is a tile list
    bool nl32_decoded = false;  // nl_off/nl_idx hold the decoded copy of the current tile list (exports)
    double nl_near_r = 0.0;     // force-time radius the near sections of the current tile list cover (0: none)
    double lj_sigma_hint = 1.0; // sigma of the latest LJ call / step description: sizes the near section at the build
    int nl_rotw = 4;            // lanes per particle (1, 2 or 4 = "4 or more") the rows of the current tile list are rotated for

    uint32_t tile_B = 1, n_tiles = 0;
    int tile_B_forced = 0, acc_block = 8;
    uint32_t *tile_cell_begin = nullptr, *tile_origin = nullptr, *lin_of_rank = nullptr;
    uint32_t tile_max_home = 0, tile_max_staged = 0;
    uint32_t *tile_desc = nullptr;   // per-tile header tables written by k_tile_header at every rebuild
    uint64_t tile_desc_len = 0;      // words allocated
    bool tile_desc_valid = false;    // tile_desc matches the current binning
    uint16_t *nl16 = nullptr;        // fixed-stride rows: row of slot i starts at nl16 + i * nl_stride
    uint32_t nl_stride = 0;          // entries per row, multiple of 16
    uint32_t nl_shift = 0;           // entry = staged index << nl_shift
    uint32_t *nl_cnt32 = nullptr;    // exact row lengths of the decoded list (exports)

    // bonds: CSR by TAG
    uint64_t n_bonds = 0;
    uint32_t *bond_off = nullptr;      // N+1
    uint32_t *bond_partner = nullptr;  // 2*n_bonds partner tags

    // angles: CSR by TAG (entry = 4 * angle index + role), triplets by angle
    uint64_t n_angles = 0;
    uint32_t *angle_off = nullptr, *angle_ent = nullptr, *angle_abc = nullptr;
    // tabulated pair potential (R37): (U_k, F_k) pairs on the device
    double *tab_uf = nullptr;
    uint32_t tab_m = 0;
    double tab_rmin = 0.0, tab_rmax = 0.0;
    // tabulated bonds (R38): same layout
    double *btab_uf = nullptr;
    uint32_t btab_m = 0;
    double btab_rmin = 0.0, btab_rmax = 0.0;
    // dihedrals: same layout, quadruplets as uint4
    uint64_t n_dihedrals = 0;
    uint32_t *dih_off = nullptr, *dih_ent = nullptr, *dih_abcd = nullptr;

    // scratch
    uint64_t *scan_tmp = nullptr;
    uint64_t scan_tmp_len = 0;
    void *stage = nullptr;  // host<->device staging
    uint64_t stage_bytes = 0;
    double *nvt_state = nullptr;   // device: xi, eta (Nose-Hoover), allocated with the state
    double *thermo_buf = nullptr;  // per-block partial sums of md_thermo + the 5 results
    uint64_t thermo_len = 0;
    DevFlags *d_flags = nullptr;
    DevFlags *h_flags = nullptr;  // pinned

    // status
    bool have_state = false, cells_valid = false, nlist_valid = false, force_valid = false;
    bool energy_valid = false;  // the energy lane of `force` belongs to the current forces (md_step skips energies)
    uint32_t force_hint = 0;    // MD_F_* of the latest md_step / md_tune description: which pair kernel reads the list
    md_step_desc last_desc{};   // what the current forces were evaluated with (re-evaluation with energies on demand)
    uint64_t last_force_step = 0;
    bool last_from_step = false;
    uint64_t step = 0;
    int d2_slot = 0;                 // DevFlags::max_d2 slot of the last half 1
    float last_d2 = 0.f;             // largest squared displacement seen at the last flag read-back
    double d2_rate = 0.0;            // observed growth of the largest displacement per step (rebuild predictor)
    uint64_t steps_since_build = 0;  // half-1 steps since the last binning
    unsigned int gate_s = 0;         // MD_SCHED_BATCH: gate index of the kernels being enqueued (0: not gated), see Gate
    unsigned int gate_nvt = 0;       // ... gate index of a thermostat update being enqueued (the half 1 it belongs to)
    unsigned int gate_set = 0;       // ... and the index a half 1 being enqueued writes to DevFlags::rebuild_at when it fires
    cudaEvent_t ev_flags = nullptr;  // recorded after the asynchronous flag read-back of md_step
    md_stats stats;
    LaunchCfg cfg[MD_N_KERNELS];
    bool tuned = false;
    uint64_t rebuilds_at_tune = 0;   // stats.rebuilds when the tuner last ran
    uint64_t retune_period = 0;      // MD_OPT_RETUNE_PERIOD: local re-scan after this many rebuilds inside md_step (0 = off)
    bool tune_skip = false;  // set by a tuner replay that could not launch its configuration
    uint64_t device_bytes = 0;
    std::vector<std::pair<void *, uint64_t>> allocs;
    // caller-provided workspace (md_set_workspace): every internal buffer is carved from it (first fit, 256-byte units);
    // without one the context allocates with cudaMalloc
    char *ws_base = nullptr;
    uint64_t ws_bytes = 0, ws_peak = 0;
    struct WsBlock { uint64_t off, size; bool used; };
    std::vector<WsBlock> ws_blocks;
    bool state_allocated = false;  // the per-particle arrays exist (allocated at the first md_configure / md_set_state)
    bool log = false;

    // per-stage event timing (md_set_profiling)
    int profiling = 0;  // 0 off, 1 every stage, 2 pair-force stages only (md_set_profiling)
    uint64_t prof_stride = 1, prof_count = 0;  // MD_OPT_PROFILE_STRIDE: mode 2 brackets every prof_stride-th pair-force launch
    std::vector<cudaEvent_t> ev_pool;
    struct Pending { int k; cudaEvent_t e0, e1; };
    std::vector<Pending> ev_pending;
};

// RAII bracket: records an event pair around a stage when profiling is on
struct ProfScope {
    md_ctx *c;
    int k;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    ProfScope(md_ctx *ctx, int kernel);
    ~ProfScope();
};
void prof_resolve_ready(md_ctx *c);  // no sync: folds the pairs that have completed
void prof_resolve(md_ctx *c);  // call after a stream sync: folds finished event pairs into stats

// ---- helpers (api.cu) -----------------------------------------------------------------------------------
int md_alloc(md_ctx *c, void **p, uint64_t bytes);
void md_free(md_ctx *c, void *p);
int md_sync(md_ctx *c);
int md_read_flags(md_ctx *c);  // D2H of DevFlags + sync

// ---- launchers (each enqueues on c->stream and returns MD_OK or an error) ------------------------------------
int launch_exclusive_scan_u32(md_ctx *c, const uint32_t *in, uint64_t n, uint32_t *out32, uint64_t *out64,
                              bool pad4, unsigned long long *total_out);
int launch_pack_state(md_ctx *c, const double *pos, const double *vel, const double *mass);
int launch_unpack_state(md_ctx *c, double *pos, double *vel, int32_t *image);
int launch_unpack_forces(md_ctx *c, double *force, double *energy);
int launch_zero_force(md_ctx *c);
int launch_copy_energy(md_ctx *c, const double4 *src);  // force[i].w = src[i].w
int md_block_limit(const md_ctx *c, int kernel);      // largest block size the kernel behind MD_K_* can be launched with
int launch_unpack_cells(md_ctx *c, uint32_t *cell_of);
int launch_build_cells(md_ctx *c);
int launch_nlist_count(md_ctx *c);
int launch_nlist_fill(md_ctx *c);
int launch_forces_lj(md_ctx *c, double eps, double sigma, int shift);
int launch_forces_dpd(md_ctx *c, double A, double gamma, double kT, double dt, uint64_t step, uint64_t seed);
int launch_forces_bonds(md_ctx *c, double k, double r0, int kind = 0);  // kind: MD_BOND_*
// extra.cu
int launch_forces_pair(md_ctx *c, int kind, const double prm[4], int shift);
int launch_table_pack(md_ctx *c, const double *U, const double *F, uint32_t m, double *dst_uf);
int launch_angles_build(md_ctx *c, const uint32_t *ta, const uint32_t *tb, const uint32_t *tc, uint64_t na);
int launch_forces_angles(md_ctx *c, double k, double theta0);
int launch_dihedrals_build(md_ctx *c, const uint32_t *ta, const uint32_t *tb, const uint32_t *tc, const uint32_t *td, uint64_t nd);
int launch_forces_dihedrals(md_ctx *c, double k, int sign, int n);
int launch_forces_langevin(md_ctx *c, double gamma, double kT, double dt, uint64_t step, uint64_t seed);
int launch_virial(md_ctx *c, const md_step_desc *w, uint64_t step, double *out6_host);
// fused: preceded by the previous step's half 2.  nvt: Nose-Hoover friction xi read from c->nvt_state (R30)
int launch_half1(md_ctx *c, double dt, bool fused, bool nvt = false);
int launch_half2(md_ctx *c, double dt, bool nvt = false);
int launch_nvt_thermostat(md_ctx *c, double dt, double kT, double tau);  // K' reduction + xi, eta update, all on the device
int launch_mtk_thermostat(md_ctx *c, double dt, double kT, double tau, int halves);  // R39: `halves` x T(dt/2): K reduction, xi / eta update, velocity scaling
int launch_thermo(md_ctx *c, double *out6_host);  // kinetic, potential, px, py, pz (device reduction, then D2H + sync)
int launch_export_pairs_count(md_ctx *c, uint32_t *cnt);
int launch_export_pairs_fill(md_ctx *c, const uint64_t *off, uint32_t *pairs);
int launch_export_rows(md_ctx *c, const uint32_t *probe_tags, uint32_t n_probe, uint32_t *counts, uint32_t *nbr,
                       uint32_t stride);
int launch_bonds_build(md_ctx *c, const uint32_t *ta, const uint32_t *tb, uint64_t n_bonds);
int launch_debug_philox(md_ctx *c, const uint32_t *ctr, const uint32_t *key, uint32_t *out, uint64_t n);
int build_cell_order(md_ctx *c);  // host: rank_of_lin table for the configured curve (+ tile tables for Morton)
// tiles.cu
int tile_measure(md_ctx *c);
int launch_tile_build(md_ctx *c, bool *fits);
int tile_build_lanes(md_ctx *c);  // lanes that cooperate on one particle in the tile build kernel in use
static inline int tile_rot_class(int w) { return w <= 1 ? 1 : (w == 2 ? 2 : 4); }
int launch_tile_lj(md_ctx *c, double eps, double sigma, int shift, bool energy);
int launch_tile_dpd(md_ctx *c, double A, double gamma, double kT, double dt, uint64_t step, uint64_t seed);
bool tile_forces_fit(md_ctx *c, bool dpd);
int launch_tile_decode(md_ctx *c, bool fill, uint32_t *cnt32);
