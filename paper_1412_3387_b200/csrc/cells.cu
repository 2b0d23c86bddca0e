// cells.cu -- S0 state pack/unpack, S1 cell binning as a deterministic counting sort, exclusive scan utility.
//
// S1 ("cell list", Fig. 4 step 1 PAPER.md:171): the paper's cell list uses atomics and is therefore
// non-deterministic.  Here atomics only COUNT (integer adds commute); the order inside a cell is then fixed by
// sorting the cell's members by tag, so the particle order after binning is a pure function of the positions.
#include "md_device.cuh"

// =====================================================================================================
// exclusive scan of uint32 counts (optionally each count rounded up to a multiple of 4) into uint32 / uint64
// three launches: tile sums -> scan of tile sums (one block) -> per-tile scan + offset
// =====================================================================================================
constexpr int SCAN_THREADS = 512;
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;

__device__ __forceinline__ uint32_t scan_item(const uint32_t *in, uint64_t i, uint64_t n, bool pad4)
{
    if (i >= n) return 0u;
    uint32_t v = in[i];
    return pad4 ? ((v + 3u) & ~3u) : v;
}

// block-wide exclusive scan of one value per thread; returns exclusive prefix, *total = block sum
__device__ __forceinline__ unsigned long long block_excl_scan(unsigned long long v, unsigned long long *total)
{
    __shared__ unsigned long long warp_sums[32];
    const unsigned lane = threadIdx.x & 31u, wid = threadIdx.x >> 5;
    unsigned long long incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        unsigned long long t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= (unsigned)o) incl += t;
    }
    if (lane == 31) warp_sums[wid] = incl;
    __syncthreads();
    if (wid == 0) {
        const unsigned nw = (blockDim.x + 31) >> 5;
        unsigned long long s = lane < nw ? warp_sums[lane] : 0ull, si = s;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            unsigned long long t = __shfl_up_sync(0xffffffffu, si, o);
            if (lane >= (unsigned)o) si += t;
        }
        warp_sums[lane] = si - s;  // exclusive warp offsets
        if (lane == 31) *total = si;
    }
    __syncthreads();
    const unsigned long long r = warp_sums[wid] + incl - v;
    __syncthreads();
    return r;
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_tile_sums(const uint32_t *in, uint64_t n, bool pad4,
                                                                 unsigned long long *tile_sums)
{
    const uint64_t base = (uint64_t)blockIdx.x * SCAN_TILE + (uint64_t)threadIdx.x * SCAN_ITEMS;
    unsigned long long s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) s += scan_item(in, base + k, n, pad4);
    __shared__ unsigned long long tot;
    (void)block_excl_scan(s, &tot);
    if (threadIdx.x == 0) tile_sums[blockIdx.x] = tot;
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_of_sums(unsigned long long *tile_sums, uint64_t n_tiles,
                                                               unsigned long long *total_out)
{
    __shared__ unsigned long long tot;
    unsigned long long carry = 0;
    for (uint64_t base = 0; base < n_tiles; base += SCAN_THREADS) {
        const uint64_t i = base + threadIdx.x;
        const unsigned long long v = i < n_tiles ? tile_sums[i] : 0ull;
        const unsigned long long ex = block_excl_scan(v, &tot);
        if (i < n_tiles) tile_sums[i] = carry + ex;
        carry += tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        tile_sums[n_tiles] = carry;
        if (total_out) *total_out = carry;
    }
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_apply(const uint32_t *in, uint64_t n, bool pad4,
                                                             const unsigned long long *tile_sums, uint32_t *out32,
                                                             uint64_t *out64)
{
    const uint64_t base = (uint64_t)blockIdx.x * SCAN_TILE + (uint64_t)threadIdx.x * SCAN_ITEMS;
    uint32_t v[SCAN_ITEMS];
    unsigned long long s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) { v[k] = scan_item(in, base + k, n, pad4); s += v[k]; }
    __shared__ unsigned long long tot;
    unsigned long long ex = block_excl_scan(s, &tot) + tile_sums[blockIdx.x];
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        const uint64_t i = base + k;
        if (i < n) {
            if (out32) out32[i] = (uint32_t)ex;
            if (out64) out64[i] = ex;
        }
        ex += v[k];
    }
    if (blockIdx.x == gridDim.x - 1 && threadIdx.x == blockDim.x - 1) {
        // ex is now the grand total (threads past n contributed 0)
        if (out32) out32[n] = (uint32_t)ex;
        if (out64) out64[n] = ex;
    }
}

int launch_exclusive_scan_u32(md_ctx *c, const uint32_t *in, uint64_t n, uint32_t *out32, uint64_t *out64,
                              bool pad4, unsigned long long *total_out)
{
    const uint64_t n_tiles = (n + SCAN_TILE - 1) / SCAN_TILE;
    if (n_tiles + 1 > c->scan_tmp_len) {
        if (c->scan_tmp) md_free(c, c->scan_tmp);
        c->scan_tmp_len = n_tiles + 1 + 1024;
        MD_TRY(md_alloc(c, (void **)&c->scan_tmp, c->scan_tmp_len * sizeof(uint64_t)));
    }
    unsigned long long *ts = (unsigned long long *)c->scan_tmp;
    k_scan_tile_sums<<<(unsigned)n_tiles, SCAN_THREADS, 0, c->stream>>>(in, n, pad4, ts);
    MD_LAUNCH_CHECK(c);
    k_scan_of_sums<<<1, SCAN_THREADS, 0, c->stream>>>(ts, n_tiles, total_out);
    MD_LAUNCH_CHECK(c);
    k_scan_apply<<<(unsigned)n_tiles, SCAN_THREADS, 0, c->stream>>>(in, n, pad4, ts, out32, (uint64_t *)out64);
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

// =====================================================================================================
// S0: tag-ordered user arrays <-> internal arrays
// =====================================================================================================
__global__ void k_pack_state(const double *__restrict__ pos, const double *__restrict__ vel,
                             const double *__restrict__ mass, Geom g, double4 *opos, double4 *ovel, int *image,
                             uint32_t *tag, uint32_t *rtag)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.N) return;
    double x[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        double v = pos[3ull * i + a];
        // wrap once into [-L/2, L/2) (R4); loops terminate for finite input
        while (v >= g.h[a]) v = __dsub_rn(v, g.L[a]);
        while (v < -g.h[a]) v = __dadd_rn(v, g.L[a]);
        x[a] = v;
        image[3ull * i + a] = 0;
    }
    opos[i] = make_double4(x[0], x[1], x[2], md_tag_to_lane(i));
    ovel[i] = make_double4(vel[3ull * i], vel[3ull * i + 1], vel[3ull * i + 2], mass ? mass[i] : 1.0);
    tag[i] = i;
    rtag[i] = i;
}

int launch_pack_state(md_ctx *c, const double *pos, const double *vel, const double *mass)
{
    k_pack_state<<<md_grid(c->N, 256), 256, 0, c->stream>>>(pos, vel, mass, c->g, c->pos, c->vel, c->image, c->tag,
                                                            c->rtag);
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

__global__ void k_unpack_state(const double4 *__restrict__ pos, const double4 *__restrict__ vel,
                               const int *__restrict__ image, const uint32_t *__restrict__ tag, uint32_t N,
                               double *opos, double *ovel, int32_t *oimage)
{
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= N) return;
    const uint64_t t = tag[s];
    if (opos) { const double4 p = pos[s]; opos[3 * t] = p.x; opos[3 * t + 1] = p.y; opos[3 * t + 2] = p.z; }
    if (ovel) { const double4 v = vel[s]; ovel[3 * t] = v.x; ovel[3 * t + 1] = v.y; ovel[3 * t + 2] = v.z; }
    if (oimage) {
        oimage[3 * t] = image[3ull * s]; oimage[3 * t + 1] = image[3ull * s + 1]; oimage[3 * t + 2] = image[3ull * s + 2];
    }
}

int launch_unpack_state(md_ctx *c, double *pos, double *vel, int32_t *image)
{
    k_unpack_state<<<md_grid(c->N, 256), 256, 0, c->stream>>>(c->pos, c->vel, c->image, c->tag, (uint32_t)c->N, pos,
                                                              vel, image);
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

__global__ void k_unpack_forces(const double4 *__restrict__ force, const uint32_t *__restrict__ tag, uint32_t N,
                                double *of, double *oe)
{
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= N) return;
    const uint64_t t = tag[s];
    const double4 f = force[s];
    if (of) { of[3 * t] = f.x; of[3 * t + 1] = f.y; of[3 * t + 2] = f.z; }
    if (oe) oe[t] = f.w;
}

int launch_unpack_forces(md_ctx *c, double *force, double *energy)
{
    k_unpack_forces<<<md_grid(c->N, 256), 256, 0, c->stream>>>(c->force, c->tag, (uint32_t)c->N, force, energy);
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

__global__ void k_unpack_cells(const uint32_t *__restrict__ cell_lin, const uint32_t *__restrict__ tag, uint32_t N,
                               uint32_t *out)
{
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < N) out[tag[s]] = cell_lin[s];
}

int launch_unpack_cells(md_ctx *c, uint32_t *cell_of)
{
    k_unpack_cells<<<md_grid(c->N, 256), 256, 0, c->stream>>>(c->cell_lin, c->tag, (uint32_t)c->N, cell_of);
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

// =====================================================================================================
// S1: binning
// =====================================================================================================
// (1) cell of every particle + population count
__global__ void k_cell_id(const double4 *__restrict__ pos, Geom g, const uint32_t *__restrict__ rank_of_lin,
                          uint32_t *cell_lin_old, uint32_t *cell_rank, uint32_t *cell_count)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.N) return;
    const double4 p = pos[i];
    const uint32_t cx = md_cell_coord(p.x, g.lo[0], g.L[0], g.dn[0], g.n[0]);
    const uint32_t cy = md_cell_coord(p.y, g.lo[1], g.L[1], g.dn[1], g.n[1]);
    const uint32_t cz = md_cell_coord(p.z, g.lo[2], g.L[2], g.dn[2], g.n[2]);
    const uint32_t lin = cx + g.n[0] * (cy + g.n[1] * cz);
    const uint32_t r = rank_of_lin ? rank_of_lin[lin] : lin;
    cell_lin_old[i] = lin;
    cell_rank[i] = r;
    atomicAdd(&cell_count[r], 1u);
}

// (3) after the scan: every particle takes a slot of its cell (arrival order arbitrary, fixed in step 4)
__global__ void k_cell_scatter(const uint32_t *__restrict__ cell_rank, uint32_t N, const uint32_t *__restrict__ cell_start,
                               uint32_t *cell_fill, uint32_t *perm)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const uint32_t r = cell_rank[i];
    const uint32_t k = atomicAdd(&cell_fill[r], 1u);
    perm[cell_start[r] + k] = i;
}

// (4) one warp per cell: order the cell's members by (sub-cell Morton key, tag) -- rank sort; tags are unique, so the
// order is a pure function of the positions.  The sub-cell key (3 bits per axis of the position inside the cell) makes
// runs of consecutive members spatially compact: a build task of 8 consecutive members has a small extent.
__device__ __forceinline__ uint32_t sub_coord(double x, double lo, double L, double dn, uint32_t n)
{
    const double f = __dmul_rn(__ddiv_rn(__dsub_rn(x, lo), L), dn);
    long long k = (long long)f;
    if (k >= (long long)n) k = (long long)n - 1;
    if (k < 0) k = 0;
    int s = (int)((f - (double)k) * 8.0);
    return (uint32_t)min(7, max(0, s));
}
__device__ __forceinline__ uint32_t spread3(uint32_t v) { return (v & 1u) | ((v & 2u) << 2) | ((v & 4u) << 4); }
__device__ __forceinline__ unsigned long long cell_sort_key(const double4 p, const Geom &g, uint32_t t, bool subsort)
{
    uint32_t sub = 0;
    if (subsort) {
        sub = spread3(sub_coord(p.x, g.lo[0], g.L[0], g.dn[0], g.n[0])) |
              (spread3(sub_coord(p.y, g.lo[1], g.L[1], g.dn[1], g.n[1])) << 1) |
              (spread3(sub_coord(p.z, g.lo[2], g.L[2], g.dn[2], g.n[2])) << 2);
    }
    return ((unsigned long long)sub << 32) | t;
}

__global__ void k_cell_sort(const uint32_t *__restrict__ perm, const uint32_t *__restrict__ cell_start,
                            const uint32_t *__restrict__ tag, const double4 *__restrict__ pos, Geom g, bool subsort,
                            uint32_t n_cells, uint32_t lpc /* lanes per cell: 8, 16 or 32 */, uint32_t *perm_sorted,
                            unsigned int *max_count)
{
    // a group of lpc lanes per cell (from the mean population: a sparse DPD cell of 8 members does not need a warp)
    const uint32_t cell = (blockIdx.x * blockDim.x + threadIdx.x) / lpc;
    const unsigned lane = threadIdx.x & (lpc - 1u);
    const unsigned gmask = lpc == 32u ? 0xffffffffu : (((1u << lpc) - 1u) << ((threadIdx.x & 31u) & ~(lpc - 1u)));
    if (cell >= n_cells) return;  // (whole groups leave: n_cells * lpc threads are a multiple of lpc)
    const uint32_t b = cell_start[cell], e = cell_start[cell + 1], n = e - b;
    if (lane == 0 && n > 0) atomicMax(max_count, n);
    // up to 2 lpc members: keys in registers (2 per lane), ranks by shuffles inside the group; more: keys re-read from memory
    if (n <= 2u * lpc) {
        uint32_t idx[2];
        unsigned long long key[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const uint32_t m = lane + lpc * h;
            idx[h] = m < n ? perm[b + m] : 0u;
            key[h] = m < n ? cell_sort_key(pos[idx[h]], g, tag[idx[h]], subsort) : ~0ull;
        }
        uint32_t rank[2] = {0u, 0u};
        for (uint32_t k = 0; k < n; ++k) {
            const unsigned long long kk = __shfl_sync(gmask, k < lpc ? key[0] : key[1], k & (lpc - 1u), lpc);
            rank[0] += kk < key[0] ? 1u : 0u;
            rank[1] += kk < key[1] ? 1u : 0u;
        }
        if (lane < n) perm_sorted[b + rank[0]] = idx[0];
        if (lane + lpc < n) perm_sorted[b + rank[1]] = idx[1];
    } else {
        for (uint32_t m = lane; m < n; m += lpc) {
            const uint32_t idx = perm[b + m];
            const unsigned long long key = cell_sort_key(pos[idx], g, tag[idx], subsort);
            uint32_t rank = 0;
            for (uint32_t k = 0; k < n; ++k) {
                const uint32_t ik = perm[b + k];
                rank += cell_sort_key(pos[ik], g, tag[ik], subsort) < key ? 1u : 0u;
            }
            perm_sorted[b + rank] = idx;
        }
    }
}

// (5) move every per-particle array into the new order; snapshot positions for the displacement check
__global__ void k_reorder(const uint32_t *__restrict__ perm_sorted, uint32_t N, const double4 *__restrict__ pos,
                          const double4 *__restrict__ vel, const double4 *__restrict__ force,
                          const int *__restrict__ image, const uint32_t *__restrict__ tag,
                          const uint32_t *__restrict__ cell_lin_old, double4 *npos, double4 *nvel, double4 *nforce,
                          int *nimage, uint32_t *ntag, uint32_t *rtag, uint32_t *cell_lin, double *pos_ref, Geom g,
                          float4 *rel)
{
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= N) return;
    const uint32_t o = perm_sorted[s];
    const double4 p = pos[o];
    npos[s] = p;
    nvel[s] = vel[o];
    nforce[s] = force[o];
    nimage[3ull * s] = image[3ull * o];
    nimage[3ull * s + 1] = image[3ull * o + 1];
    nimage[3ull * s + 2] = image[3ull * o + 2];
    const uint32_t t = tag[o];
    ntag[s] = t;
    rtag[t] = s;
    const uint32_t lin = cell_lin_old[o];
    cell_lin[s] = lin;
    if (MD_STAGE_FROM_REL) rel[s] = md_rel_record(p.x, p.y, p.z, lin, g);
    pos_ref[3ull * s] = p.x;
    pos_ref[3ull * s + 1] = p.y;
    pos_ref[3ull * s + 2] = p.z;
}

template <typename T>
static inline void swap_ptr(T *&a, T *&b) { T *t = a; a = b; b = t; }

int launch_build_cells(md_ctx *c)
{
    const uint32_t N = (uint32_t)c->N;
    cudaStream_t st = c->stream;
    MD_CUDA_CHECK(c, cudaMemsetAsync(c->cell_count, 0, sizeof(uint32_t) * c->n_cells, st));
    MD_CUDA_CHECK(c, cudaMemsetAsync(&c->d_flags->max_cell_count, 0, sizeof(unsigned int), st));
    // cell_lin_old lives in perm_sorted's sibling scratch: use tag_alt as temporary for old linear ids
    uint32_t *cell_lin_old = c->tag_alt;
    const int blk = c->cfg[MD_K_CELLS].block;  // the streaming kernels of the binning follow the tuner
    k_cell_id<<<md_grid(N, blk), blk, 0, st>>>(c->pos, c->g, c->rank_of_lin, cell_lin_old, c->cell_rank_tmp, c->cell_count);
    MD_LAUNCH_CHECK(c);
    MD_TRY(launch_exclusive_scan_u32(c, c->cell_count, c->n_cells, c->cell_start, nullptr, false, nullptr));
    MD_CUDA_CHECK(c, cudaMemsetAsync(c->cell_count, 0, sizeof(uint32_t) * c->n_cells, st));
    k_cell_scatter<<<md_grid(N, blk), blk, 0, st>>>(c->cell_rank_tmp, N, c->cell_start, c->cell_count, c->perm);
    MD_LAUNCH_CHECK(c);
    const double ppc = (double)c->N / (double)c->n_cells;
    const uint32_t lpc = ppc <= 6.0 ? 8u : (ppc <= 13.0 ? 16u : 32u);  // 2 lpc members fit in registers; beyond: slow path
    k_cell_sort<<<md_grid((uint64_t)c->n_cells * lpc, 256), 256, 0, st>>>(c->perm, c->cell_start, c->tag, c->pos, c->g,
                                                                        c->use_tiles, c->n_cells, lpc, c->perm_sorted,
                                                                        &c->d_flags->max_cell_count);
    MD_LAUNCH_CHECK(c);
    // new tags go to cell_rank_tmp (free now), then pointers are swapped
    uint32_t *ntag = c->cell_rank_tmp;
    k_reorder<<<md_grid(N, blk), blk, 0, st>>>(c->perm_sorted, N, c->pos, c->vel, c->force, c->image, c->tag,
                                               cell_lin_old, c->pos_alt, c->vel_alt, c->force_alt, c->image_alt, ntag,
                                               c->rtag, c->cell_lin, c->pos_ref, c->g, c->rel);
    MD_LAUNCH_CHECK(c);
    swap_ptr(c->pos, c->pos_alt);
    swap_ptr(c->vel, c->vel_alt);
    swap_ptr(c->force, c->force_alt);
    swap_ptr(c->image, c->image_alt);
    // tag <- ntag: rotate the three uint32 scratch arrays (tag, cell_rank_tmp, tag_alt keep distinct storage)
    uint32_t *old_tag = c->tag;
    c->tag = ntag;
    c->cell_rank_tmp = old_tag;
    return MD_OK;
}

// =====================================================================================================
// bonds: CSR by tag, built on the device from the caller's pair list (each bond appears in both rows)
// =====================================================================================================
__global__ void k_bond_count(const uint32_t *__restrict__ ta, const uint32_t *__restrict__ tb, uint64_t nb,
                             uint32_t *cnt)
{
    const uint64_t m = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= nb) return;
    atomicAdd(&cnt[ta[m]], 1u);
    atomicAdd(&cnt[tb[m]], 1u);
}

__global__ void k_bond_fill(const uint32_t *__restrict__ ta, const uint32_t *__restrict__ tb, uint64_t nb,
                            const uint32_t *__restrict__ off, uint32_t *fill, uint32_t *partner)
{
    const uint64_t m = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= nb) return;
    const uint32_t a = ta[m], b = tb[m];
    partner[off[a] + atomicAdd(&fill[a], 1u)] = b;
    partner[off[b] + atomicAdd(&fill[b], 1u)] = a;
}

// rows are summed in ascending partner order so that the result does not depend on atomic arrival order
__global__ void k_bond_sort_rows(const uint32_t *__restrict__ off, uint32_t N, uint32_t *partner)
{
    const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= N) return;
    const uint32_t b = off[t], e = off[t + 1];
    for (uint32_t i = b + 1; i < e; ++i) {  // insertion sort, rows are tiny
        const uint32_t v = partner[i];
        uint32_t j = i;
        while (j > b && partner[j - 1] > v) { partner[j] = partner[j - 1]; --j; }
        partner[j] = v;
    }
}

int launch_bonds_build(md_ctx *c, const uint32_t *ta, const uint32_t *tb, uint64_t nb)
{
    cudaStream_t st = c->stream;
    const uint32_t N = (uint32_t)c->N;
    uint32_t *cnt = c->perm;  // scratch (N uint32), only valid to borrow outside a binning
    MD_CUDA_CHECK(c, cudaMemsetAsync(cnt, 0, sizeof(uint32_t) * N, st));
    k_bond_count<<<md_grid(nb, 256), 256, 0, st>>>(ta, tb, nb, cnt);
    MD_LAUNCH_CHECK(c);
    MD_TRY(launch_exclusive_scan_u32(c, cnt, N, c->bond_off, nullptr, false, nullptr));
    MD_CUDA_CHECK(c, cudaMemsetAsync(cnt, 0, sizeof(uint32_t) * N, st));
    k_bond_fill<<<md_grid(nb, 256), 256, 0, st>>>(ta, tb, nb, c->bond_off, cnt, c->bond_partner);
    MD_LAUNCH_CHECK(c);
    k_bond_sort_rows<<<md_grid(N, 256), 256, 0, st>>>(c->bond_off, N, c->bond_partner);
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}
