// nlist.cu -- S2 Verlet neighbour-list build (Fig. 4) and its exports.
//
// W cooperating threads per particle stride over the members of the 27 stencil cells (Fig. 4 step 2), test
// r^2 < r_list^2 (step 3; list radius r_cut + r_buff), take a W-wide exclusive prefix sum of the hit
// flags (steps 4-5, here one ballot + popc) and write the hits compacted into the particle's row (step 6) while a
// running total n_tot advances (step 7); the row length is stored at the end (step 8).  No atomics.
//
// Storage is CSR with 64-bit row offsets (config 5 has 5.5e9 entries): a COUNT pass, an exclusive scan and a FILL
// pass; both passes evaluate the same bit-reproducible fp64 decision (R2), so the counts always match.
// Because particles are stored sorted by cell and positions are wrapped at build time, the periodic image of a
// stencil cell is known per cell: the shift +-L is applied to d = x_i - x_j exactly as the minimum-image rule of
// R8 would (same IEEE operation), so no per-pair branch is needed.
#include "md_device.cuh"

template <int W, bool FILL>
__global__ void __launch_bounds__(1024) k_nlist(const double4 *__restrict__ pos, const uint32_t *__restrict__ cell_lin,
                                                const uint32_t *__restrict__ cell_start,
                                                const uint32_t *__restrict__ rank_of_lin, Geom g, double r_list2,
                                                uint32_t *__restrict__ nl_cnt, const uint64_t *__restrict__ nl_off,
                                                uint32_t *__restrict__ nl_idx)
{
    const uint32_t gid = (uint32_t)(((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) / W);
    const unsigned lane = threadIdx.x & (W - 1);
    const unsigned seg_mask = md_seg_mask<W>();
    const unsigned seg_shift = (threadIdx.x & 31u) & ~(unsigned)(W - 1);
    if (gid >= g.N) return;  // whole segments leave together (N-tail), segment masks keep the rest legal

    const uint32_t i = gid;
    const double4 pi = pos[i];
    const uint32_t lin = cell_lin[i];
    const int cx = (int)(lin % g.n[0]);
    const int cy = (int)((lin / g.n[0]) % g.n[1]);
    const int cz = (int)(lin / (g.n[0] * g.n[1]));
    const uint64_t row = FILL ? nl_off[i] : 0ull;
    uint32_t n_tot = 0;

    for (int dz = -1; dz <= 1; ++dz) {
        int nz = cz + dz;
        double sz = 0.0;
        if (nz < 0) { nz += (int)g.n[2]; sz = g.L[2]; }            // d = z_i - z_j is near -L -> add L
        else if (nz >= (int)g.n[2]) { nz -= (int)g.n[2]; sz = -g.L[2]; }
        for (int dy = -1; dy <= 1; ++dy) {
            int ny = cy + dy;
            double sy = 0.0;
            if (ny < 0) { ny += (int)g.n[1]; sy = g.L[1]; }
            else if (ny >= (int)g.n[1]) { ny -= (int)g.n[1]; sy = -g.L[1]; }
            for (int dx = -1; dx <= 1; ++dx) {
                int nx = cx + dx;
                double sx = 0.0;
                if (nx < 0) { nx += (int)g.n[0]; sx = g.L[0]; }
                else if (nx >= (int)g.n[0]) { nx -= (int)g.n[0]; sx = -g.L[0]; }
                const uint32_t nlin = (uint32_t)nx + g.n[0] * ((uint32_t)ny + g.n[1] * (uint32_t)nz);
                const uint32_t r = rank_of_lin ? rank_of_lin[nlin] : nlin;
                const uint32_t b = cell_start[r], e = cell_start[r + 1];
                for (uint32_t base = b; base < e; base += W) {
                    const uint32_t j = base + lane;
                    bool hit = false;
                    if (j < e && j != i) {
                        const double4 pj = pos[j];
                        // d = x_i - x_j, then the cell's image shift (the one correction of the minimum image)
                        double ddx = __dsub_rn(pi.x, pj.x), ddy = __dsub_rn(pi.y, pj.y), ddz = __dsub_rn(pi.z, pj.z);
                        if (sx != 0.0) ddx = __dadd_rn(ddx, sx);
                        if (sy != 0.0) ddy = __dadd_rn(ddy, sy);
                        if (sz != 0.0) ddz = __dadd_rn(ddz, sz);
                        hit = md_r2_exact(ddx, ddy, ddz) < r_list2;
                    }
                    const unsigned bal = (__ballot_sync(seg_mask, hit) >> seg_shift) & (W == 32 ? 0xffffffffu : ((1u << W) - 1u));
                    if (FILL && hit) nl_idx[row + n_tot + __popc(bal & ((1u << lane) - 1u))] = j;
                    n_tot += __popc(bal);
                }
            }
        }
    }
    if (!FILL && lane == 0) nl_cnt[i] = n_tot;
}

static int launch_nlist(md_ctx *c, bool fill)
{
    const LaunchCfg &cf = c->cfg[MD_K_NLIST];
    const uint64_t threads = c->N * (uint64_t)cf.w;
    const unsigned grid = md_grid(threads, cf.block);
    const double rl2 = c->r_list * c->r_list;
    MD_DISPATCH_W(cf.w, {
        if (fill)
            k_nlist<W_, true><<<grid, cf.block, 0, c->stream>>>(c->pos, c->cell_lin, c->cell_start, c->rank_of_lin, c->g,
                                                              rl2, c->nl_cnt, c->nl_off, c->nl_idx);
        else
            k_nlist<W_, false><<<grid, cf.block, 0, c->stream>>>(c->pos, c->cell_lin, c->cell_start, c->rank_of_lin,
                                                               c->g, rl2, c->nl_cnt, c->nl_off, c->nl_idx);
    });
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

int launch_nlist_count(md_ctx *c) { return launch_nlist(c, false); }
int launch_nlist_fill(md_ctx *c) { return launch_nlist(c, true); }

// =====================================================================================================
// exports (parity read-back): unique pairs (tag_i < tag_j) and probe rows
// =====================================================================================================
__global__ void k_pairs_count(const uint32_t *__restrict__ nl_cnt, const uint64_t *__restrict__ nl_off,
                              const uint32_t *__restrict__ nl_idx, const uint32_t *__restrict__ tag, uint32_t N,
                              uint32_t *cnt)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const uint32_t ti = tag[i], n = nl_cnt[i];
    const uint64_t row = nl_off[i];
    uint32_t k = 0;
    for (uint32_t m = 0; m < n; ++m) k += (ti < tag[nl_idx[row + m]]) ? 1u : 0u;
    cnt[i] = k;
}

__global__ void k_pairs_fill(const uint32_t *__restrict__ nl_cnt, const uint64_t *__restrict__ nl_off,
                             const uint32_t *__restrict__ nl_idx, const uint32_t *__restrict__ tag, uint32_t N,
                             const uint64_t *__restrict__ off, uint32_t *pairs)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const uint32_t ti = tag[i], n = nl_cnt[i];
    const uint64_t row = nl_off[i];
    uint64_t o = off[i];
    for (uint32_t m = 0; m < n; ++m) {
        const uint32_t tj = tag[nl_idx[row + m]];
        if (ti < tj) { pairs[2 * o] = ti; pairs[2 * o + 1] = tj; ++o; }
    }
}

int launch_export_pairs_count(md_ctx *c, uint32_t *cnt)
{
    k_pairs_count<<<md_grid(c->N, 128), 128, 0, c->stream>>>(c->nl_cnt_exp, c->nl_off, c->nl_idx, c->tag, (uint32_t)c->N, cnt);
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

int launch_export_pairs_fill(md_ctx *c, const uint64_t *off, uint32_t *pairs)
{
    k_pairs_fill<<<md_grid(c->N, 128), 128, 0, c->stream>>>(c->nl_cnt_exp, c->nl_off, c->nl_idx, c->tag, (uint32_t)c->N, off,
                                                           pairs);
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

__global__ void k_rows(const uint32_t *__restrict__ probe, uint32_t n_probe, const uint32_t *__restrict__ rtag,
                       const uint32_t *__restrict__ nl_cnt, const uint64_t *__restrict__ nl_off,
                       const uint32_t *__restrict__ nl_idx, const uint32_t *__restrict__ tag, uint32_t N,
                       uint32_t *counts, uint32_t *nbr, uint32_t stride)
{
    const uint32_t p = blockIdx.x;
    if (p >= n_probe) return;
    const uint32_t t = probe[p];
    if (t >= N) { if (threadIdx.x == 0) counts[p] = 0xffffffffu; return; }
    const uint32_t i = rtag[t], n = nl_cnt[i];
    const uint64_t row = nl_off[i];
    if (threadIdx.x == 0) counts[p] = n;
    for (uint32_t m = threadIdx.x; m < n && m < stride; m += blockDim.x) nbr[(uint64_t)p * stride + m] = tag[nl_idx[row + m]];
}

int launch_export_rows(md_ctx *c, const uint32_t *probe_tags, uint32_t n_probe, uint32_t *counts, uint32_t *nbr,
                       uint32_t stride)
{
    if (n_probe == 0) return MD_OK;
    k_rows<<<n_probe, 64, 0, c->stream>>>(probe_tags, n_probe, c->rtag, c->nl_cnt_exp, c->nl_off, c->nl_idx, c->tag,
                                          (uint32_t)c->N, counts, nbr, stride);
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}
