// tiles.cu -- the B200 hot path: cell-brick ("tile") kernels with the stencil staged in shared memory.
//
// Particles are stored sorted by cell along the Morton curve, so a brick of B^3 cells (B = 1, 2, 4) is one contiguous
// range of particles ("home" particles) and one CTA owns it.  The CTA stages every particle of the (B+2)^3 stencil
// cells in shared memory as coordinates RELATIVE to the brick centre with the periodic image already applied
// ("Look up cell neighbors"; north_star "cell-neighbor stencils staged in shared memory").  Consequences:
//   * neighbour-list entries are 16-bit indices into the staged block, not 32-bit global indices: the index stream,
//     which dominates the algorithmic HBM bytes, is halved;
//   * every neighbour gather is a shared-memory load, never an L2/HBM access;
//   * no minimum-image arithmetic per pair: the image is applied once per staged particle;
//   * in MD_MIXED the staged coordinates are fp32 and small (|x| < ~2 cell widths), so separations keep ~1e-7
//     absolute accuracy although absolute coordinates would not (hard part 3).
// Decisions (r^2 < r_list^2 at build time, r^2 < rc^2 in the force kernels) are taken on the staged coordinates only
// when they are outside a guard band around the threshold that bounds the staging error; inside the band the pair
// is re-tested with the exact fp64 expression of DESIGN.md R2 on the global positions, so lists and cut-off
// decisions are those of the plain definition, bit for bit.
//
// Neighbour-list build (Fig. 4) with w = 32: a warp strides over the 9 x-runs of the 27 stencil
// cells, one ballot per 32 candidates (Fig. 4 steps 2-3), for BUILD_P home particles of one cell at a time (the
// candidate is loaded once and tested against BUILD_P particles held in registers).  The ballot words are kept in
// shared memory; per chunk of particles the CTA scans the row lengths, reserves the rows in the global array with ONE
// atomicAdd (placement only: content and order of every row are deterministic) and writes the rows compacted by
// popc prefix sums (steps 4-8), one lane per ballot word: no second distance pass, no per-entry atomics.
#include <algorithm>
#include <type_traits>

#include "md_device.cuh"

constexpr int TILE_MAX_BLOCK = 512;  // __launch_bounds__ of the tile kernels (up to 128 registers per thread)
constexpr int BUILD_P = 4;           // home particles per warp task in the build kernel

struct TileParams {
    uint32_t B;        // brick edge in cells
    uint32_t nsc_max;  // (B+2)^3
    uint32_t n_tiles;
    const uint32_t *tile_cell_begin;  // [n_tiles+1] first cell rank of each tile
    const uint32_t *tile_origin;      // [3 n_tiles] lowest cell coordinate of the brick
    const uint32_t *lin_of_rank;      // cell rank -> linear id
    const uint32_t *rank_of_lin;      // linear id -> cell rank
    const uint32_t *cell_start;       // [n_cells+1] first particle slot of each cell rank
    double cw[3];                     // cell widths
};

struct TileCtx {
    uint32_t x0, y0, z0, ex, ey, ez, sx, sy, sz, n_sc, n_staged, n_home, g0, cb, n_hc;
};

// shared-memory header, carved from the dynamic allocation (sizes depend on the brick)
struct TileSmem {
    uint32_t *gstart;   // [nsc]   global slot of the first particle of each staged cell
    uint32_t *sstart;   // [nsc+1] staged index of the first particle of each staged cell
    uint32_t *hc_sc;    // [B^3]   staged-cell index of each home cell
    uint32_t *hc_first; // [B^3+1] first home particle (tile-local) of each home cell
    double *cgeo;       // [nsc*6] per staged cell: centre inside the box (3), centre of its image rel. brick centre (3)
    char *rest;         // records etc.
};

__host__ __device__ inline size_t tile_header_bytes(uint32_t B)
{
    const size_t nsc = (size_t)(B + 2) * (B + 2) * (B + 2), nhc = (size_t)B * B * B;
    size_t b = sizeof(uint32_t) * (nsc + (nsc + 1) + nhc + (nhc + 1));
    b = (b + 15) & ~(size_t)15;
    b += sizeof(double) * 6 * nsc;
    return (b + 15) & ~(size_t)15;
}

__device__ __forceinline__ TileSmem tile_carve(char *smem, uint32_t B)
{
    const uint32_t nsc = (B + 2) * (B + 2) * (B + 2), nhc = B * B * B;
    TileSmem t;
    t.gstart = (uint32_t *)smem;
    t.sstart = t.gstart + nsc;
    t.hc_sc = t.sstart + nsc + 1;
    t.hc_first = t.hc_sc + nhc;
    size_t b = sizeof(uint32_t) * (nsc + (nsc + 1) + nhc + (nhc + 1));
    b = (b + 15) & ~(size_t)15;
    t.cgeo = (double *)(smem + b);
    t.rest = smem + tile_header_bytes(B);
    return t;
}

// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void tile_setup(const TileParams &tp, const Geom &g, uint32_t t, const TileSmem &h, TileCtx &tc)
{
    tc.x0 = tp.tile_origin[3 * t];
    tc.y0 = tp.tile_origin[3 * t + 1];
    tc.z0 = tp.tile_origin[3 * t + 2];
    tc.ex = min(tp.B, g.n[0] - tc.x0);
    tc.ey = min(tp.B, g.n[1] - tc.y0);
    tc.ez = min(tp.B, g.n[2] - tc.z0);
    tc.sx = tc.ex + 2;
    tc.sy = tc.ey + 2;
    tc.sz = tc.ez + 2;
    tc.n_sc = tc.sx * tc.sy * tc.sz;
    tc.cb = tp.tile_cell_begin[t];
    tc.n_hc = tp.tile_cell_begin[t + 1] - tc.cb;
    tc.g0 = tp.cell_start[tc.cb];
    tc.n_home = tp.cell_start[tc.cb + tc.n_hc] - tc.g0;
    for (uint32_t sc = threadIdx.x; sc < tc.n_sc; sc += blockDim.x) {
        const uint32_t ix = sc % tc.sx, iy = (sc / tc.sx) % tc.sy, iz = sc / (tc.sx * tc.sy);
        const uint32_t cx = (tc.x0 + ix + g.n[0] - 1) % g.n[0];
        const uint32_t cy = (tc.y0 + iy + g.n[1] - 1) % g.n[1];
        const uint32_t cz = (tc.z0 + iz + g.n[2] - 1) % g.n[2];
        const uint32_t r = tp.rank_of_lin[cx + g.n[0] * (cy + g.n[1] * cz)];
        const uint32_t gs = tp.cell_start[r];
        h.gstart[sc] = gs;
        h.sstart[sc] = tp.cell_start[r + 1] - gs;  // count for now
        double *cg = h.cgeo + 6 * sc;
        cg[0] = g.lo[0] + ((double)cx + 0.5) * tp.cw[0];
        cg[1] = g.lo[1] + ((double)cy + 0.5) * tp.cw[1];
        cg[2] = g.lo[2] + ((double)cz + 0.5) * tp.cw[2];
        cg[3] = ((double)ix - 0.5 - 0.5 * (double)tc.ex) * tp.cw[0];
        cg[4] = ((double)iy - 0.5 - 0.5 * (double)tc.ey) * tp.cw[1];
        cg[5] = ((double)iz - 0.5 - 0.5 * (double)tc.ez) * tp.cw[2];
    }
    // home cells (consecutive ranks): their staged-cell index and first tile-local particle
    for (uint32_t hc = threadIdx.x; hc <= tc.n_hc; hc += blockDim.x) {
        const uint32_t r = tc.cb + hc;
        h.hc_first[hc] = tp.cell_start[r] - tc.g0;
        if (hc < tc.n_hc) {
            const uint32_t lin = tp.lin_of_rank[r];
            const uint32_t cx = lin % g.n[0], cy = (lin / g.n[0]) % g.n[1], cz = lin / (g.n[0] * g.n[1]);
            h.hc_sc[hc] = (cx - tc.x0 + 1) + tc.sx * ((cy - tc.y0 + 1) + tc.sy * (cz - tc.z0 + 1));
        }
    }
    __syncthreads();
    if (threadIdx.x < 32) {  // exclusive scan of the counts by warp 0
        uint32_t carry = 0;
        for (uint32_t base = 0; base < tc.n_sc; base += 32) {
            const uint32_t sc = base + threadIdx.x;
            const uint32_t v = sc < tc.n_sc ? h.sstart[sc] : 0u;
            uint32_t inc = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t u = __shfl_up_sync(0xffffffffu, inc, o);
                if ((int)threadIdx.x >= o) inc += u;
            }
            if (sc < tc.n_sc) h.sstart[sc] = carry + inc - v;
            carry += __shfl_sync(0xffffffffu, inc, 31);
        }
        if (threadIdx.x == 0) h.sstart[tc.n_sc] = carry;
    }
    __syncthreads();
    tc.n_staged = h.sstart[tc.n_sc];
}

// staged cell that holds staged index s (binary search over sstart[0..n_sc])
__device__ __forceinline__ uint32_t tile_cell_of_staged(const TileSmem &h, uint32_t n_sc, uint32_t s)
{
    uint32_t lo = 0, hi = n_sc;  // invariant: sstart[lo] <= s < sstart[hi]
    while (hi - lo > 1) {
        const uint32_t mid = (lo + hi) >> 1;
        if (h.sstart[mid] <= s) lo = mid; else hi = mid;
    }
    return lo;
}

// home cell of tile-local home particle p (n_hc <= 64)
__device__ __forceinline__ uint32_t tile_home_cell(const TileSmem &h, uint32_t n_hc, uint32_t p)
{
    uint32_t lo = 0, hi = n_hc;
    while (hi - lo > 1) {
        const uint32_t mid = (lo + hi) >> 1;
        if (h.hc_first[mid] <= p) lo = mid; else hi = mid;
    }
    return lo;
}

// staged index of tile-local home particle p that lives in home cell hc
__device__ __forceinline__ uint32_t tile_staged_of_home(const TileSmem &h, uint32_t hc, uint32_t p)
{
    return h.sstart[h.hc_sc[hc]] + (p - h.hc_first[hc]);
}

template <typename R4> struct RecTraits;
template <> struct RecTraits<float4> {
    typedef float real;
    static __device__ __forceinline__ float4 make(double x, double y, double z, double w) { return make_float4((float)x, (float)y, (float)z, 0.f); }
    static __device__ __forceinline__ float4 far(float s) { return make_float4(s * 1e15f, s * 1e15f, s * 1e15f, 0.f); }
};
template <> struct RecTraits<double4> {
    typedef double real;
    static __device__ __forceinline__ double4 make(double x, double y, double z, double w) { return make_double4(x, y, z, w); }
    static __device__ __forceinline__ double4 far(double s) { return make_double4(s * 1e150, s * 1e150, s * 1e150, 0.0); }
};

// stage every stencil particle: coordinates relative to the brick centre, periodic image applied.
// x_staged = c_s + minimg(x - C_w): C_w = centre of the particle's cell inside the box, c_s = centre of that cell's
// image relative to the brick centre.  |x - C_w| <= w/2 + drift << L/2, so this also undoes an integrator wrap.
template <typename R4, bool WITH_VEL>
__device__ __forceinline__ void tile_stage(const Geom &g, const TileCtx &tc, const TileSmem &h,
                                           const double4 *__restrict__ pos, const double4 *__restrict__ vel, R4 *rec,
                                           double4 *svel)
{
    for (uint32_t s = threadIdx.x; s < tc.n_staged; s += blockDim.x) {
        const uint32_t sc = tile_cell_of_staged(h, tc.n_sc, s);
        const uint32_t gi = h.gstart[sc] + (s - h.sstart[sc]);
        const double4 p = pos[gi];
        const double *cg = h.cgeo + 6 * sc;
        const double x = cg[3] + md_min_image(p.x - cg[0], g.L[0], g.h[0]);
        const double y = cg[4] + md_min_image(p.y - cg[1], g.L[1], g.h[1]);
        const double z = cg[5] + md_min_image(p.z - cg[2], g.L[2], g.h[2]);
        rec[s] = RecTraits<R4>::make(x, y, z, p.w);
        if (WITH_VEL) svel[s] = vel[gi];
    }
    if (threadIdx.x == 0) rec[tc.n_staged] = RecTraits<R4>::far(1);  // dummy record for row padding
}

// global slot of staged index s
__device__ __forceinline__ uint32_t tile_global_of_staged(const TileSmem &h, uint32_t n_sc, uint32_t s)
{
    const uint32_t sc = tile_cell_of_staged(h, n_sc, s);
    return h.gstart[sc] + (s - h.sstart[sc]);
}

// the plain definition on the global (wrapped) positions: exact fp64, no FMA (R2, R8)
__device__ __noinline__ double tile_exact_r2_impl(const double4 *__restrict__ pos, double Lx, double Ly, double Lz,
                                                  uint32_t gi, uint32_t gj)
{
    const double4 a = pos[gi], b = pos[gj];
    const double dx = md_min_image(__dsub_rn(a.x, b.x), Lx, 0.5 * Lx);
    const double dy = md_min_image(__dsub_rn(a.y, b.y), Ly, 0.5 * Ly);
    const double dz = md_min_image(__dsub_rn(a.z, b.z), Lz, 0.5 * Lz);
    return md_r2_exact(dx, dy, dz);
}
__device__ __forceinline__ double tile_exact_r2(const double4 *__restrict__ pos, const Geom &g, uint32_t gi, uint32_t gj)
{
    return tile_exact_r2_impl(pos, g.L[0], g.L[1], g.L[2], gi, gj);
}

// ===============================================================================================================
// sizes of the largest tile (for shared-memory sizing), one thread per tile
// ===============================================================================================================
__global__ void k_tile_sizes(TileParams tp, Geom g, unsigned int *max_home, unsigned int *max_staged)
{
    const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= tp.n_tiles) return;
    const uint32_t x0 = tp.tile_origin[3 * t], y0 = tp.tile_origin[3 * t + 1], z0 = tp.tile_origin[3 * t + 2];
    const uint32_t sx = min(tp.B, g.n[0] - x0) + 2, sy = min(tp.B, g.n[1] - y0) + 2, sz = min(tp.B, g.n[2] - z0) + 2;
    uint32_t staged = 0;
    for (uint32_t iz = 0; iz < sz; ++iz)
        for (uint32_t iy = 0; iy < sy; ++iy)
            for (uint32_t ix = 0; ix < sx; ++ix) {
                const uint32_t cx = (x0 + ix + g.n[0] - 1) % g.n[0], cy = (y0 + iy + g.n[1] - 1) % g.n[1],
                               cz = (z0 + iz + g.n[2] - 1) % g.n[2];
                const uint32_t r = tp.rank_of_lin[cx + g.n[0] * (cy + g.n[1] * cz)];
                staged += tp.cell_start[r + 1] - tp.cell_start[r];
            }
    const uint32_t cb = tp.tile_cell_begin[t], ce = tp.tile_cell_begin[t + 1];
    atomicMax(max_home, tp.cell_start[ce] - tp.cell_start[cb]);
    atomicMax(max_staged, staged);
}

// ===============================================================================================================
// S2 neighbour-list build, one CTA per tile
// ===============================================================================================================
template <typename R4>
__global__ void __launch_bounds__(TILE_MAX_BLOCK) k_tile_build(TileParams tp, Geom g, const double4 *__restrict__ pos,
                                                               typename RecTraits<R4>::real thr_in,
                                                               typename RecTraits<R4>::real thr_out, double rl2_exact,
                                                               uint32_t wpr /* ballot words per x-run */,
                                                               uint32_t max_staged, unsigned long long *cursor,
                                                               unsigned long long capacity, uint32_t *row_off,
                                                               uint32_t *nl_cnt, uint16_t *nl16)
{
    typedef typename RecTraits<R4>::real real;
    extern __shared__ __align__(16) char smem_raw[];
    const TileSmem h = tile_carve(smem_raw, tp.B);
    R4 *rec = (R4 *)h.rest;
    const uint32_t nw = blockDim.x >> 5;
    const uint32_t chunk = nw * BUILD_P;  // home particles per chunk
    uint32_t *counts = (uint32_t *)(h.rest + sizeof(R4) * (max_staged + 1));  // [chunk] counts, then row offsets
    uint32_t *words = counts + chunk;                                         // [chunk * 9 * wpr]
    __shared__ unsigned long long s_base;
    __shared__ uint32_t s_ok;

    TileCtx tc;
    tile_setup(tp, g, blockIdx.x, h, tc);
    tile_stage<R4, false>(g, tc, h, pos, nullptr, rec, nullptr);
    __syncthreads();

    const unsigned lane = threadIdx.x & 31u, wid = threadIdx.x >> 5;
    const uint32_t wpp = 9 * wpr;

    // tasks: groups of BUILD_P consecutive particles of one home cell
    uint32_t n_tasks = 0;
    for (uint32_t hc = 0; hc < tc.n_hc; ++hc) n_tasks += (h.hc_first[hc + 1] - h.hc_first[hc] + BUILD_P - 1) / BUILD_P;

    for (uint32_t task0 = 0; task0 < n_tasks; task0 += nw) {
        // ---- pass A: hit masks (Fig. 4 steps 1-3); warp `wid` takes task task0 + wid
        const uint32_t task = task0 + wid;
        uint32_t hc = 0, p0 = 0, np = 0;  // home cell, first particle (tile-local), particles in this task
        if (task < n_tasks) {
            uint32_t t = task;
            for (hc = 0; hc < tc.n_hc; ++hc) {
                const uint32_t nt = (h.hc_first[hc + 1] - h.hc_first[hc] + BUILD_P - 1) / BUILD_P;
                if (t < nt) break;
                t -= nt;
            }
            p0 = h.hc_first[hc] + t * BUILD_P;
            np = min((uint32_t)BUILD_P, h.hc_first[hc + 1] - p0);
        }
        uint32_t cnt[BUILD_P];
#pragma unroll
        for (int q = 0; q < BUILD_P; ++q) cnt[q] = 0;
        if (np > 0) {
            const uint32_t sch = h.hc_sc[hc];
            const uint32_t ixh = sch % tc.sx, iyh = (sch / tc.sx) % tc.sy, izh = sch / (tc.sx * tc.sy);
            const uint32_t self0 = h.sstart[sch] + (p0 - h.hc_first[hc]);
            R4 me[BUILD_P];
#pragma unroll
            for (int q = 0; q < BUILD_P; ++q) me[q] = (uint32_t)q < np ? rec[self0 + q] : RecTraits<R4>::far(-1);
            uint32_t *wp = words + (size_t)wid * BUILD_P * wpp;
#pragma unroll 1
            for (int run = 0; run < 9; ++run) {
                const uint32_t iy = iyh + (run % 3) - 1, iz = izh + (run / 3) - 1;
                const uint32_t sc0 = (ixh - 1) + tc.sx * (iy + tc.sy * iz);
                const uint32_t b = h.sstart[sc0], e = h.sstart[sc0 + 3];
                uint32_t k = run * wpr;
                for (uint32_t base = b; base < e; base += 32, ++k) {
                    const uint32_t j = base + lane;
                    const bool valid = j < e;
                    const R4 pj = rec[valid ? j : tc.n_staged];  // past the run: the far-away dummy record
                    unsigned bal[BUILD_P];
#pragma unroll
                    for (int q = 0; q < BUILD_P; ++q) {
                        const real dx = me[q].x - pj.x, dy = me[q].y - pj.y, dz = me[q].z - pj.z;
                        const real r2 = dx * dx + dy * dy + dz * dz;
                        bool hit = r2 < thr_in && j != self0 + q;
                        if (r2 >= thr_in && r2 < thr_out && j != self0 + q) {
                            // guard band: decide with the exact definition
                            const uint32_t scj = j >= h.sstart[sc0 + 2] ? sc0 + 2 : (j >= h.sstart[sc0 + 1] ? sc0 + 1 : sc0);
                            const uint32_t gj = h.gstart[scj] + (j - h.sstart[scj]);
                            hit = tile_exact_r2(pos, g, tc.g0 + p0 + q, gj) < rl2_exact;
                        }
                        bal[q] = __ballot_sync(0xffffffffu, hit);
                        cnt[q] += __popc(bal[q]);
                    }
                    if (lane < BUILD_P) {
                        unsigned v = bal[0];
#pragma unroll
                        for (int q = 1; q < BUILD_P; ++q) v = lane == (unsigned)q ? bal[q] : v;
                        wp[lane * wpp + k] = v;
                    }
                }
                for (; k < (uint32_t)(run + 1) * wpr; ++k)
                    if (lane < BUILD_P) wp[lane * wpp + k] = 0u;
            }
        }
        if (lane < BUILD_P) {
            uint32_t v = cnt[0];
#pragma unroll
            for (int q = 1; q < BUILD_P; ++q) v = lane == (unsigned)q ? cnt[q] : v;
            counts[wid * BUILD_P + lane] = lane < np ? v : 0u;
        }
        __syncthreads();

        // ---- row offsets of the chunk (rows padded to 8 entries = 16 bytes), one reservation per chunk
        if (wid == 0) {
            uint32_t carry = 0;
            for (uint32_t base = 0; base < chunk; base += 32) {
                const uint32_t c = base + lane < chunk ? counts[base + lane] : 0u;
                const uint32_t v = (c + 7u) >> 3;
                uint32_t inc = v;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const uint32_t u = __shfl_up_sync(0xffffffffu, inc, o);
                    if ((int)lane >= o) inc += u;
                }
                if (base + lane < chunk) counts[base + lane] = (carry + inc - v) | (c << 20);  // offset | count
                carry += __shfl_sync(0xffffffffu, inc, 31);
            }
            if (lane == 0) {
                const unsigned long long tot = 8ull * carry;
                const unsigned long long bb = atomicAdd(cursor, tot);
                s_base = bb;
                s_ok = (bb + tot <= capacity) ? 1u : 0u;  // no room: host sees cursor > capacity, grows, rebuilds
            }
        }
        __syncthreads();

        // ---- pass B: compacted write (Fig. 4 steps 4-8): warp per particle, lane per ballot word
        if (s_ok && np > 0) {
            const uint32_t sch = h.hc_sc[hc];
            const uint32_t ixh = sch % tc.sx, iyh = (sch / tc.sx) % tc.sy, izh = sch / (tc.sx * tc.sy);
            for (uint32_t q = 0; q < np; ++q) {
                const uint32_t oc = counts[wid * BUILD_P + q];
                const uint32_t off8 = oc & 0xfffffu, n_tot = oc >> 20;
                const unsigned long long row0 = s_base + 8ull * off8;
                uint16_t *row = nl16 + row0;
                const uint32_t *wp = words + ((size_t)wid * BUILD_P + q) * wpp;
                uint32_t carry = 0;
                for (uint32_t wbase = 0; wbase < wpp; wbase += 32) {
                    const uint32_t wi = wbase + lane;
                    unsigned bits = wi < wpp ? wp[wi] : 0u;
                    const uint32_t c = __popc(bits);
                    uint32_t inc = c;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const uint32_t u = __shfl_up_sync(0xffffffffu, inc, o);
                        if ((int)lane >= o) inc += u;
                    }
                    uint32_t o = carry + inc - c;
                    if (bits) {
                        const uint32_t run = wi / wpr, k = wi - run * wpr;
                        const uint32_t iy = iyh + (run % 3) - 1, iz = izh + (run / 3) - 1;
                        const uint32_t sc0 = (ixh - 1) + tc.sx * (iy + tc.sy * iz);
                        const uint32_t jb = h.sstart[sc0] + 32u * k;
                        while (bits) {
                            const uint32_t bpos = __ffs(bits) - 1;
                            bits &= bits - 1;
                            row[o++] = (uint16_t)(jb + bpos);
                        }
                    }
                    carry += __shfl_sync(0xffffffffu, inc, 31);
                }
                const uint32_t padded = (n_tot + 7u) & ~7u;
                if (n_tot + lane < padded) row[n_tot + lane] = (uint16_t)tc.n_staged;  // dummy record (far away)
                if (lane == 0) {
                    row_off[tc.g0 + p0 + q] = (uint32_t)(row0 >> 3);
                    nl_cnt[tc.g0 + p0 + q] = n_tot;
                }
            }
        }
        __syncthreads();
    }
}

// ===============================================================================================================
// S4a LJ forces, one CTA per tile, W threads per home particle
// ===============================================================================================================
struct LJTile {
    double rc2_exact, sig2, eps24, eps4, uc;
    double thr_in, thr_out;  // rc^2 -+ guard
};

template <int W, bool MIXED, int ACC_BLOCK>
__global__ void __launch_bounds__(TILE_MAX_BLOCK) k_tile_lj(TileParams tp, Geom g, const double4 *__restrict__ pos,
                                                            const uint32_t *__restrict__ row_off,
                                                            const uint32_t *__restrict__ nl_cnt,
                                                            const uint16_t *__restrict__ nl16, LJTile lj,
                                                            uint32_t max_staged, double4 *__restrict__ force)
{
    typedef typename std::conditional<MIXED, float4, double4>::type R4;
    typedef typename RecTraits<R4>::real real;
    extern __shared__ __align__(16) char smem_raw[];
    const TileSmem h = tile_carve(smem_raw, tp.B);
    R4 *rec = (R4 *)h.rest;

    TileCtx tc;
    tile_setup(tp, g, blockIdx.x, h, tc);
    tile_stage<R4, false>(g, tc, h, pos, nullptr, rec, nullptr);
    __syncthreads();

    const unsigned lane = threadIdx.x & (W - 1);
    const unsigned seg_mask = md_seg_mask<W>();
    const uint32_t n_groups = blockDim.x / W;
    const real thr_in = (real)lj.thr_in, thr_out = (real)lj.thr_out;
    const real sig2 = (real)lj.sig2, eps24 = (real)lj.eps24, eps4 = (real)lj.eps4, uc = (real)lj.uc;

    for (uint32_t p = threadIdx.x / W; p < tc.n_home; p += n_groups) {
        const uint32_t hc = tile_home_cell(h, tc.n_hc, p);
        const R4 me = rec[tile_staged_of_home(h, hc, p)];
        const uint32_t cnt = nl_cnt[tc.g0 + p];
        const uint32_t nblk = (cnt + 7u) >> 3;
        const uint4 *row = (const uint4 *)(nl16 + 8ull * row_off[tc.g0 + p]);
        double fx = 0.0, fy = 0.0, fz = 0.0, en = 0.0;
        for (uint32_t b = lane; b < nblk; b += W) {
            const uint4 q = __ldg(row + b);
            const uint32_t qq[4] = {q.x, q.y, q.z, q.w};
            real ax = 0, ay = 0, az = 0, ae = 0;
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                const uint32_t j = (qq[e >> 1] >> ((e & 1) * 16)) & 0xffffu;
                const R4 pj = rec[j];
                const real dx = me.x - pj.x, dy = me.y - pj.y, dz = me.z - pj.z;
                const real r2 = dx * dx + dy * dy + dz * dz;
                bool in = r2 < thr_in;
                if (!in && r2 < thr_out) {  // guard band around rc^2: the plain fp64 definition decides (R26)
                    in = tile_exact_r2(pos, g, tc.g0 + p, tile_global_of_staged(h, tc.n_sc, j)) < lj.rc2_exact;
                }
                const real rinv2 = md_rcp(r2);
                const real s2 = sig2 * rinv2;
                const real s6 = s2 * s2 * s2;
                real f = eps24 * s6 * ((real)2 * s6 - (real)1) * rinv2;
                real u = (real)0.5 * (eps4 * s6 * (s6 - (real)1) - uc);
                f = in ? f : (real)0;
                u = in ? u : (real)0;
                ax += f * dx; ay += f * dy; az += f * dz; ae += u;
                if (MIXED && ((e + 1) % ACC_BLOCK == 0)) {  // widen the fp32 block sum, accumulate in fp64
                    fx += (double)ax; fy += (double)ay; fz += (double)az; en += (double)ae;
                    ax = ay = az = ae = 0;
                }
            }
            if (!MIXED) { fx += ax; fy += ay; fz += az; en += ae; }
        }
        fx = md_seg_sum<W>(fx, seg_mask);
        fy = md_seg_sum<W>(fy, seg_mask);
        fz = md_seg_sum<W>(fz, seg_mask);
        en = md_seg_sum<W>(en, seg_mask);
        if (lane == 0) force[tc.g0 + p] = make_double4(fx, fy, fz, en);
    }
}

// ===============================================================================================================
// S4b DPD forces, one CTA per tile, W threads per home particle, fp64; positions, velocities and tags staged
// ===============================================================================================================
struct DPDTile {
    double rc2_exact, inv_rc, rc, A, gamma, sr, thr_in, thr_out;
    uint64_t step, seed;
};

template <int W>
__global__ void __launch_bounds__(TILE_MAX_BLOCK) k_tile_dpd(TileParams tp, Geom g, const double4 *__restrict__ pos,
                                                             const double4 *__restrict__ vel,
                                                             const uint32_t *__restrict__ row_off,
                                                             const uint32_t *__restrict__ nl_cnt,
                                                             const uint16_t *__restrict__ nl16, DPDTile dp,
                                                             uint32_t max_staged, double4 *__restrict__ force)
{
    extern __shared__ __align__(16) char smem_raw[];
    const TileSmem h = tile_carve(smem_raw, tp.B);
    double4 *rec = (double4 *)h.rest;
    double4 *svel = rec + (max_staged + 1);

    TileCtx tc;
    tile_setup(tp, g, blockIdx.x, h, tc);
    tile_stage<double4, true>(g, tc, h, pos, vel, rec, svel);
    if (threadIdx.x == 0) svel[tc.n_staged] = make_double4(0, 0, 0, 1);
    __syncthreads();

    const unsigned lane = threadIdx.x & (W - 1);
    const unsigned seg_mask = md_seg_mask<W>();
    const uint32_t n_groups = blockDim.x / W;

    for (uint32_t p = threadIdx.x / W; p < tc.n_home; p += n_groups) {
        const uint32_t hc = tile_home_cell(h, tc.n_hc, p);
        const uint32_t self = tile_staged_of_home(h, hc, p);
        const double4 me = rec[self];
        const double4 vi = svel[self];
        const uint32_t ti = md_lane_to_tag(me.w);
        const uint32_t cnt = nl_cnt[tc.g0 + p];
        const uint32_t nblk = (cnt + 7u) >> 3;
        const uint4 *row = (const uint4 *)(nl16 + 8ull * row_off[tc.g0 + p]);
        double fx = 0.0, fy = 0.0, fz = 0.0, en = 0.0;
        for (uint32_t b = lane; b < nblk; b += W) {
            const uint4 q = __ldg(row + b);
            const uint32_t qq[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                const uint32_t j = (qq[e >> 1] >> ((e & 1) * 16)) & 0xffffu;
                const double4 pj = rec[j];
                const double dx = me.x - pj.x, dy = me.y - pj.y, dz = me.z - pj.z;
                const double r2 = dx * dx + dy * dy + dz * dz;
                bool in = r2 < dp.thr_in;
                if (!in && r2 < dp.thr_out)
                    in = tile_exact_r2(pos, g, tc.g0 + p, tile_global_of_staged(h, tc.n_sc, j)) < dp.rc2_exact;
                if (in && r2 > 0.0) {
                    const double4 vj = svel[j];
                    const double rinv = rsqrt(r2);
                    const double r = r2 * rinv;
                    const double w = 1.0 - r * dp.inv_rc;
                    const double rv = (dx * (vi.x - vj.x) + dy * (vi.y - vj.y) + dz * (vi.z - vj.z)) * rinv;
                    const double theta = md_dpd_theta(ti, md_lane_to_tag(pj.w), dp.step, dp.seed);
                    const double f = (dp.A * w - dp.gamma * w * w * rv + dp.sr * w * theta) * rinv;
                    fx += f * dx; fy += f * dy; fz += f * dz;
                    en += 0.25 * dp.A * dp.rc * w * w;
                }
            }
        }
        fx = md_seg_sum<W>(fx, seg_mask);
        fy = md_seg_sum<W>(fy, seg_mask);
        fz = md_seg_sum<W>(fz, seg_mask);
        en = md_seg_sum<W>(en, seg_mask);
        if (lane == 0) force[tc.g0 + p] = make_double4(fx, fy, fz, en);
    }
}

// ===============================================================================================================
// decode the 16-bit tile list into the general 32-bit CSR (exports / parity read-back only)
// ===============================================================================================================
__global__ void k_tile_decode(TileParams tp, Geom g, const uint32_t *__restrict__ row_off,
                              const uint32_t *__restrict__ nl_cnt, const uint16_t *__restrict__ nl16,
                              const uint64_t *__restrict__ nl_off, uint32_t *nl_idx)
{
    extern __shared__ __align__(16) char smem_raw[];
    const TileSmem h = tile_carve(smem_raw, tp.B);
    TileCtx tc;
    tile_setup(tp, g, blockIdx.x, h, tc);
    const unsigned lane = threadIdx.x & 31u, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    for (uint32_t p = wid; p < tc.n_home; p += nw) {
        const uint32_t cnt = nl_cnt[tc.g0 + p];
        const uint16_t *row = nl16 + 8ull * row_off[tc.g0 + p];
        uint32_t *out = nl_idx + nl_off[tc.g0 + p];
        for (uint32_t k = lane; k < cnt; k += 32) out[k] = tile_global_of_staged(h, tc.n_sc, row[k]);
    }
}

// ===============================================================================================================
// host side
// ===============================================================================================================
static TileParams make_tp(md_ctx *c)
{
    TileParams tp;
    tp.B = c->tile_B;
    tp.nsc_max = (c->tile_B + 2) * (c->tile_B + 2) * (c->tile_B + 2);
    tp.n_tiles = c->n_tiles;
    tp.tile_cell_begin = c->tile_cell_begin;
    tp.tile_origin = c->tile_origin;
    tp.lin_of_rank = c->lin_of_rank;
    tp.rank_of_lin = c->rank_of_lin;
    tp.cell_start = c->cell_start;
    for (int a = 0; a < 3; ++a) tp.cw[a] = c->box[a] / (double)c->dims[a];
    return tp;
}

// bound on |r2_staged - r2_true| for staged coordinates of magnitude <= E, separations <= R (see file header)
static double guard_fp32(double E, double R)
{
    const double u = 5.9604644775390625e-08;  // 2^-24
    const double delta = 2.0 * E * u + u * R;
    return 1.5 * (2.0 * 1.7320508075688772 * R * delta + 3.0 * delta * delta + 4.0 * u * R * R);
}
static double guard_fp64(double E, double R)
{
    const double u = 1.1102230246251565e-16;  // 2^-53
    const double delta = 6.0 * E * u + u * R;
    return 4.0 * (2.0 * 1.7320508075688772 * R * delta + 3.0 * delta * delta + 4.0 * u * R * R);
}
static double tile_extent(md_ctx *c)
{
    double E = 0.0;
    for (int a = 0; a < 3; ++a) E = std::max(E, (0.5 * c->tile_B + 1.0) * c->box[a] / c->dims[a] + c->r_buff + 1e-6);
    return E;
}

static size_t tile_smem_common(md_ctx *c, size_t rec_bytes, bool with_vel)
{
    size_t s = tile_header_bytes(c->tile_B);
    s += rec_bytes * (c->tile_max_staged + 1);
    if (with_vel) s += sizeof(double4) * (c->tile_max_staged + 1);
    return s;
}

int tile_measure(md_ctx *c)
{
    MD_CUDA_CHECK(c, cudaMemsetAsync(&c->d_flags->max_home, 0, 2 * sizeof(unsigned int), c->stream));
    k_tile_sizes<<<md_grid(c->n_tiles, 128), 128, 0, c->stream>>>(make_tp(c), c->g, &c->d_flags->max_home, &c->d_flags->max_staged);
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

template <typename K>
static int set_smem(md_ctx *c, K kernel, size_t bytes)
{
    if (bytes > 48 * 1024) MD_CUDA_CHECK(c, cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    return MD_OK;
}

static const size_t TILE_SMEM_LIMIT = 227 * 1024 - 64;

// returns MD_OK and sets *fits = false if the largest tile does not fit in shared memory (caller falls back)
int launch_tile_build(md_ctx *c, bool *fits)
{
    const bool f32 = c->precision == MD_MIXED;
    const uint32_t ms = c->tile_max_staged;
    const uint32_t wpr = std::max(1u, (3 * c->h_flags->max_cell_count + 31) / 32);
    const int block = std::min(c->cfg[MD_K_NLIST].block, TILE_MAX_BLOCK);
    const uint32_t chunk = (uint32_t)(block / 32) * BUILD_P;
    size_t smem = tile_smem_common(c, f32 ? sizeof(float4) : sizeof(double4), false);
    smem += sizeof(uint32_t) * chunk;                     // counts / row offsets
    smem += sizeof(uint32_t) * (size_t)chunk * 9 * wpr;   // ballot words
    // row offset and count share one word in the chunk scan: 20 bits of offset (units of 8), 12 bits of count
    const bool packable = (uint64_t)chunk * ((27ull * c->h_flags->max_cell_count + 7) / 8) < (1u << 20) &&
                          27ull * c->h_flags->max_cell_count < 4096;
    *fits = smem <= TILE_SMEM_LIMIT && ms < 65535 && packable;
    if (!*fits) return MD_OK;
    const double R = c->r_list * 1.001, E = tile_extent(c), rl2 = c->r_list * c->r_list;
    MD_CUDA_CHECK(c, cudaMemsetAsync(&c->d_flags->cursor, 0, sizeof(unsigned long long), c->stream));
    TileParams tp = make_tp(c);
    if (f32) {
        const double gd = guard_fp32(E, R);
        MD_TRY(set_smem(c, k_tile_build<float4>, smem));
        k_tile_build<float4><<<c->n_tiles, block, smem, c->stream>>>(tp, c->g, c->pos, (float)(rl2 - gd), (float)(rl2 + gd), rl2, wpr, ms,
                                                                    &c->d_flags->cursor, c->nl16_capacity, c->row_off, c->nl_cnt, c->nl16);
    } else {
        const double gd = guard_fp64(E, R);
        MD_TRY(set_smem(c, k_tile_build<double4>, smem));
        k_tile_build<double4><<<c->n_tiles, block, smem, c->stream>>>(tp, c->g, c->pos, rl2 - gd, rl2 + gd, rl2, wpr, ms,
                                                                     &c->d_flags->cursor, c->nl16_capacity, c->row_off, c->nl_cnt, c->nl16);
    }
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

int launch_tile_lj(md_ctx *c, double eps, double sigma, int shift)
{
    LaunchCfg cf = c->cfg[MD_K_LJ];
    cf.block = std::min(cf.block, TILE_MAX_BLOCK);
    const bool mixed = c->precision == MD_MIXED;
    LJTile p;
    p.rc2_exact = c->rc * c->rc;
    p.sig2 = sigma * sigma;
    p.eps24 = 24.0 * eps;
    p.eps4 = 4.0 * eps;
    p.uc = 0.0;
    if (shift) {
        const double s2 = p.sig2 / p.rc2_exact, s6 = s2 * s2 * s2;
        p.uc = 4.0 * eps * (s6 * s6 - s6);
    }
    const double E = tile_extent(c), R = c->rc * 1.001;
    const double gd = mixed ? guard_fp32(E, R) : guard_fp64(E, R);
    p.thr_in = p.rc2_exact - gd;
    p.thr_out = p.rc2_exact + gd;
    const size_t smem = tile_smem_common(c, mixed ? sizeof(float4) : sizeof(double4), false);
    TileParams tp = make_tp(c);
    MD_DISPATCH_W(cf.w, {
        if (mixed) {
            if (c->acc_block == 1) {
                MD_TRY(set_smem(c, k_tile_lj<W_, true, 1>, smem));
                k_tile_lj<W_, true, 1><<<c->n_tiles, cf.block, smem, c->stream>>>(tp, c->g, c->pos, c->row_off, c->nl_cnt, c->nl16, p,
                                                                               c->tile_max_staged, c->force);
            } else {
                MD_TRY(set_smem(c, k_tile_lj<W_, true, 8>, smem));
                k_tile_lj<W_, true, 8><<<c->n_tiles, cf.block, smem, c->stream>>>(tp, c->g, c->pos, c->row_off, c->nl_cnt, c->nl16, p,
                                                                               c->tile_max_staged, c->force);
            }
        } else {
            MD_TRY(set_smem(c, k_tile_lj<W_, false, 8>, smem));
            k_tile_lj<W_, false, 8><<<c->n_tiles, cf.block, smem, c->stream>>>(tp, c->g, c->pos, c->row_off, c->nl_cnt, c->nl16, p,
                                                                            c->tile_max_staged, c->force);
        }
    });
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

int launch_tile_dpd(md_ctx *c, double A, double gamma, double kT, double dt, uint64_t step, uint64_t seed)
{
    LaunchCfg cf = c->cfg[MD_K_DPD];
    cf.block = std::min(cf.block, TILE_MAX_BLOCK);
    DPDTile p;
    p.rc2_exact = c->rc * c->rc;
    p.inv_rc = 1.0 / c->rc;
    p.rc = c->rc;
    p.A = A;
    p.gamma = gamma;
    p.sr = sqrt(2.0 * gamma * kT) / sqrt(dt);
    p.step = step;
    p.seed = seed;
    const double gd = guard_fp64(tile_extent(c), c->rc * 1.001);
    p.thr_in = p.rc2_exact - gd;
    p.thr_out = p.rc2_exact + gd;
    const size_t smem = tile_smem_common(c, sizeof(double4), true);
    TileParams tp = make_tp(c);
    MD_DISPATCH_W(cf.w, {
        MD_TRY(set_smem(c, k_tile_dpd<W_>, smem));
        k_tile_dpd<W_><<<c->n_tiles, cf.block, smem, c->stream>>>(tp, c->g, c->pos, c->vel, c->row_off, c->nl_cnt, c->nl16, p,
                                                               c->tile_max_staged, c->force);
    });
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

bool tile_forces_fit(md_ctx *c, bool dpd)
{
    const size_t rec = (!dpd && c->precision == MD_MIXED) ? sizeof(float4) : sizeof(double4);
    return tile_smem_common(c, rec, dpd) <= TILE_SMEM_LIMIT;
}

int launch_tile_decode(md_ctx *c)
{
    const size_t smem = tile_header_bytes(c->tile_B);
    k_tile_decode<<<c->n_tiles, 256, smem, c->stream>>>(make_tp(c), c->g, c->row_off, c->nl_cnt, c->nl16, c->nl_off, c->nl_idx);
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}
