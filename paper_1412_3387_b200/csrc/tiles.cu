// tiles.cu -- the B200 hot path: cell-brick ("tile") kernels with the stencil staged in shared memory.
//
// Particles are stored sorted by cell along the Morton curve, so a brick of B^3 cells (B = 1, 2, 4) is one contiguous
// range of particles ("home" particles) and one CTA owns it.  The CTA stages every particle of the (B+2)^3 stencil
// cells in shared memory as coordinates RELATIVE to the brick centre with the periodic image already applied
// ("Look up cell neighbors"; north_star "cell-neighbor stencils staged in shared memory").  Consequences:
//   * neighbour-list entries are 16-bit references into the staged block, not 32-bit global indices: the index stream,
//     which dominates the algorithmic HBM bytes, is halved;
//   * every neighbour gather is a shared-memory load, never an L2/HBM access;
//   * no minimum-image arithmetic per pair: the image is applied once per staged particle;
//   * the staged coordinates are small (|x| < ~2.5 cell widths), so fp32 separations keep ~1e-6 absolute accuracy
//     although absolute fp32 coordinates would not (hard part 3).
//
// Neighbour list (Fig. 4), ballot variant k_tile_build, w = 32 (the default is k_tile_build8 further
// down: 4 candidate phases x 8 home particles per warp, no ballot): a warp strides over the 9 x-runs of the 27 stencil cells, one
// ballot per 32 candidates (Fig. 4 steps 2-3) for BUILD_P home particles of one cell at a time (a candidate is loaded
// once and tested against BUILD_P particles held in registers).  The distance test is the fp32 dot-product form
// |b|^2 - 2 a.b < R^2 - |a|^2 (three FFMA per candidate, |b|^2 staged with the record) against R^2 = r_list^2 + guard,
// where the guard bounds the fp32 error: the stored list is therefore a SUPERSET of the exact list by at most the
// pairs inside the guard band (relative width ~1e-5), which is a valid Verlet list (it only has to
// contain every pair that can come within r_cut before the next rebuild).  Hits are compacted with popc prefix sums
// of the ballot (steps 4-7) into a row assembled in shared memory and written out with 16-byte stores; rows have a
// fixed stride, so there is no count pass, no scan, no reservation and no atomic anywhere, and every warp works
// independently of the others.  The EXPORTED list (md_get_nlist / md_get_nlist_rows) is filtered with the exact fp64
// expression of DESIGN.md R2 on the positions the list was built from, so it equals the plain definition bit for bit.
//
// Force kernels take the r < rc decision on the staged coordinates only outside a guard band around rc^2; inside
// the band the pair is re-tested with the exact fp64 expression on the global positions (R26).
#include <algorithm>
#include <cstdlib>
#include <type_traits>

#include "md_device.cuh"

constexpr int TILE_MAX_BLOCK = MD_TILE_MAX_BLOCK;  // __launch_bounds__ of the tile kernels (up to 128 registers per thread)
constexpr int BUILD_P = 4;           // home particles per warp task in the build kernel
constexpr uint32_t N_DUMMY = 8;      // far-away dummy records after the staged ones, one per bank class (row padding)
constexpr uint32_t RB_EXTRA = 96;    // build kernel: row assembly buffers hold this many entries more than a stored row

struct TileParams {
    uint32_t B;        // brick edge in cells
    uint32_t nsc_max;  // (B+2)^3
    uint32_t n_tiles;
    uint32_t stride;   // entries per neighbour row (multiple of 16)
    uint32_t shift;    // list entry = staged index << shift (4: byte offset of a float4 record; 0: plain index)
    const uint32_t *tile_cell_begin;  // [n_tiles+1] first cell rank of each tile
    const uint32_t *tile_origin;      // [3 n_tiles] lowest cell coordinate of the brick
    const uint32_t *lin_of_rank;      // cell rank -> linear id
    const uint32_t *rank_of_lin;      // linear id -> cell rank
    const uint32_t *cell_start;       // [n_cells+1] first particle slot of each cell rank
    double cw[3];                     // cell widths
    uint32_t rot_mul, rot_mask;       // bank-class rotation of the row of home particle p: rot_mul * (p & rot_mask)
    const uint32_t *desc;             // per-tile header precomputed at the rebuild (k_tile_header), or nullptr
    uint32_t desc_words;              // words per tile in desc
};

constexpr uint32_t TILE_DESC_CTX = 16;  // words reserved for the TileCtx at the start of a tile's descriptor
__host__ __device__ inline uint32_t tile_desc_table_words(uint32_t B)
{
    const uint32_t nsc = (B + 2) * (B + 2) * (B + 2), nhc = B * B * B;
    return nsc + (nsc + 1) + nhc + (nhc + 1);  // gstart, sstart, hc_sc, hc_first: contiguous in TileSmem
}

struct TileCtx {
    uint32_t x0, y0, z0, ex, ey, ez, sx, sy, sz, n_sc, n_staged, n_home, g0, cb, n_hc;
};

// shared-memory header, carved from the dynamic allocation (sizes depend on the brick)
struct TileSmem {
    uint32_t *gstart;   // [nsc]   global slot of the first particle of each staged cell
    uint32_t *sstart;   // [nsc+1] staged index of the first particle of each staged cell
    uint32_t *hc_sc;    // [B^3]   staged-cell index of each home cell
    uint32_t *hc_first; // [B^3+1] first home particle (tile-local) of each home cell
    uint32_t *hc_task;  // [B^3+1] first build task of each home cell (build kernel only)
    double *cgeo;       // [nsc*6] per staged cell: centre inside the box (3), centre of its image rel. brick centre (3)
    float4 *coff;       // [nsc]   the latter in fp32 (what tile_stage_rel adds to the cell-relative records)
    char *rest;         // records etc.
};

__host__ __device__ inline size_t tile_header_bytes(uint32_t B)
{
    const size_t nsc = (size_t)(B + 2) * (B + 2) * (B + 2), nhc = (size_t)B * B * B;
    size_t b = sizeof(uint32_t) * (nsc + (nsc + 1) + nhc + 2 * (nhc + 1));
    b = (b + 15) & ~(size_t)15;
    b += sizeof(double) * 6 * nsc;
    b = (b + 15) & ~(size_t)15;
    b += sizeof(float4) * nsc;
    return b;
}

__device__ __forceinline__ TileSmem tile_carve(char *smem, uint32_t B)
{
    const uint32_t nsc = (B + 2) * (B + 2) * (B + 2), nhc = B * B * B;
    TileSmem t;
    t.gstart = (uint32_t *)smem;
    t.sstart = t.gstart + nsc;
    t.hc_sc = t.sstart + nsc + 1;
    t.hc_first = t.hc_sc + nhc;
    t.hc_task = t.hc_first + nhc + 1;
    size_t b = sizeof(uint32_t) * (nsc + (nsc + 1) + nhc + 2 * (nhc + 1));
    b = (b + 15) & ~(size_t)15;
    t.cgeo = (double *)(smem + b);
    b += sizeof(double) * 6 * nsc;
    b = (b + 15) & ~(size_t)15;
    t.coff = (float4 *)(smem + b);
    t.rest = smem + tile_header_bytes(B);
    return t;
}

// Offsets of the staged cells for the fp32 records (md_rel_record), per axis: snapped centre of the cell with (wrapped)
// index along that axis, plus its periodic image shift, minus the snapped brick reference -- every term a multiple of the
// grid q0, so the offset is exact in fp32, record + offset is an exact fp32 sum, and the difference of two cells' offsets
// is the same in every tile.  The only thing the grid drops is L - round(L) of an image shift: it goes into the residual
// field of that axis (value + 255).  24 threads fill axo[8 a + i], axf[8 a + i] (a staged block is at most 6 cells wide);
// a staged cell (ix, iy, iz) then takes (axo[ix], axo[8 + iy], axo[16 + iz]) and the three fields.
__device__ __forceinline__ void tile_axis_offsets(const Geom &g, const TileCtx &tc, float *axo, uint32_t *axf)
{
    if (threadIdx.x < 24u) {
        const int a = (int)(threadIdx.x >> 3);
        const uint32_t i = threadIdx.x & 7u;
        const uint32_t o = a == 0 ? tc.x0 : (a == 1 ? tc.y0 : tc.z0), e = a == 0 ? tc.ex : (a == 1 ? tc.ey : tc.ez);
        if (i < e + 2u) {
            const uint32_t n = g.n[a], u1 = o + i;  // unwrapped index + 1
            const uint32_t cwrap = (u1 + n - 1u) % n;
            const int shift = u1 == 0u ? -1 : (u1 > n ? 1 : 0);
            // snapped reference point of the brick (near its centre): staged coordinates are relative to it
            const double rc_ = __dadd_rn(g.lo[a], __dmul_rn(__dadd_rn((double)o, 0.5 * (double)e), g.cw[a]));
            const double ref = __dmul_rn(rint(__dmul_rn(rc_, g.q0i)), g.q0);
            const double Lq = __dmul_rn(rint(__dmul_rn(g.L[a], g.q0i)), g.q0);
            const double off = (md_cell_centre_q(cwrap, a, g) - ref) + (double)shift * Lq;  // multiples of q0: exact
            axo[8 * a + i] = (float)off;
            axf[8 * a + i] = (uint32_t)(max(-255, min(255, md_round_to_int((double)shift * (g.L[a] - Lq) * g.qri))) + 255);
        }
    }
    __syncthreads();
}

// COFF: also the fp32 cell offsets (h.coff) that the kernels staging from the fp32 records add; the fp64 kernels skip them
template <bool COFF = true>
__device__ __forceinline__ void tile_setup(const TileParams &tp, const Geom &g, uint32_t t, const TileSmem &h, TileCtx &tc)
{
    if (tp.desc) {
        // the tables depend on the binning only: k_tile_header wrote them at the rebuild; one coalesced copy and one
        // barrier instead of four dependent global round trips, a scan and three barriers
        const uint32_t *d = tp.desc + (size_t)t * tp.desc_words;
        const uint32_t words = tile_desc_table_words(tp.B);
        for (uint32_t i = threadIdx.x; i < words; i += blockDim.x) h.gstart[i] = __ldg(d + TILE_DESC_CTX + i);
        uint32_t *tcw = (uint32_t *)&tc;
#pragma unroll
        for (int i = 0; i < (int)(sizeof(TileCtx) / 4); ++i) tcw[i] = __ldg(d + i);
        __shared__ float s_axo[24];
        __shared__ uint32_t s_axf[24];
        if (COFF) tile_axis_offsets(g, tc, s_axo, s_axf);
        for (uint32_t sc = threadIdx.x; sc < tc.n_sc; sc += blockDim.x) {
            const uint32_t ix = sc % tc.sx, iy = (sc / tc.sx) % tc.sy, iz = sc / (tc.sx * tc.sy);
            if (COFF) {  // kernels that stage the fp32 records
                h.coff[sc] = make_float4(s_axo[ix], s_axo[8 + iy], s_axo[16 + iz],
                                         __uint_as_float(s_axf[ix] | (s_axf[8 + iy] << 10) | (s_axf[16 + iz] << 20)));
            } else {     // fp64 kernels: centre of the cell inside the box, centre of its image relative to the brick centre
                const uint32_t cx = (tc.x0 + ix + g.n[0] - 1) % g.n[0];
                const uint32_t cy = (tc.y0 + iy + g.n[1] - 1) % g.n[1];
                const uint32_t cz = (tc.z0 + iz + g.n[2] - 1) % g.n[2];
                double *cg = h.cgeo + 6 * sc;
                cg[0] = g.lo[0] + ((double)cx + 0.5) * tp.cw[0];
                cg[1] = g.lo[1] + ((double)cy + 0.5) * tp.cw[1];
                cg[2] = g.lo[2] + ((double)cz + 0.5) * tp.cw[2];
                cg[3] = ((double)ix - 0.5 - 0.5 * (double)tc.ex) * tp.cw[0];
                cg[4] = ((double)iy - 0.5 - 0.5 * (double)tc.ey) * tp.cw[1];
                cg[5] = ((double)iz - 0.5 - 0.5 * (double)tc.ez) * tp.cw[2];
            }
        }
        __syncthreads();
        return;
    }
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
    __shared__ float s_axo2[24];
    __shared__ uint32_t s_axf2[24];
    if (COFF) tile_axis_offsets(g, tc, s_axo2, s_axf2);
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
        if (COFF)
            h.coff[sc] = make_float4(s_axo2[ix], s_axo2[8 + iy], s_axo2[16 + iz],
                                     __uint_as_float(s_axf2[ix] | (s_axf2[8 + iy] << 10) | (s_axf2[16 + iz] << 20)));
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

// global slot of staged index s
__device__ __forceinline__ uint32_t tile_global_of_staged(const TileSmem &h, uint32_t n_sc, uint32_t s)
{
    const uint32_t sc = tile_cell_of_staged(h, n_sc, s);
    return h.gstart[sc] + (s - h.sstart[sc]);
}

// Walks every staged record cell by cell: a group of LPC lanes (8, 16 or 32, from the mean cell population) takes a
// staged cell, two members per lane in flight: load(global slot) for both, then store(staged index, staged cell, value).
// Replaces a per-record cell table (one pass less, no search per record).
template <typename T, typename Load, typename Store>
__device__ __forceinline__ void tile_for_each_staged(const TileCtx &tc, const TileSmem &h, Load load, Store store)
{
    const uint32_t mean = tc.n_staged / max(tc.n_sc, 1u);
    const uint32_t lpc = mean <= 12u ? 8u : (mean <= 26u ? 16u : 32u);  // two members per lane cover a typical cell
    const uint32_t lane = threadIdx.x & 31u, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const uint32_t cpw = 32u / lpc, sub = lane / lpc, m = lane % lpc;
    for (uint32_t sc = wid * cpw + sub; sc < tc.n_sc; sc += nw * cpw) {
        const uint32_t b = h.sstart[sc], n = h.sstart[sc + 1] - b, gs = h.gstart[sc];
        for (uint32_t k = m; k < n; k += 2u * lpc) {
            T v[2];
#pragma unroll
            for (int u = 0; u < 2; ++u)
                if (k + u * lpc < n) v[u] = load(gs + k + u * lpc);
#pragma unroll
            for (int u = 0; u < 2; ++u)
                if (k + u * lpc < n) store(b + k + u * lpc, sc, v[u]);
        }
    }
}

template <typename R4> struct RecTraits;
template <> struct RecTraits<float4> {
    typedef float real;
    // w = |r|^2 of the ROUNDED coordinates (the build kernel's dot-product test)
    static __device__ __forceinline__ float4 make(double x, double y, double z, double w)
    {
        const float fx = (float)x, fy = (float)y, fz = (float)z;
        return make_float4(fx, fy, fz, fx * fx + fy * fy + fz * fz);
    }
    static __device__ __forceinline__ float4 far() { return make_float4(1e15f, 1e15f, 1e15f, 3e30f); }
};
template <> struct RecTraits<double4> {
    typedef double real;
    static __device__ __forceinline__ double4 make(double x, double y, double z, double w) { return make_double4(x, y, z, w); }
    static __device__ __forceinline__ double4 far() { return make_double4(1e150, 1e150, 1e150, 0.0); }
};

// stage every stencil particle: coordinates relative to the brick centre, periodic image applied.
// x_staged = c_s + minimg(x - C_w): C_w = centre of the particle's cell inside the box, c_s = centre of that cell's
// image relative to the brick centre.  |x - C_w| <= w/2 + drift << L/2, so this also undoes an integrator wrap.
// scell: [max_staged] scratch, staged cell of each staged record (filled here; replaces a search per record).
template <typename R4, bool WITH_VEL>
__device__ __forceinline__ void tile_stage(const Geom &g, const TileCtx &tc, const TileSmem &h,
                                           const double4 *__restrict__ pos, const double4 *__restrict__ vel, R4 *rec,
                                           double4 *svel, uint8_t *scell, double scale = 1.0)
{
    const uint32_t lane = threadIdx.x & 31u, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    for (uint32_t sc = wid; sc < tc.n_sc; sc += nw) {
        const uint32_t b = h.sstart[sc], e = h.sstart[sc + 1];
        for (uint32_t s = b + lane; s < e; s += 32) scell[s] = (uint8_t)sc;
    }
    __syncthreads();
    for (uint32_t s = threadIdx.x; s < tc.n_staged; s += blockDim.x) {
        const uint32_t sc = scell[s];
        const uint32_t gi = h.gstart[sc] + (s - h.sstart[sc]);
        const double4 p = pos[gi];
        const double *cg = h.cgeo + 6 * sc;
        const double x = cg[3] + md_min_image(p.x - cg[0], g.L[0], g.h[0]);
        const double y = cg[4] + md_min_image(p.y - cg[1], g.L[1], g.h[1]);
        const double z = cg[5] + md_min_image(p.z - cg[2], g.L[2], g.h[2]);
        rec[s] = RecTraits<R4>::make(x * scale, y * scale, z * scale, p.w);
        if (WITH_VEL) svel[s] = vel[gi];
    }
    if (threadIdx.x < N_DUMMY) rec[tc.n_staged + threadIdx.x] = RecTraits<R4>::far();  // dummy records: row padding
}

// fp32 records from the cell-relative fp32 positions `rel` (kept current by the binning and by half 1, see
// md_rel_record): staged coordinate = fl(fl(x - C_w) + fl(c_s)), times `scale`.  No fp64, 16 bytes per particle.
template <bool WITH_R2>
__device__ __forceinline__ void tile_stage_rel(const TileCtx &tc, const TileSmem &h, const float4 *__restrict__ rel,
                                               float4 *rec, uint8_t *scell, float scale,
                                               const double4 *__restrict__ pos, const Geom &g)
{
    const uint32_t lane = threadIdx.x & 31u, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    if (!MD_STAGE_FROM_REL) {
        for (uint32_t sc = wid; sc < tc.n_sc; sc += nw) {
            const uint32_t b = h.sstart[sc], e = h.sstart[sc + 1];
            for (uint32_t s = b + lane; s < e; s += 32) scell[s] = (uint8_t)sc;
        }
        __syncthreads();
        // fp64 staging: the coordinate relative to the brick centre is formed in fp64 and rounded ONCE (R25)
        const double dscale = (double)scale;
        for (uint32_t s0 = threadIdx.x; s0 < tc.n_staged; s0 += 2 * blockDim.x) {
            double4 pp[2];
            uint32_t scs[2];
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const uint32_t s = s0 + u * blockDim.x;
                if (s < tc.n_staged) {
                    scs[u] = scell[s];
                    pp[u] = pos[h.gstart[scs[u]] + (s - h.sstart[scs[u]])];
                }
            }
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const uint32_t s = s0 + u * blockDim.x;
                if (s < tc.n_staged) {
                    const double *cg = h.cgeo + 6 * scs[u];
                    const float x = (float)((cg[3] + md_min_image(pp[u].x - cg[0], g.L[0], g.h[0])) * dscale);
                    const float y = (float)((cg[4] + md_min_image(pp[u].y - cg[1], g.L[1], g.h[1])) * dscale);
                    const float z = (float)((cg[5] + md_min_image(pp[u].z - cg[2], g.L[2], g.h[2])) * dscale);
                    rec[s] = make_float4(x, y, z, WITH_R2 ? x * x + y * y + z * z : 0.f);
                }
            }
        }
        if (threadIdx.x < N_DUMMY) rec[tc.n_staged + threadIdx.x] = RecTraits<float4>::far();
        return;
    }
    // a warp takes two staged cells at a time; the (up to) four loads of a lane -- members 0..31 and 32..63 of each --
    // are issued before the first is used (the loop is a chain of L2 round trips otherwise); longer cells loop on.
    // (No per-record cell table: `scell` is not filled on this path.)
    for (uint32_t sc0 = 2u * wid; sc0 < tc.n_sc; sc0 += 2u * nw) {
        float4 r[4];
        uint32_t sb[2], sn[2], gs[2];
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const uint32_t sc = min(sc0 + u, tc.n_sc - 1u);
            sb[u] = h.sstart[sc];
            sn[u] = sc0 + u < tc.n_sc ? h.sstart[sc + 1] - sb[u] : 0u;
            gs[u] = h.gstart[sc];
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const uint32_t k = lane + 32u * (u >> 1);
            if (k < sn[u & 1]) r[u] = __ldg(rel + gs[u & 1] + k);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const uint32_t k = lane + 32u * (u >> 1);
            if (k < sn[u & 1]) {
                const float4 o = h.coff[min(sc0 + (u & 1), tc.n_sc - 1u)];
                const float x = (r[u].x + o.x) * scale, y = (r[u].y + o.y) * scale, z = (r[u].z + o.z) * scale;
                rec[sb[u & 1] + k] = make_float4(x, y, z, WITH_R2 ? x * x + y * y + z * z : 0.f);
            }
        }
#pragma unroll 1
        for (int u = 0; u < 2; ++u) {  // cells of more than 64 members
            const float4 o = h.coff[min(sc0 + u, tc.n_sc - 1u)];
            for (uint32_t k = 64u + lane; k < sn[u]; k += 32) {
                const float4 q = __ldg(rel + gs[u] + k);
                const float x = (q.x + o.x) * scale, y = (q.y + o.y) * scale, z = (q.z + o.z) * scale;
                rec[sb[u] + k] = make_float4(x, y, z, WITH_R2 ? x * x + y * y + z * z : 0.f);
            }
        }
    }
    if (threadIdx.x < N_DUMMY) rec[tc.n_staged + threadIdx.x] = RecTraits<float4>::far();
}

// k_tile_lj3's staging.  The cell-relative records lie on the grid q0 (md_rel_record) and so do the cell offsets
// (tile_grid_offset: the offset of every staged cell rounded to the grid; what that drops joins the residuals), hence
//     staged coordinate = record + offset     is an EXACT fp32 sum (every staged coordinate is below 2^24 q0),
//     staged residual   = record residual + offset residual   (one integer add on the packed 10-bit fields),
// and coordinate + qr * residual is the true brick-relative coordinate to ~ qr = q0 / 510 (~1e-9 at config 2).  The far
// loop reads x, y, z; the near section rebuilds separations from both in fp64 without leaving shared memory (R25).
// 16 bytes per staged particle from L2, a handful of instructions per record, no fp64 and no conversion.
__device__ __forceinline__ void tile_stage_exact(const TileCtx &tc, const TileSmem &h, const float4 *__restrict__ rel,
                                                 float4 *rec)
{
    // a warp takes two staged cells at a time; the (up to) four loads of a lane -- members 0..31 and 32..63 of each --
    // are issued before the first is used (the loop is a chain of L2 round trips otherwise); longer cells loop on
    const uint32_t lane = threadIdx.x & 31u, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    for (uint32_t sc0 = 2u * wid; sc0 < tc.n_sc; sc0 += 2u * nw) {
        float4 r[4];
        uint32_t sb[2], sn[2], gs[2];
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const uint32_t sc = min(sc0 + u, tc.n_sc - 1u);
            sb[u] = h.sstart[sc];
            sn[u] = sc0 + u < tc.n_sc ? h.sstart[sc + 1] - sb[u] : 0u;
            gs[u] = h.gstart[sc];
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const uint32_t k = lane + 32u * (u >> 1);
            if (k < sn[u & 1]) r[u] = __ldg(rel + gs[u & 1] + k);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const uint32_t k = lane + 32u * (u >> 1);
            if (k < sn[u & 1]) {
                const float4 o = h.coff[min(sc0 + (u & 1), tc.n_sc - 1u)];
                rec[sb[u & 1] + k] = make_float4(r[u].x + o.x, r[u].y + o.y, r[u].z + o.z,
                                                 __uint_as_float(__float_as_uint(r[u].w) + __float_as_uint(o.w)));
            }
        }
#pragma unroll 1
        for (int u = 0; u < 2; ++u) {  // cells of more than 64 members
            const float4 o = h.coff[min(sc0 + u, tc.n_sc - 1u)];
            for (uint32_t k = 64u + lane; k < sn[u]; k += 32) {
                const float4 q = __ldg(rel + gs[u] + k);
                rec[sb[u] + k] = make_float4(q.x + o.x, q.y + o.y, q.z + o.z,
                                             __uint_as_float(__float_as_uint(q.w) + __float_as_uint(o.w)));
            }
        }
    }
    if (threadIdx.x < N_DUMMY) rec[tc.n_staged + threadIdx.x] = RecTraits<float4>::far();
}

// the plain definition on global (wrapped) positions: exact fp64, no FMA (R2, R8)
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
// once per rebuild, one CTA per tile: the tile's header tables (tile_setup's slow path) go to global memory, and the
// sizes of the largest tile (shared-memory sizing) to the flags
// ===============================================================================================================
__global__ void k_tile_header(TileParams tp, Geom g, uint32_t *desc, unsigned int *max_home, unsigned int *max_staged)
{
    extern __shared__ __align__(16) char smem_raw[];
    const TileSmem h = tile_carve(smem_raw, tp.B);
    TileCtx tc;
    tile_setup<false>(tp, g, blockIdx.x, h, tc);  // tp.desc == nullptr here
    uint32_t *d = desc + (size_t)blockIdx.x * tp.desc_words;
    const uint32_t words = tile_desc_table_words(tp.B);
    for (uint32_t i = threadIdx.x; i < words; i += blockDim.x) d[TILE_DESC_CTX + i] = h.gstart[i];
    if (threadIdx.x == 0) {
        const uint32_t *tcw = (const uint32_t *)&tc;
        for (int i = 0; i < (int)(sizeof(TileCtx) / 4); ++i) d[i] = tcw[i];
        atomicMax(max_home, tc.n_home);
        atomicMax(max_staged, tc.n_staged);
    }
}

// ===============================================================================================================
// S2 neighbour-list build, one CTA per tile, one warp per task of P home particles of one cell
// ===============================================================================================================
__device__ __forceinline__ unsigned md_lanemask_lt()
{
    unsigned m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

template <int P>
__global__ void __launch_bounds__(TILE_MAX_BLOCK) k_tile_build(TileParams tp, Geom g, const float4 *__restrict__ rel, const double4 *__restrict__ pos,
                                                               float thr_out /* r_list^2 + guard */,
                                                               uint32_t max_staged, uint32_t *__restrict__ nl_cnt,
                                                               uint16_t *__restrict__ nl16, DevFlags *flags)
{
    extern __shared__ __align__(16) char smem_raw[];
    const TileSmem h = tile_carve(smem_raw, tp.B);
    float4 *rec = (float4 *)h.rest;
    const uint32_t nw = blockDim.x >> 5;
    uint16_t *rowbuf = (uint16_t *)(h.rest + sizeof(float4) * (max_staged + N_DUMMY));  // [nw][P][stride + RB_EXTRA]
    uint32_t *scratch = (uint32_t *)(rowbuf + (size_t)nw * P * (tp.stride + RB_EXTRA));  // [nw][P][24]
    uint8_t *scell = (uint8_t *)(scratch + nw * P * 24);                                 // [max_staged]

    TileCtx tc;
    tile_setup(tp, g, blockIdx.x, h, tc);
    tile_stage_rel<true>(tc, h, rel, rec, scell, 1.f, pos, g);
    if (threadIdx.x < 32) {  // first task of each home cell: exclusive scan of ceil(count / P), n_hc <= 64
        uint32_t carry = 0;
        for (uint32_t base = 0; base <= tc.n_hc; base += 32) {
            const uint32_t hc = base + threadIdx.x;
            const uint32_t v = hc < tc.n_hc ? (h.hc_first[hc + 1] - h.hc_first[hc] + P - 1) / P : 0u;
            uint32_t inc = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t u = __shfl_up_sync(0xffffffffu, inc, o);
                if ((int)threadIdx.x >= o) inc += u;
            }
            if (hc <= tc.n_hc) h.hc_task[hc] = carry + inc - v;
            carry += __shfl_sync(0xffffffffu, inc, 31);
        }
    }
    __syncthreads();

    const unsigned lane = threadIdx.x & 31u, wid = threadIdx.x >> 5;
    const unsigned lt = md_lanemask_lt();
    const uint32_t n_tasks = h.hc_task[tc.n_hc];
    const uint32_t stride = tp.stride, rcap = tp.stride + RB_EXTRA;
    // bank classes (see the layout note above k_tile_lj3): candidates are visited in groups of 32 aligned to 8 staged
    // indices, so the class (staged index & 7) of a lane's candidate is the constant lane & 7
    const uint32_t cls = lane & 7u;
    const unsigned cmask_lt = (0x01010101u << cls) & lt, cmask = 0x01010101u << cls;
    uint16_t *rb = rowbuf + (size_t)wid * P * rcap;
    uint32_t *scr = scratch + wid * P * 24;  // per warp and row: n_c[8], first hole H_c[8], first overflow entry O_c[8]
    unsigned long long total = 0;
    uint32_t worst = 0;

    for (uint32_t task = wid; task < n_tasks; task += nw) {
        // home cell of the task (binary search over hc_task), first particle, particles in this task
        uint32_t hc = 0;
        {
            uint32_t lo = 0, hi = tc.n_hc;
            while (hi - lo > 1) {
                const uint32_t mid = (lo + hi) >> 1;
                if (h.hc_task[mid] <= task) lo = mid; else hi = mid;
            }
            hc = lo;
        }
        const uint32_t p0 = h.hc_first[hc] + (task - h.hc_task[hc]) * P;
        const uint32_t np = min((uint32_t)P, h.hc_first[hc + 1] - p0);
        const uint32_t sch = h.hc_sc[hc];
        const uint32_t ixh = sch % tc.sx, iyh = (sch / tc.sx) % tc.sy, izh = sch / (tc.sx * tc.sy);
        const uint32_t self0 = h.sstart[sch] + (p0 - h.hc_first[hc]);
        // hit <=> |b|^2 - 2 a.b < thr - |a|^2
        float ax[P], ay[P], az[P], th[P];
        uint32_t cntc[P];  // entries of this lane's class found so far, per home particle
#pragma unroll
        for (int q = 0; q < P; ++q) {
            const float4 m = rec[self0 + min((uint32_t)q, np - 1)];
            ax[q] = -2.f * m.x; ay[q] = -2.f * m.y; az[q] = -2.f * m.z;
            th[q] = (uint32_t)q < np ? thr_out - m.w : -3e38f;  // absent particles never hit
            cntc[q] = 0;
        }
#pragma unroll 1
        for (int run = 0; run < 9; ++run) {
            const uint32_t iy = iyh + (run % 3) - 1, iz = izh + (run / 3) - 1;
            const uint32_t sc0 = (ixh - 1) + tc.sx * (iy + tc.sy * iz);
            const uint32_t b = h.sstart[sc0], e = h.sstart[sc0 + 3];
#pragma unroll 1
            for (uint32_t base = b & ~7u; base < e; base += 32) {
                const uint32_t j = base + lane;
                const float4 pj = rec[(j >= b && j < e) ? j : tc.n_staged];  // outside the run: a far-away dummy record
                unsigned bal[P];
#pragma unroll
                for (int q = 0; q < P; ++q) {
                    float t = fmaf(ax[q], pj.x, pj.w);
                    t = fmaf(ay[q], pj.y, t);
                    t = fmaf(az[q], pj.z, t);
                    bal[q] = __ballot_sync(0xffffffffu, t < th[q]);
                }
                if (self0 + (P - 1) - base < 32u + (P - 1)) {  // this group of 32 holds some of the task's own particles
#pragma unroll
                    for (int q = 0; q < P; ++q) {
                        const uint32_t d = self0 + q - base;
                        if (d < 32u) bal[q] &= ~(1u << d);
                    }
                }
                const uint16_t ent = (uint16_t)(j << tp.shift);
#pragma unroll
                for (int q = 0; q < P; ++q) {
                    if (bal[q]) {
                        // k-th entry of class c goes to block k, slot (c - k - rot) & 7 (Fig. 4 steps 4-7 per class)
                        const uint32_t k = cntc[q] + __popc(bal[q] & cmask_lt);
                        const uint32_t o = 8u * k + ((cls - k - tp.rot_mul * ((p0 + q) & tp.rot_mask)) & 7u);
                        if (((bal[q] >> lane) & 1u) && o < rcap) rb[q * rcap + o] = ent;
                        cntc[q] += __popc(bal[q] & cmask);
                    }
                }
            }
        }
        __syncwarp();
        // finish the P = 4 rows together: lane = 8 * row + class
        {
            static_assert(P == 4, "row finishing maps 8 lanes (bank classes) to each of 4 rows");
            const uint32_t qr = lane >> 3;
            const bool live = qr < np;
            uint32_t nc = cntc[0];
            nc = qr == 1 ? cntc[1] : nc;
            nc = qr == 2 ? cntc[2] : nc;
            nc = qr == 3 ? cntc[3] : nc;
            if (!live) nc = 0;
            const uint32_t rot = tp.rot_mul * ((p0 + qr) & tp.rot_mask);
            uint32_t n = nc, mx = nc;
#pragma unroll
            for (int o = 1; o < 8; o <<= 1) {
                n += __shfl_xor_sync(0xffffffffu, n, o);
                mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
            }
            // row length in blocks of 8; a class longer than the assembly buffer lost entries -> overflow
            uint32_t need = (n + 7u) & ~7u;
            if (8u * mx > rcap) need = max(need, 8u * mx - RB_EXTRA);
            worst = max(worst, need);
            const uint32_t nblk = min((n + 7u) >> 3, stride >> 3);
            uint16_t *r = rb + qr * rcap;
            // holes (class shorter than the row) take the entries of longer classes, then dummies of their class
            const uint32_t nck = min(nc, rcap >> 3);
            const uint32_t holes = nblk > nck ? nblk - nck : 0u, over = nck > nblk ? nck - nblk : 0u;
            uint32_t hs = holes, os = over;
#pragma unroll
            for (int o = 1; o < 8; o <<= 1) {
                const uint32_t a = __shfl_up_sync(0xffffffffu, hs, o, 8), bb = __shfl_up_sync(0xffffffffu, os, o, 8);
                if ((int)cls >= o) { hs += a; os += bb; }
            }
            const uint32_t n_holes = __shfl_sync(0xffffffffu, hs, 7, 8), n_over = __shfl_sync(0xffffffffu, os, 7, 8);
            uint32_t *sc = scr + 24 * qr;
            sc[cls] = nck;
            sc[8 + cls] = hs - holes;
            sc[16 + cls] = os - over;
            __syncwarp();
            for (uint32_t o = cls; o < n_holes; o += 8) {
                uint32_t c = 0;
#pragma unroll
                for (int k = 1; k < 8; ++k) c += o >= sc[8 + k] ? 1u : 0u;
                // classes without holes share their successor's start: the count above lands on the last class whose
                // first hole is <= o, which is the one that owns hole o
                const uint32_t bk = sc[c] + (o - sc[8 + c]);
                uint16_t v;
                if (o < n_over) {
                    uint32_t cs = 0;
#pragma unroll
                    for (int k = 1; k < 8; ++k) cs += o >= sc[16 + k] ? 1u : 0u;
                    const uint32_t k2 = nblk + (o - sc[16 + cs]);
                    v = r[8u * k2 + ((cs - k2 - rot) & 7u)];
                } else {
                    v = (uint16_t)((tc.n_staged + ((c - tc.n_staged) & 7u)) << tp.shift);
                }
                r[8u * bk + ((c - bk - rot) & 7u)] = v;
            }
            __syncwarp();
#pragma unroll
            for (int q = 0; q < P; ++q) {
                const uint32_t nb = __shfl_sync(0xffffffffu, nblk, 8 * q);
                uint4 *dst = (uint4 *)(nl16 + (size_t)(tc.g0 + p0 + q) * stride);
                const uint4 *src = (const uint4 *)(rb + q * rcap);
                for (uint32_t v = lane; v < nb; v += 32) dst[v] = src[v];
            }
            if (live && cls == 0) {
                nl_cnt[tc.g0 + p0 + qr] = min(n, 8u * nblk);
                total += n;
            }
        }
        __syncwarp();
    }
    total += __shfl_xor_sync(0xffffffffu, total, 8);
    total += __shfl_xor_sync(0xffffffffu, total, 16);
    if (lane == 0 && total) atomicAdd(&flags->nl_total, total);
    if (worst > stride) atomicMax(&flags->nl_overflow, worst);
}

// ===============================================================================================================
// S2, the default build: k_tile_build8.  A warp task is 8 consecutive home particles of one cell; lane = 8 phase + h
// holds home particle h and visits the candidates j = base + phase, base + 4 + phase, ... (base a multiple of 8), so
// the 8 lanes of a quarter-warp read ONE staged record (a broadcast: one wavefront per quarter) and test it against
// their 8 home particles.  The bank class of a candidate is j & 7 = phase or phase + 4: each (home particle, class) is
// owned by exactly one lane, which keeps the running count of that class in a register and writes a hit straight to
// its slot (block k, slot (class - k - rot) & 7) of the row assembled in shared memory -- Fig. 4's compaction
// with the prefix sum replaced by per-lane counters: no ballot, no popc, no atomics, no
// communication between lanes until the row is finished (holes, copy-out: as in k_tile_build, 4 rows at a time).
// ===============================================================================================================
// Near section of a row assembled in shared memory (k_tile_build8, MD_MIXED; R25): every neighbour closer than
// r_near + r_buff now -- i.e. every pair that can come within r_near before the next rebuild -- is moved into the LAST
// K = ceil(n_near / 8) blocks of the row, which the mixed-precision force kernel evaluates in fp64.  Called by the 8 lanes
// of a row together (lane = class): the lane owns the column of its class, slot (cls - b - rot) & 7 of every block b.  A
// near entry above the section first changes places with a far entry (or dummy) of the SAME column inside the section,
// so the bank-class layout of the far blocks survives; what is left over (columns with more than K near entries) goes
// to the free section slots of other columns (the near section is read entry by entry: its layout is free).
// M: one bit per block (uint32_t for rows of up to 32 blocks, else 64; longer rows get no near section).  Returns K.
template <typename M>
__device__ __forceinline__ uint32_t near_partition(uint16_t *r, const float4 *rec, const float4 mh, float thr_near,
                                                   uint32_t nblk, uint32_t cls, uint32_t rrot, uint32_t sh, uint16_t *hp)
{
    constexpr uint32_t BITS = 8u * (uint32_t)sizeof(M);
    const M one = (M)1;
    const float nax = -2.f * mh.x, nay = -2.f * mh.y, naz = -2.f * mh.z, nth = thr_near - mh.w;
    const uint32_t nb = nblk <= BITS ? nblk : 0u;
    M nearbits = 0;
#pragma unroll 2
    for (uint32_t b = 0; b < nb; ++b) {
        const uint32_t s = (uint32_t)r[8u * b + ((cls - b - rrot) & 7u)] >> sh;
        const float4 pc = rec[s];
        const float t = fmaf(naz, pc.z, fmaf(nay, pc.y, fmaf(nax, pc.x, pc.w)));
        nearbits |= (M)(t < nth ? 1u : 0u) << b;
    }
    uint32_t n_near = sizeof(M) == 8 ? (uint32_t)__popcll((unsigned long long)nearbits) : (uint32_t)__popc((uint32_t)nearbits);
#pragma unroll
    for (int o = 1; o < 8; o <<= 1) n_near += __shfl_xor_sync(0xffffffffu, n_near, o);
    const uint32_t K = min((n_near + 7u) >> 3, nb);
    const uint32_t b0 = nb - K;  // first block of the near section
    const M all = nb >= BITS ? ~(M)0 : (one << nb) - one;
    const M sect = all & ~(b0 >= BITS ? ~(M)0 : (one << b0) - one);
    M hole = ~nearbits & sect;        // section slots of my column that hold no near entry
    M over = nearbits & ~sect & all;  // near entries of my column outside the section
    auto low = [](M m) -> uint32_t {
        return sizeof(M) == 8 ? (uint32_t)__ffsll((long long)m) - 1u : (uint32_t)__ffs((int)m) - 1u;
    };
    auto cnt = [](M m) -> uint32_t {
        return sizeof(M) == 8 ? (uint32_t)__popcll((unsigned long long)m) : (uint32_t)__popc((uint32_t)m);
    };
    while (hole && over) {
        const uint32_t i = low(hole), j = low(over);
        uint16_t *pa = r + 8u * i + ((cls - i - rrot) & 7u), *pb = r + 8u * j + ((cls - j - rrot) & 7u);
        const uint16_t t = *pa; *pa = *pb; *pb = t;
        hole &= hole - one;
        over &= over - one;
    }
    // left-overs across the 8 columns of the row: the o-th stranded near entry takes the o-th free section slot
    const uint32_t nh = cnt(hole), no = cnt(over);
    uint32_t hsum = nh, osum = no;
#pragma unroll
    for (int o = 1; o < 8; o <<= 1) {
        const uint32_t a = __shfl_up_sync(0xffffffffu, hsum, o, 8), bb = __shfl_up_sync(0xffffffffu, osum, o, 8);
        if ((int)cls >= o) { hsum += a; osum += bb; }
    }
    const uint32_t n_over = __shfl_sync(0xffffffffu, osum, 7, 8);
    if (__any_sync(0xffffffffu, n_over != 0u)) {
        __syncwarp();
        {
            uint32_t o = hsum - nh;
            for (M m = hole; m && o < 48u && o < n_over; m &= m - one, ++o) {
                const uint32_t i = low(m);
                hp[o] = (uint16_t)(8u * i + ((cls - i - rrot) & 7u));
            }
        }
        __syncwarp();
        {
            uint32_t o = osum - no;
            for (M m = over; m && o < 48u; m &= m - one, ++o) {
                const uint32_t j = low(m);
                uint16_t *pa = r + hp[o], *pb = r + 8u * j + ((cls - j - rrot) & 7u);
                const uint16_t t = *pa; *pa = *pb; *pb = t;
            }
        }
    }
    __syncwarp();
    return K;
}

constexpr int BUILD8_P = 8;

// one x-run of 3 stencil cells [b, e) for one lane: candidates b' + ph, b' + ph + 4, ... (b' = b rounded down to 8).
// Branch-free: the slot is computed for every candidate, the store and the count are predicated on the hit.
// SELF: the run holds the lane's own particle (staged index b + selfd), which is not its own neighbour.
template <bool SELF>
__device__ __forceinline__ void b8_run(const float4 *rec, uint32_t b, uint32_t e, uint32_t ph, float ax, float ay, float az,
                                       float th, uint32_t selfd, uint32_t c0, uint32_t c1, uint32_t rcap, uint16_t *myrow,
                                       uint32_t sh, uint32_t &k0, uint32_t &k1)
{
    const uint32_t len = e - b;
    const uint32_t base0 = b & ~7u;
    uint32_t d0 = base0 + ph - b;  // candidate index relative to b; "negative" wraps to a huge value and fails d0 < len
    // 4 candidates per trip and no remainder loop: candidates past the run fail d < len; what is read there are other
    // cells' records, the dummies or (at the very end of the staged array) the row buffers -- never used
    const float4 *pr = rec + base0 + ph;
    uint32_t ent = (base0 + ph) << sh;
    const uint32_t dent = 16u << sh, e4 = 4u << sh;
#pragma unroll 2
    for (uint32_t base = base0; base < e; base += 16, d0 += 16, pr += 16, ent += dent) {
        float t[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const float4 pc = pr[4 * u];
            t[u] = fmaf(az, pc.z, fmaf(ay, pc.y, fmaf(ax, pc.x, pc.w)));
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            bool hit = t[u] < th && d0 + 4u * u < len;
            if (SELF) hit = hit && d0 + 4u * u != selfd;
            if (u & 1) {
                const uint32_t o = 8u * k1 + ((c1 - k1) & 7u);
                if (hit && o < rcap) myrow[o] = (uint16_t)(ent + u * e4);
                k1 += hit ? 1u : 0u;
            } else {
                const uint32_t o = 8u * k0 + ((c0 - k0) & 7u);
                if (hit && o < rcap) myrow[o] = (uint16_t)(ent + u * e4);
                k0 += hit ? 1u : 0u;
            }
        }
    }
}

__global__ void __launch_bounds__(TILE_MAX_BLOCK) k_tile_build8(TileParams tp, Geom g, const float4 *__restrict__ rel, const double4 *__restrict__ pos,
                                                                float thr_out /* r_list^2 + guard */,
                                                                float thr_near /* (r_near + r_buff)^2 + guard, or 0: no near section */,
                                                                uint32_t max_staged, uint32_t *__restrict__ nl_cnt,
                                                                uint16_t *__restrict__ nl16, DevFlags *flags)
{
    constexpr int P = BUILD8_P;
    extern __shared__ __align__(16) char smem_raw[];
    const TileSmem h = tile_carve(smem_raw, tp.B);
    float4 *rec = (float4 *)h.rest;
    const uint32_t nw = blockDim.x >> 5;
    // rows of a task are 16 bytes further apart than their capacity: lanes that write the same slot of their 8 rows
    // (the usual case, the counts run in step) then fall into different banks
    const uint32_t stride = tp.stride, rcap = tp.stride + RB_EXTRA, rpitch = rcap + 8;
    uint16_t *rowbuf = (uint16_t *)(h.rest + sizeof(float4) * (max_staged + N_DUMMY));  // [nw][P][rpitch]
    uint32_t *scratch = (uint32_t *)(rowbuf + (size_t)nw * P * rpitch);                 // [nw][4][24]
    uint8_t *scell = (uint8_t *)(scratch + nw * 4 * 24);                                // [max_staged]

    TileCtx tc;
    tile_setup(tp, g, blockIdx.x, h, tc);
    tile_stage_rel<true>(tc, h, rel, rec, scell, 1.f, pos, g);
    if (threadIdx.x < 32) {  // first task of each home cell: exclusive scan of ceil(count / P), n_hc <= 64
        uint32_t carry = 0;
        for (uint32_t base = 0; base <= tc.n_hc; base += 32) {
            const uint32_t hc = base + threadIdx.x;
            const uint32_t v = hc < tc.n_hc ? (h.hc_first[hc + 1] - h.hc_first[hc] + P - 1) / P : 0u;
            uint32_t inc = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t u = __shfl_up_sync(0xffffffffu, inc, o);
                if ((int)threadIdx.x >= o) inc += u;
            }
            if (hc <= tc.n_hc) h.hc_task[hc] = carry + inc - v;
            carry += __shfl_sync(0xffffffffu, inc, 31);
        }
    }
    __syncthreads();

    const unsigned lane = threadIdx.x & 31u, wid = threadIdx.x >> 5;
    const uint32_t hh = lane & 7u, ph = lane >> 3;  // home particle of the task, candidate phase
    const uint32_t n_tasks = h.hc_task[tc.n_hc];
    uint16_t *rb = rowbuf + (size_t)wid * P * rpitch;
    uint16_t *myrow = rb + hh * rpitch;
    uint32_t *scr = scratch + wid * 4 * 24;
    const uint32_t sh = tp.shift;
    unsigned long long total = 0;
    uint32_t worst = 0;

    for (uint32_t task = wid; task < n_tasks; task += nw) {
        uint32_t hc = 0;
        {
            uint32_t lo = 0, hi = tc.n_hc;
            while (hi - lo > 1) {
                const uint32_t mid = (lo + hi) >> 1;
                if (h.hc_task[mid] <= task) lo = mid; else hi = mid;
            }
            hc = lo;
        }
        const uint32_t p0 = h.hc_first[hc] + (task - h.hc_task[hc]) * P;
        const uint32_t np = min((uint32_t)P, h.hc_first[hc + 1] - p0);
        const uint32_t sch = h.hc_sc[hc];
        const uint32_t ixh = sch % tc.sx, iyh = (sch / tc.sx) % tc.sy, izh = sch / (tc.sx * tc.sy);
        const uint32_t self0 = h.sstart[sch] + (p0 - h.hc_first[hc]);
        // hit <=> |b|^2 - 2 a.b < thr - |a|^2
        const float4 m = rec[self0 + min(hh, np - 1)];
        const float ax = -2.f * m.x, ay = -2.f * m.y, az = -2.f * m.z;
        const float th = hh < np ? thr_out - m.w : -3e38f;  // absent particles never hit
        const uint32_t self = self0 + hh;
        const uint32_t rot = tp.rot_mul * ((p0 + hh) & tp.rot_mask);
        // slot of the k-th entry of class c: 8 k + ((c - k - rot) & 7); c = ph (k0) or ph + 4 (k1)
        uint32_t k0 = 0, k1 = 0;
        const uint32_t c0 = ph - rot, c1 = ph + 4u - rot;
#pragma unroll 1
        for (int run = 0; run < 9; ++run) {
            const uint32_t iy = iyh + (run % 3) - 1, iz = izh + (run / 3) - 1;
            const uint32_t sc0 = (ixh - 1) + tc.sx * (iy + tc.sy * iz);
            const uint32_t b = h.sstart[sc0], e = h.sstart[sc0 + 3];
            if (run == 4) b8_run<true>(rec, b, e, ph, ax, ay, az, th, self - b, c0, c1, rcap, myrow, sh, k0, k1);
            else b8_run<false>(rec, b, e, ph, ax, ay, az, th, 0u, c0, c1, rcap, myrow, sh, k0, k1);
        }
        __syncwarp();
        // finish 4 rows at a time: lane = 8 * row + class; the count of (row, class) lives in lane 8 (class & 3) + row
#pragma unroll 1
        for (uint32_t r0 = 0; r0 < np; r0 += 4) {
            const uint32_t cls = lane & 7u, qr = r0 + (lane >> 3);
            const uint32_t owner = 8u * (cls & 3u) + (qr & 7u);
            const uint32_t ka = __shfl_sync(0xffffffffu, k0, owner), kb = __shfl_sync(0xffffffffu, k1, owner);
            const bool live = qr < np;
            const uint32_t nc = live ? (cls < 4u ? ka : kb) : 0u;
            const uint32_t rrot = tp.rot_mul * ((p0 + qr) & tp.rot_mask);
            uint32_t n = nc, mx = nc;
#pragma unroll
            for (int o = 1; o < 8; o <<= 1) {
                n += __shfl_xor_sync(0xffffffffu, n, o);
                mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
            }
            // row length in blocks of 8; a class longer than the assembly buffer lost entries -> overflow
            uint32_t need = (n + 7u) & ~7u;
            if (8u * mx > rcap) need = max(need, 8u * mx - RB_EXTRA);
            worst = max(worst, need);
            const uint32_t nblk = min((n + 7u) >> 3, stride >> 3);
            uint16_t *r = rb + (qr & 7u) * rpitch;
            // holes (class shorter than the row) take the entries of longer classes, then dummies of their class
            const uint32_t nck = min(nc, rcap >> 3);
            const uint32_t holes = nblk > nck ? nblk - nck : 0u, over = nck > nblk ? nck - nblk : 0u;
            uint32_t hs = holes, os = over;
#pragma unroll
            for (int o = 1; o < 8; o <<= 1) {
                const uint32_t a = __shfl_up_sync(0xffffffffu, hs, o, 8), bb = __shfl_up_sync(0xffffffffu, os, o, 8);
                if ((int)cls >= o) { hs += a; os += bb; }
            }
            const uint32_t n_holes = __shfl_sync(0xffffffffu, hs, 7, 8), n_over = __shfl_sync(0xffffffffu, os, 7, 8);
            uint32_t *sc = scr + 24 * (lane >> 3);
            sc[cls] = nck;
            sc[8 + cls] = hs - holes;
            sc[16 + cls] = os - over;
            __syncwarp();
            for (uint32_t o = cls; o < n_holes; o += 8) {
                uint32_t c = 0;
#pragma unroll
                for (int k = 1; k < 8; ++k) c += o >= sc[8 + k] ? 1u : 0u;
                const uint32_t bk = sc[c] + (o - sc[8 + c]);
                uint16_t v;
                if (o < n_over) {
                    uint32_t cs = 0;
#pragma unroll
                    for (int k = 1; k < 8; ++k) cs += o >= sc[16 + k] ? 1u : 0u;
                    const uint32_t k2 = nblk + (o - sc[16 + cs]);
                    v = r[8u * k2 + ((cs - k2 - rrot) & 7u)];
                } else {
                    v = (uint16_t)((tc.n_staged + ((c - tc.n_staged) & 7u)) << sh);
                }
                r[8u * bk + ((c - bk - rrot) & 7u)] = v;
            }
            __syncwarp();
            // ---- near section (MD_MIXED, R25): every neighbour closer than r_near + r_buff now -- i.e. every
            // pair that can come within r_near before the next rebuild -- is moved into the LAST K = ceil(n_near / 8)
            // blocks of the row, which the mixed-precision force kernel evaluates in fp64 on the global positions.  The
            // lane owns the column of its class: slot (cls - b - rot) & 7 of every block b.  A near entry above the
            // section first changes places with a far entry (or dummy) of the SAME column inside the section, so the
            // bank-class layout of the far blocks survives; what is left over (columns with more than K near entries)
            // goes to the free slots of other columns (the near section is read entry by entry, its layout is free).
            uint32_t K = 0;
            if (thr_near > 0.f) {
                const float4 mh = rec[self0 + min(qr, np - 1)];
                uint16_t *hp = (uint16_t *)(scr + 24 * (lane >> 3));  // 48 slot positions per row in flight
                K = stride <= 256u ? near_partition<uint32_t>(r, rec, mh, thr_near, nblk, cls, rrot, sh, hp)
                                   : near_partition<unsigned long long>(r, rec, mh, thr_near, nblk, cls, rrot, sh, hp);
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const uint32_t nb = __shfl_sync(0xffffffffu, nblk, 8 * q);
                if (r0 + q < np) {
                    uint4 *dst = (uint4 *)(nl16 + (size_t)(tc.g0 + p0 + r0 + q) * stride);
                    const uint4 *src = (const uint4 *)(rb + (r0 + q) * rpitch);
                    for (uint32_t v = lane; v < nb; v += 32) dst[v] = src[v];
                }
            }
            if (live && cls == 0) {
                nl_cnt[tc.g0 + p0 + qr] = min(n, 8u * nblk) | (K << MD_NL_NEAR_SHIFT);
                total += n;
            }
            __syncwarp();
        }
    }
    total += __shfl_xor_sync(0xffffffffu, total, 8);
    total += __shfl_xor_sync(0xffffffffu, total, 16);
    if (lane == 0 && total) atomicAdd(&flags->nl_total, total);
    if (worst > stride) atomicMax(&flags->nl_overflow, worst);
}

// ===============================================================================================================
// S4a LJ forces, one CTA per tile, W threads per home particle
// ===============================================================================================================
struct LJTile {
    double rc2_exact, sig2, eps24, eps4, uc;
    double thr_in, thr_out;  // rc^2 -+ guard
    double near2;            // MD_MIXED: pairs with r^2 below this are evaluated in fp64 on the global positions (R25)
};

// one pair by the plain fp64 definition on the global positions (MD_MIXED, pairs of the first shell: DESIGN.md R25)
__device__ __noinline__ void lj_near_pair(const double4 *__restrict__ pos, double Lx, double Ly, double Lz, uint32_t gi,
                                          uint32_t gj, double rc2_exact, double sig2, double eps24, double eps4, double uc,
                                          double *acc /* fx, fy, fz, energy: accumulated */)
{
    const double4 a = pos[gi], b = pos[gj];
    const double dx = md_min_image(__dsub_rn(a.x, b.x), Lx, 0.5 * Lx);
    const double dy = md_min_image(__dsub_rn(a.y, b.y), Ly, 0.5 * Ly);
    const double dz = md_min_image(__dsub_rn(a.z, b.z), Lz, 0.5 * Lz);
    const double r2 = md_r2_exact(dx, dy, dz);
    if (r2 < rc2_exact) {
        const double rinv2 = 1.0 / r2;
        const double s2 = sig2 * rinv2, s6 = s2 * s2 * s2;
        const double f = eps24 * s6 * (2.0 * s6 - 1.0) * rinv2;
        acc[0] += f * dx; acc[1] += f * dy; acc[2] += f * dz;
        acc[3] += 0.5 * (eps4 * s6 * (s6 - 1.0) - uc);
    }
}

// record referenced by a list entry: PRE = the entry is (staged index << 4), i.e. the byte offset of a float4 record
template <typename R4, bool PRE>
__device__ __forceinline__ R4 tile_rec(const R4 *rec, uint32_t ent)
{
    if (PRE) return *(const R4 *)((const char *)rec + (size_t)ent * (sizeof(R4) / 16));
    return rec[ent];
}

template <int W, bool MIXED, int ACC_BLOCK, bool ENERGY, bool PRE>
__global__ void __launch_bounds__(TILE_MAX_BLOCK) k_tile_lj(TileParams tp, Geom g, const double4 *__restrict__ pos,
                                                            const float4 *__restrict__ rel,
                                                            const uint32_t *__restrict__ nl_cnt,
                                                            const uint16_t *__restrict__ nl16, LJTile lj,
                                                            uint32_t max_staged, double4 *__restrict__ force, Gate gate)
{
    if (md_gate_closed(gate)) return;
    typedef typename std::conditional<MIXED, float4, double4>::type R4;
    typedef typename RecTraits<R4>::real real;
    extern __shared__ __align__(16) char smem_raw[];
    const TileSmem h = tile_carve(smem_raw, tp.B);
    R4 *rec = (R4 *)h.rest;
    uint8_t *scell = (uint8_t *)(h.rest + sizeof(R4) * (max_staged + N_DUMMY));

    TileCtx tc;
    tile_setup<MIXED>(tp, g, blockIdx.x, h, tc);
    if constexpr (MIXED) tile_stage_rel<false>(tc, h, rel, (float4 *)rec, scell, 1.f, pos, g);
    else tile_stage<R4, false>(g, tc, h, pos, nullptr, rec, nullptr, scell);
    __syncthreads();

    const unsigned lane = threadIdx.x & (W - 1);
    const unsigned seg_mask = md_seg_mask<W>();
    const uint32_t n_groups = blockDim.x / W;
    const real thr_in = (real)lj.thr_in, thr_out = (real)lj.thr_out;
    const real sig2 = (real)lj.sig2, eps24 = (real)lj.eps24, eps4 = (real)lj.eps4, uc = (real)lj.uc;
    const uint32_t stride8 = tp.stride >> 3;

    for (uint32_t p = threadIdx.x / W; p < tc.n_home; p += n_groups) {
        const uint32_t hc = tile_home_cell(h, tc.n_hc, p);
        const R4 me = rec[tile_staged_of_home(h, hc, p)];
        const uint32_t cnt = nl_cnt[tc.g0 + p] & MD_NL_CNT_MASK;
        const uint32_t nblk = (cnt + 7u) >> 3;
        const uint4 *row = (const uint4 *)nl16 + (size_t)(tc.g0 + p) * stride8;
        double fx = 0.0, fy = 0.0, fz = 0.0, en = 0.0;
        uint4 q = lane < nblk ? __ldg(row + lane) : make_uint4(0, 0, 0, 0);
        for (uint32_t b = lane; b < nblk; b += W) {
            const uint4 qn = b + W < nblk ? __ldg(row + b + W) : q;  // prefetch the next block of 8 entries
            const uint32_t qq[4] = {q.x, q.y, q.z, q.w};
            real ax = 0, ay = 0, az = 0, ae = 0;
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                const uint32_t ent = (e & 1) ? (qq[e >> 1] >> 16) : (qq[e >> 1] & 0xffffu);
                const R4 pj = tile_rec<R4, PRE>(rec, ent);
                const real dx = me.x - pj.x, dy = me.y - pj.y, dz = me.z - pj.z;
                const real r2 = dx * dx + dy * dy + dz * dz;
                bool in = r2 < thr_in;
                if (!in && r2 < thr_out) {  // guard band around rc^2: the plain fp64 definition decides (R26)
                    const uint32_t j = PRE ? ent >> 4 : ent;
                    in = tile_exact_r2(pos, g, tc.g0 + p, tile_global_of_staged(h, tc.n_sc, j)) < lj.rc2_exact;
                }
                if (MIXED && r2 < (real)lj.near2) {  // first shell: fp64 on the global positions
                    double acc[4] = {0.0, 0.0, 0.0, 0.0};
                    lj_near_pair(pos, g.L[0], g.L[1], g.L[2], tc.g0 + p, tile_global_of_staged(h, tc.n_sc, PRE ? ent >> 4 : ent),
                                 lj.rc2_exact, lj.sig2, lj.eps24, lj.eps4, lj.uc, acc);
                    fx += acc[0]; fy += acc[1]; fz += acc[2];
                    if (ENERGY) en += acc[3];
                    in = false;
                }
                const real rinv2 = md_rcp(r2);
                const real s2 = sig2 * rinv2;
                const real s6 = s2 * s2 * s2;
                real f = eps24 * s6 * ((real)2 * s6 - (real)1) * rinv2;
                f = in ? f : (real)0;
                ax += f * dx; ay += f * dy; az += f * dz;
                if (ENERGY) {
                    real u = (real)0.5 * (eps4 * s6 * (s6 - (real)1) - uc);
                    ae += in ? u : (real)0;
                }
                if (MIXED && ((e + 1) % ACC_BLOCK == 0)) {  // widen the fp32 block sum, accumulate in fp64
                    fx += (double)ax; fy += (double)ay; fz += (double)az;
                    ax = ay = az = 0;
                    if (ENERGY) { en += (double)ae; ae = 0; }
                }
            }
            if (!MIXED) { fx += ax; fy += ay; fz += az; en += ae; }
            q = qn;
        }
        fx = md_seg_sum<W>(fx, seg_mask);
        fy = md_seg_sum<W>(fy, seg_mask);
        fz = md_seg_sum<W>(fz, seg_mask);
        if (ENERGY) en = md_seg_sum<W>(en, seg_mask);
        if (lane == 0) force[tc.g0 + p] = make_double4(fx, fy, fz, en);
    }
}

// ===============================================================================================================
// S4a, mixed precision, the bench path: k_tile_lj3
//
// Row layout written by k_tile_build: a row is a sequence of blocks of 8 entries; slot e of block b of the row of
// tile-local home particle p holds a record whose staged index s has bank class  s & 7 == (e + b + 4 (p & 1)) & 7
// (a real neighbour, or the dummy record of that class); the few entries of classes longer than the row sit in
// holes of shorter classes.  A float4 record is 16 bytes, so the class is the 16-byte bank group of the record, and
// an LDS.128 is served one quarter-warp (8 lanes) per wavefront when the 8 records lie in 8 different groups.
// With W = 4 the lanes of a quarter-warp hold blocks b..b+3 of an even particle and b..b+3 of the next (odd) one,
// with W >= 8 they hold 8 consecutive blocks of one particle: at unrolled slot e the 8 records have the 8 different
// classes (e + b' + ...) & 7 -> the gather is conflict-free except for the relocated entries.
//
// Arithmetic (R1, R25, R26).  Far blocks (all but the last K of a row): packed fp32.  Coordinates stay in box
// units (the staging is exact, tile_stage_exact); s2 = sigma^2 / r^2, per pair g = (s6 - 1/2) s6 s2 and
// F_i = (48 eps / sigma^2) sum_j g d_ij.  The r < rc decision: d = r^2 - rc^2 in fp32; |d| >= guard decides by sign; a block of
// 8 entries in which some |d| < guard is re-evaluated with the exact fp64 test.  8 contributions are summed in fp32, the
// block sum is widened and accumulated in fp64 (MD_OPT_ACC_BLOCK = 8).  Near section (the last K blocks: every neighbour
// that can be closer than MD_NEAR_SIGMAS sigma before the next rebuild, see near_partition): fp64 on separations rebuilt
// from the staged records and their residuals (lj3_near) -- fp32 cannot hold the 1e-4 bar on the first shell.
// ===============================================================================================================
struct LJ3U {
    double rc2_exact;     // rc^2 (exact re-test)
    double sig2;          // sigma^2
    double guard64;       // decision band of the near section around rc^2 (rebuilt fp64 separations)
    double fscale;        // 48 eps / sigma^2
    float rc2s, guard;    // rc^2 and the guard band of the fp32 far loop
    float sig2f;
};


__device__ __forceinline__ float4 lds_f4(uint32_t addr)
{
    float4 v;
    asm("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}
// 16-byte read-only load of list entries; the L2 sector promotion pulls the rest of the (contiguous) row into L2
__device__ __forceinline__ uint4 ldg_row(const uint4 *p)
{
    uint4 v;
    asm volatile("ld.global.nc.L2::256B.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ unsigned long long lds_u64(uint32_t addr)
{
    unsigned long long v;
    asm("ld.shared.b64 %0, [%1];" : "=l"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ unsigned long long f2_pack(float a, float b)
{
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b));
    return r;
}
// same, but opaque to the optimiser: the pair is formed once and stays in an aligned register pair (loop invariants)
__device__ __forceinline__ unsigned long long f2_pack_fixed(float a, float b)
{
    unsigned long long r;
    asm volatile("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b));
    return r;
}
__device__ __forceinline__ void f2_unpack(unsigned long long v, float &a, float &b)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v));
}
__device__ __forceinline__ unsigned long long f2_mul(unsigned long long a, unsigned long long b)
{
    unsigned long long r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ unsigned long long f2_add(unsigned long long a, unsigned long long b)
{
    unsigned long long r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ unsigned long long f2_fma(unsigned long long a, unsigned long long b, unsigned long long c)
{
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}

// slow path of one block of 8 entries.  The fast path treats a pair inside the guard band as out of range, so what is
// left to do is ADD the pairs of the band that the exact fp64 test puts inside rc (R26).
__device__ __noinline__ void lj3_block_corr(const uint4 q, uint32_t rec_addr, float mx, float my, float mz, float rc2s,
                                           float guard, float sig2, const double4 *__restrict__ pos, double Lx, double Ly, double Lz,
                                           double rc2_exact, uint32_t gi, const uint32_t *gstart, const uint32_t *sstart,
                                           uint32_t n_sc, float *out)
{
    const uint32_t qq[4] = {q.x, q.y, q.z, q.w};
    float ax = 0.f, ay = 0.f, az = 0.f;
#pragma unroll 1
    for (int e = 0; e < 8; ++e) {
        const uint32_t off = (e & 1) ? (qq[e >> 1] >> 16) : (qq[e >> 1] & 0xffffu);
        const float4 pj = lds_f4(rec_addr + off);
        const float dx = mx - pj.x, dy = my - pj.y, dz = mz - pj.z;
        const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
        if (fabsf(r2 - rc2s) < guard) {
            const uint32_t s = off >> 4;
            uint32_t lo = 0, hi = n_sc;
            while (hi - lo > 1) {
                const uint32_t mid = (lo + hi) >> 1;
                if (sstart[mid] <= s) lo = mid; else hi = mid;
            }
            if (tile_exact_r2_impl(pos, Lx, Ly, Lz, gi, gstart[lo] + (s - sstart[lo])) < rc2_exact) {
                const float rinv2 = md_rcp(r2) * sig2;
                const float s6 = rinv2 * rinv2 * rinv2;
                const float f = (s6 - 0.5f) * (s6 * rinv2);
                ax = fmaf(f, dx, ax); ay = fmaf(f, dy, ay); az = fmaf(f, dz, az);
            }
        }
    }
    out[0] = ax; out[1] = ay; out[2] = az;
}

__device__ __forceinline__ double md_rcp_nr1(double x);

// Near section of a row (its first K blocks, see near_partition): fp32 separations cannot hold the 1e-4 bar on the steep
// part of the potential (|dF/dr| ~ 450 at r ~ sigma: a coordinate error of 5e-7 is 2e-4 in the force; R25), so
// these blocks are evaluated in fp64 on separations rebuilt from the staged records and their residuals
// (tile_stage_exact): d = (x_i - x_j) + qr (res_i - res_j), the first term an exact fp32 difference of grid values, good
// to ~1e-9, with the same shared-memory gather as the far loop and inside the same loop over the row's blocks.
// r < rc: decided by the rebuilt r^2 outside a band of width `guard`, by the exact expression on the global positions
// inside it (R26).  Returns sum g d of one block of 8 entries.
__device__ __noinline__ void lj3_near(const uint2 *__restrict__ halves, uint32_t n_halves, uint32_t lane, uint32_t W,
                                      uint32_t rec_addr, float4 me, double qr, double sig2, double rc2, double guard,
                                      const double4 *__restrict__ pos, double Lx, double Ly, double Lz, uint32_t gi,
                                      const uint32_t *gstart, const uint32_t *sstart, uint32_t n_sc, double *out)
{
    const uint32_t mw = __float_as_uint(me.w);
    // d = (x_i - x_j) + qr (f_i - f_j), f the biased residual fields (0 .. 1020), without an int -> double conversion: the
    // double with high word 0x43300000 and low word n IS 2^52 + n, so with n = f_i + 1024 - f_j (positive) and
    // Cq = qr (2^52 + 1024):  d = fma(qr, 2^52 + n, (x_i - Cq) - x_j), every step exact (qr is a power of two, the coordinates
    // are multiples of 512 qr below 2^33 qr), one rounding at the end
    const int mrx = md_res_x(mw) + 1024, mry = md_res_y(mw) + 1024, mrz = md_res_z(mw) + 1024;
    const double Cq = qr * (MD_TWO52 + 1024.0);
    const double mx = (double)me.x - Cq, my = (double)me.y - Cq, mz = (double)me.z - Cq;
    double ax = 0.0, ay = 0.0, az = 0.0;
    uint2 q = lane < n_halves ? __ldg(halves + lane) : make_uint2(0u, 0u);  // (prefetched into L1 by the caller)
    for (uint32_t u = lane; u < n_halves; u += W) {
        const uint2 qn = u + W < n_halves ? __ldg(halves + u + W) : q;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const uint32_t ww = e < 2 ? q.x : q.y;
            const uint32_t off = (e & 1) ? (ww >> 16) : (ww & 0xffffu);
            const float4 pj = lds_f4(rec_addr + off);
            const uint32_t pw = __float_as_uint(pj.w);
            const double dx = fma(qr, __hiloint2double(0x43300000, mrx - md_res_x(pw)), mx - (double)pj.x);
            const double dy = fma(qr, __hiloint2double(0x43300000, mry - md_res_y(pw)), my - (double)pj.y);
            const double dz = fma(qr, __hiloint2double(0x43300000, mrz - md_res_z(pw)), mz - (double)pj.z);
            const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
            const double d = r2 - rc2;
            bool in = d < -guard;
            if (!in && d < guard) {  // (the dummy records of the padding are far outside)
                const uint32_t s = off >> 4;
                uint32_t lo = 0, hi = n_sc;
                while (hi - lo > 1) {
                    const uint32_t mid = (lo + hi) >> 1;
                    if (sstart[mid] <= s) lo = mid; else hi = mid;
                }
                in = tile_exact_r2_impl(pos, Lx, Ly, Lz, gi, gstart[lo] + (s - sstart[lo])) < rc2;
            }
            const double ri = sig2 * md_rcp_nr1(r2);
            const double s6 = ri * ri * ri;
            double f = (s6 - 0.5) * (s6 * ri);
            f = in ? f : 0.0;
            ax = fma(f, dx, ax); ay = fma(f, dy, ay); az = fma(f, dz, az);
        }
        q = qn;
    }
    out[0] = ax; out[1] = ay; out[2] = az;
}

template <int W, bool X2>
__global__ void __launch_bounds__(MD_LJ3_MAX_BLOCK, 4) k_tile_lj3(TileParams tp, Geom g, const double4 *__restrict__ pos,
                                                             const float4 *__restrict__ rel,
                                                             const uint32_t *__restrict__ nl_cnt,
                                                             const uint16_t *__restrict__ nl16, LJ3U lj,
                                                             uint32_t max_staged,
                                                             double4 *__restrict__ force, Gate gate)
{
    if (md_gate_closed(gate)) return;
    extern __shared__ __align__(16) char smem_raw[];
    float4 *rec = (float4 *)smem_raw;  // records first: their shared-memory address is a launch constant
    const TileSmem h = tile_carve(smem_raw + sizeof(float4) * (max_staged + N_DUMMY), tp.B);
    uint8_t *scell = (uint8_t *)h.rest;

    TileCtx tc;
    tile_setup(tp, g, blockIdx.x, h, tc);
    tile_stage_exact(tc, h, rel, rec);
    // staged index of every home particle (replaces a search per particle)
    uint16_t *hsidx = (uint16_t *)(scell + ((max_staged + 16) & ~15u));
    for (uint32_t hc = threadIdx.x >> 5; hc < tc.n_hc; hc += blockDim.x >> 5) {
        const uint32_t p0 = h.hc_first[hc], p1 = h.hc_first[hc + 1], s0 = h.sstart[h.hc_sc[hc]];
        for (uint32_t p = p0 + (threadIdx.x & 31u); p < p1; p += 32) hsidx[p] = (uint16_t)(s0 + (p - p0));
    }
    // next unassigned home particle of each residue class (p mod 2 for W >= 4, mod 4 for W = 2, mod 8 for W = 1: the
    // row rotation)
    constexpr uint32_t NRES = W == 1 ? 8u : (W == 2 ? 4u : 2u);
    __shared__ uint32_t next_p[8];
    if (threadIdx.x < NRES) next_p[threadIdx.x] = blockDim.x / (NRES * W);
    __syncthreads();

    const unsigned lane = threadIdx.x & (W - 1);
    const unsigned seg_mask = md_seg_mask<W>();
    const uint32_t rec_addr = (uint32_t)__cvta_generic_to_shared(rec);
    const float rc2s = lj.rc2s, guard = lj.guard, nguard = -lj.guard;
    const uint32_t stride8 = tp.stride >> 3;

    // software pipeline over the group's particles: the row length and the first block of the NEXT particle are
    // requested before the current one is evaluated (rows have a fixed stride, so block `lane` of a row always exists)
    // Particles are handed out dynamically (rows differ in length): a group takes the next particle of ITS parity --
    // the bank-class layout ties the parity of the home index to the half of the quarter-warp the group sits in --
    // from a shared counter, one particle ahead of the one it evaluates.
    const uint32_t grp = threadIdx.x / W, par = grp & (NRES - 1u);
    auto grab = [&]() -> uint32_t {
        uint32_t v = 0;
        if (lane == 0) v = atomicAdd(&next_p[par], 1u);
        return NRES * __shfl_sync(seg_mask, v, 0, W) + par;
    };
    uint32_t p = grp;
    uint32_t cnt_c = 0;
    uint4 q_c = make_uint4(0, 0, 0, 0);
    if (p < tc.n_home) {
        cnt_c = __ldg(nl_cnt + tc.g0 + p);
        q_c = ldg_row((const uint4 *)nl16 + (size_t)(tc.g0 + p) * stride8 + lane);
    }
    while (p < tc.n_home) {
        const float4 me = rec[hsidx[p]];
        const uint32_t n_near_blk = cnt_c >> MD_NL_NEAR_SHIFT;                          // the last K blocks: fp64 (lj3_near)
        const uint32_t nblk = (((cnt_c & MD_NL_CNT_MASK) + 7u) >> 3) - n_near_blk;      // far blocks: fp32 below
        const uint4 *row = (const uint4 *)nl16 + (size_t)(tc.g0 + p) * stride8;
        uint4 q = q_c;
        const uint32_t pn = grab();
        if (pn < tc.n_home) {
            cnt_c = __ldg(nl_cnt + tc.g0 + pn);
            q_c = ldg_row((const uint4 *)nl16 + (size_t)(tc.g0 + pn) * stride8 + lane);
        }
        double fx = 0.0, fy = 0.0, fz = 0.0;
        // the lane's first half-block of the near section is requested now (into L1, no register) and used after the far loop
        const uint2 *halves = (const uint2 *)(row + nblk);
        if (lane < 2u * n_near_blk) asm volatile("prefetch.global.L1 [%0];" ::"l"(halves + lane));
        for (uint32_t b = lane; b < nblk; b += W) {
            const uint4 qn = b + W < nblk ? __ldg(row + b + W) : q;  // prefetch the next block of 8 entries
            const uint32_t qq[4] = {q.x, q.y, q.z, q.w};
            float ax, ay, az, band = 3e38f;
            if (X2) {
                unsigned long long ax2 = 0ull, ay2 = 0ull, az2 = 0ull;  // (0.f, 0.f)
                const unsigned long long mrc2 = f2_pack(-rc2s, -rc2s), mhalf = f2_pack(-0.5f, -0.5f);
                const unsigned long long sg2 = f2_pack(lj.sig2f, lj.sig2f);
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const float4 pa = lds_f4(rec_addr + (qq[e] & 0xffffu));
                    const float4 pb = lds_f4(rec_addr + (qq[e] >> 16));
                    const unsigned long long dx = f2_pack(me.x - pa.x, me.x - pb.x);
                    const unsigned long long dy = f2_pack(me.y - pa.y, me.y - pb.y);
                    const unsigned long long dz = f2_pack(me.z - pa.z, me.z - pb.z);
                    const unsigned long long r2 = f2_fma(dz, dz, f2_fma(dy, dy, f2_mul(dx, dx)));
                    const unsigned long long d = f2_add(r2, mrc2);
                    float r2a, r2b, da, db;
                    f2_unpack(r2, r2a, r2b);
                    f2_unpack(d, da, db);
                    band = fminf(band, fminf(fabsf(da), fabsf(db)));
                    const unsigned long long ri = f2_mul(f2_pack(md_rcp(r2a), md_rcp(r2b)), sg2);
                    const unsigned long long s6 = f2_mul(f2_mul(ri, ri), ri);
                    const unsigned long long ff = f2_mul(f2_add(s6, mhalf), f2_mul(s6, ri));
                    float fa, fb;
                    f2_unpack(ff, fa, fb);
                    fa = da < nguard ? fa : 0.f;
                    fb = db < nguard ? fb : 0.f;
                    const unsigned long long f = f2_pack(fa, fb);
                    ax2 = f2_fma(f, dx, ax2);
                    ay2 = f2_fma(f, dy, ay2);
                    az2 = f2_fma(f, dz, az2);
                }
                float t0, t1;
                f2_unpack(ax2, t0, t1); ax = t0 + t1;
                f2_unpack(ay2, t0, t1); ay = t0 + t1;
                f2_unpack(az2, t0, t1); az = t0 + t1;
            } else {
                ax = ay = az = 0.f;
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const uint32_t off = (e & 1) ? (qq[e >> 1] >> 16) : (qq[e >> 1] & 0xffffu);
                    const float4 pj = lds_f4(rec_addr + off);
                    const float dx = me.x - pj.x, dy = me.y - pj.y, dz = me.z - pj.z;
                    const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                    const float d = r2 - rc2s;
                    band = fminf(band, fabsf(d));
                    const float rinv2 = md_rcp(r2) * lj.sig2f;
                    const float s6 = rinv2 * rinv2 * rinv2;
                    float f = (s6 - 0.5f) * (s6 * rinv2);
                    f = d < nguard ? f : 0.f;
                    ax = fmaf(f, dx, ax); ay = fmaf(f, dy, ay); az = fmaf(f, dz, az);
                }
            }
            if (band < guard) {  // some pair of this block is inside the guard band: exact decisions (rare)
                float o[3];
                lj3_block_corr(q, rec_addr, me.x, me.y, me.z, rc2s, guard, lj.sig2f, pos, g.L[0], g.L[1], g.L[2], lj.rc2_exact,
                               tc.g0 + p, h.gstart, h.sstart, tc.n_sc, o);
                ax += o[0]; ay += o[1]; az += o[2];
            }
            fx += (double)ax; fy += (double)ay; fz += (double)az;
            q = qn;
        }
        if (n_near_blk) {  // the fp64 near section
            double o[3];
            lj3_near(halves, 2u * n_near_blk, lane, W, rec_addr, me, g.qr, lj.sig2, lj.rc2_exact, lj.guard64, pos, g.L[0],
                     g.L[1], g.L[2], tc.g0 + p, h.gstart, h.sstart, tc.n_sc, o);
            fx += o[0]; fy += o[1]; fz += o[2];
        }
        fx = md_seg_sum<W>(fx, seg_mask);
        fy = md_seg_sum<W>(fy, seg_mask);
        fz = md_seg_sum<W>(fz, seg_mask);
        if (lane == 0) force[tc.g0 + p] = make_double4(fx * lj.fscale, fy * lj.fscale, fz * lj.fscale, 0.0);
        p = pn;
    }
}

// ===============================================================================================================
// S4a, fp64 (configs 1 and 5): k_tile_lj3d, the fp64 twin of k_tile_lj3.  Records are split into (x, y) pairs of 16
// bytes -- so the bank-class row layout makes the LDS.128 gather conflict-free exactly as for float4 records -- and a
// separate z array (LDS.64).  Coordinates are staged divided by sigma; g = (s6 - 1/2) s8, F_i = (48 eps / sigma) sum g d'.
// The reciprocal is MUFU.RCP64H plus one Newton step (relative error ~2^-46, far inside the 1e-10 bar); the r < rc
// decision uses the same guard band (fp64 width ~1e-14) with the exact re-test of R2.
// ===============================================================================================================
__device__ __forceinline__ double md_rcp_nr1(double x)
{
    // MUFU.RCP64H (relative error e ~ 2^-23) and one third-order step y (1 + e + e^2): relative error e^3 ~ 2^-69, i.e. a
    // correctly rounded reciprocal up to the last bit.  (A plain Newton step leaves 2^-46; times the r^-14 sensitivity
    // of the pair term that is 2e-11 absolute on a first-shell pair -- above the 1e-10 bar for the few particles of a
    // million whose net force nearly cancels.)
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y, 1.0);
    return fma(y, fma(e, e, e), y);
}
__device__ __forceinline__ double2 lds_d2(uint32_t addr)
{
    double2 v;
    asm("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ double lds_d(uint32_t addr)
{
    double v;
    asm("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}

struct LJ3D {
    double rc2_exact, inv_sigma, fscale, rc2s, guard;
    double eps4, uc;  // energies: U = 4 eps (s12 - s6) - U(rc), half to each particle
};

template <bool PRE>
__device__ __noinline__ void lj3d_block_corr(const uint4 q, uint32_t xy_addr, uint32_t z_addr, double mx, double my, double mz,
                                            double rc2s, double guard, const double4 *__restrict__ pos, double Lx, double Ly,
                                            double Lz, double rc2_exact, double eps4, double uc, uint32_t gi,
                                            const uint32_t *gstart, const uint32_t *sstart, uint32_t n_sc, double *out)
{
    const uint32_t qq[4] = {q.x, q.y, q.z, q.w};
    double ax = 0.0, ay = 0.0, az = 0.0, ae = 0.0;
#pragma unroll 1
    for (int e = 0; e < 8; ++e) {
        const uint32_t ent = (e & 1) ? (qq[e >> 1] >> 16) : (qq[e >> 1] & 0xffffu);
        const uint32_t s = PRE ? ent >> 4 : ent;
        const double2 pxy = lds_d2(xy_addr + 16u * s);
        const double pz = lds_d(z_addr + 8u * s);
        const double dx = mx - pxy.x, dy = my - pxy.y, dz = mz - pz;
        const double r2 = dx * dx + dy * dy + dz * dz;
        if (fabs(r2 - rc2s) < guard) {
            uint32_t lo = 0, hi = n_sc;
            while (hi - lo > 1) {
                const uint32_t mid = (lo + hi) >> 1;
                if (sstart[mid] <= s) lo = mid; else hi = mid;
            }
            if (tile_exact_r2_impl(pos, Lx, Ly, Lz, gi, gstart[lo] + (s - sstart[lo])) < rc2_exact) {
                const double rinv2 = md_rcp_nr1(r2);
                const double s6 = rinv2 * rinv2 * rinv2;
                const double f = (s6 - 0.5) * (s6 * rinv2);
                ax += f * dx; ay += f * dy; az += f * dz;
                ae += 0.5 * (eps4 * (s6 * s6 - s6) - uc);
            }
        }
    }
    out[0] = ax; out[1] = ay; out[2] = az; out[3] = ae;
}

template <int W, bool PRE, bool ENERGY>
__global__ void __launch_bounds__(TILE_MAX_BLOCK) k_tile_lj3d(TileParams tp, Geom g, const double4 *__restrict__ pos,
                                                              const uint32_t *__restrict__ nl_cnt,
                                                              const uint16_t *__restrict__ nl16, LJ3D lj,
                                                              uint32_t max_staged, double4 *__restrict__ force, Gate gate)
{
    if (md_gate_closed(gate)) return;
    extern __shared__ __align__(16) char smem_raw[];
    double2 *rxy = (double2 *)smem_raw;                       // records first: launch-constant shared addresses
    double *rz = (double *)(rxy + (max_staged + N_DUMMY));
    const TileSmem h = tile_carve((char *)(rz + ((max_staged + N_DUMMY + 1) & ~1u)), tp.B);
    uint8_t *scell = (uint8_t *)h.rest;
    uint16_t *hsidx = (uint16_t *)(scell + ((max_staged + 16) & ~15u));

    TileCtx tc;
    tile_setup<false>(tp, g, blockIdx.x, h, tc);
    {   // stage: coordinates relative to the brick centre, periodic image applied, divided by sigma (see tile_stage)
        const uint32_t lane32 = threadIdx.x & 31u, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
        for (uint32_t hc = wid; hc < tc.n_hc; hc += nw) {
            const uint32_t p0 = h.hc_first[hc], p1 = h.hc_first[hc + 1], s0 = h.sstart[h.hc_sc[hc]];
            for (uint32_t p = p0 + lane32; p < p1; p += 32) hsidx[p] = (uint16_t)(s0 + (p - p0));
        }
        tile_for_each_staged<double4>(
            tc, h, [&](uint32_t gi) { return pos[gi]; },
            [&](uint32_t s, uint32_t sc, const double4 &p) {
                const double *cg = h.cgeo + 6 * sc;
                rxy[s] = make_double2((cg[3] + md_min_image(p.x - cg[0], g.L[0], g.h[0])) * lj.inv_sigma,
                                      (cg[4] + md_min_image(p.y - cg[1], g.L[1], g.h[1])) * lj.inv_sigma);
                rz[s] = (cg[5] + md_min_image(p.z - cg[2], g.L[2], g.h[2])) * lj.inv_sigma;
            });
        if (threadIdx.x < N_DUMMY) {
            rxy[tc.n_staged + threadIdx.x] = make_double2(1e150, 1e150);
            rz[tc.n_staged + threadIdx.x] = 1e150;
        }
    }
    __syncthreads();

    const unsigned lane = threadIdx.x & (W - 1);
    const unsigned seg_mask = md_seg_mask<W>();
    const uint32_t n_groups = blockDim.x / W;
    const uint32_t xy_addr = (uint32_t)__cvta_generic_to_shared(rxy), z_addr = (uint32_t)__cvta_generic_to_shared(rz);
    const double rc2s = lj.rc2s, guard = lj.guard, nguard = -lj.guard;
    const uint32_t stride8 = tp.stride >> 3;

    uint32_t p = threadIdx.x / W;
    uint32_t cnt_c = 0;
    uint4 q_c = make_uint4(0, 0, 0, 0);
    if (p < tc.n_home) {  // software pipeline over the group's particles, as in k_tile_lj3
        cnt_c = __ldg(nl_cnt + tc.g0 + p) & MD_NL_CNT_MASK;
        q_c = __ldg((const uint4 *)nl16 + (size_t)(tc.g0 + p) * stride8 + lane);
    }
    for (; p < tc.n_home; p += n_groups) {
        const uint32_t self = hsidx[p];
        const double2 mxy = rxy[self];
        const double mz = rz[self];
        const uint32_t nblk = (cnt_c + 7u) >> 3;
        const uint4 *row = (const uint4 *)nl16 + (size_t)(tc.g0 + p) * stride8;
        uint4 q = q_c;
        if (p + n_groups < tc.n_home) {
            cnt_c = __ldg(nl_cnt + tc.g0 + p + n_groups) & MD_NL_CNT_MASK;
            q_c = __ldg(row + (size_t)n_groups * stride8 + lane);
        }
        double fx = 0.0, fy = 0.0, fz = 0.0, en = 0.0;
        for (uint32_t b = lane; b < nblk; b += W) {
            const uint4 qn = b + W < nblk ? __ldg(row + b + W) : q;  // prefetch the next block of 8 entries
            const uint32_t qq[4] = {q.x, q.y, q.z, q.w};
            bool band = false;
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                const uint32_t ent = (e & 1) ? (qq[e >> 1] >> 16) : (qq[e >> 1] & 0xffffu);
                // PRE: ent = staged index << 4 = byte offset of the (x, y) record
                const double2 pxy = lds_d2(xy_addr + (PRE ? ent : 16u * ent));
                const double pz = lds_d(z_addr + (PRE ? ent >> 1 : 8u * ent));
                const double dx = mxy.x - pxy.x, dy = mxy.y - pxy.y, dz = mz - pz;
                const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                const double d = r2 - rc2s;
                band |= fabs(d) < guard;
                const double rinv2 = md_rcp_nr1(r2);
                const double s6 = rinv2 * rinv2 * rinv2;
                double f = (s6 - 0.5) * (s6 * rinv2);
                f = d < nguard ? f : 0.0;
                fx = fma(f, dx, fx); fy = fma(f, dy, fy); fz = fma(f, dz, fz);
                if (ENERGY) en += d < nguard ? 0.5 * (lj.eps4 * (s6 * s6 - s6) - lj.uc) : 0.0;
            }
            if (band) {  // some pair of this block is inside the guard band: exact decisions (rare)
                double o[4];
                lj3d_block_corr<PRE>(q, xy_addr, z_addr, mxy.x, mxy.y, mz, rc2s, guard, pos, g.L[0], g.L[1], g.L[2],
                                     lj.rc2_exact, lj.eps4, lj.uc, tc.g0 + p, h.gstart, h.sstart, tc.n_sc, o);
                fx += o[0]; fy += o[1]; fz += o[2];
                if (ENERGY) en += o[3];
            }
            q = qn;
        }
        fx = md_seg_sum<W>(fx, seg_mask);
        fy = md_seg_sum<W>(fy, seg_mask);
        fz = md_seg_sum<W>(fz, seg_mask);
        if (ENERGY) en = md_seg_sum<W>(en, seg_mask);
        if (lane == 0) force[tc.g0 + p] = make_double4(fx * lj.fscale, fy * lj.fscale, fz * lj.fscale, en);
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
                                                             const uint32_t *__restrict__ nl_cnt,
                                                             const uint16_t *__restrict__ nl16, DPDTile dp,
                                                             uint32_t max_staged, double4 *__restrict__ force, Gate gate)
{
    if (md_gate_closed(gate)) return;
    extern __shared__ __align__(16) char smem_raw[];
    const TileSmem h = tile_carve(smem_raw, tp.B);
    double4 *rec = (double4 *)h.rest;
    double4 *svel = rec + (max_staged + N_DUMMY);
    uint8_t *scell = (uint8_t *)(svel + (max_staged + N_DUMMY));

    TileCtx tc;
    tile_setup<false>(tp, g, blockIdx.x, h, tc);
    tile_stage<double4, true>(g, tc, h, pos, vel, rec, svel, scell);
    if (threadIdx.x < N_DUMMY) svel[tc.n_staged + threadIdx.x] = make_double4(0, 0, 0, 1);
    __syncthreads();

    const unsigned lane = threadIdx.x & (W - 1);
    const unsigned seg_mask = md_seg_mask<W>();
    const uint32_t n_groups = blockDim.x / W;
    const uint32_t stride8 = tp.stride >> 3;
    const uint32_t sh = tp.shift;

    for (uint32_t p = threadIdx.x / W; p < tc.n_home; p += n_groups) {
        const uint32_t hc = tile_home_cell(h, tc.n_hc, p);
        const uint32_t self = tile_staged_of_home(h, hc, p);
        const double4 me = rec[self];
        const double4 vi = svel[self];
        const uint32_t ti = md_lane_to_tag(me.w);
        const uint32_t cnt = nl_cnt[tc.g0 + p] & MD_NL_CNT_MASK;
        const uint32_t nblk = (cnt + 7u) >> 3;
        const uint4 *row = (const uint4 *)nl16 + (size_t)(tc.g0 + p) * stride8;
        double fx = 0.0, fy = 0.0, fz = 0.0, en = 0.0;
        for (uint32_t b = lane; b < nblk; b += W) {
            const uint4 q = __ldg(row + b);
            const uint32_t qq[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                const uint32_t j = ((qq[e >> 1] >> ((e & 1) * 16)) & 0xffffu) >> sh;
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
// S4b, two-phase variant (the default): k_tile_dpd2.  Only ~38 % of the list entries of a DPD fluid are inside rc
// (r_list = 1.4 rc), and the pair term is heavy (fp64 rsqrt, 10 Philox rounds): evaluated in place, every lane of a
// warp pays for it at every entry at which ANY lane is in range.  Phase 1 runs the distance test over the group's
// row and compacts the in-range entries (W-lane prefix sum of the hit counts, the paper's Fig. 4 compaction applied
// to the force loop) into a per-group list in shared memory; phase 2 deals that list out evenly to the W lanes.
// Records are split into 16-byte pairs (x,y) (z,vx) (vy,vz) + a tag array, so that with the bank-class row layout the
// gathers are conflict-free (see k_tile_lj3d).
// ===============================================================================================================
__device__ __forceinline__ double md_rsqrt_nr1(double x)
{
    // MUFU.RSQ64H and one third-order step: with e = 1 - x y^2, 1/sqrt(x) = y (1 + e/2 + 3 e^2/8 + ...): error ~ e^3
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x * y, y, 1.0);
    return fma(y, e * fma(0.375, e, 0.5), y);
}

template <int W>
__global__ void __launch_bounds__(MD_DPD2_MAX_BLOCK, 4) k_tile_dpd2(TileParams tp, Geom g, const double4 *__restrict__ pos,
                                                              const double4 *__restrict__ vel,
                                                              const uint32_t *__restrict__ nl_cnt,
                                                              const uint16_t *__restrict__ nl16, DPDTile dp,
                                                              uint32_t max_staged, uint32_t max_home,
                                                              double4 *__restrict__ force, Gate gate)
{
    if (md_gate_closed(gate)) return;
    extern __shared__ __align__(16) char smem_raw[];
    const uint32_t ns = max_staged + N_DUMMY;
    double2 *ra = (double2 *)smem_raw;  // (x, y)
    double2 *rb = ra + ns;              // (z, vx)
    double2 *rc = rb + ns;              // (vy, vz)
    uint32_t *rt = (uint32_t *)(rc + ns);                                   // tag
    const TileSmem h = tile_carve((char *)(rt + ((ns + 3u) & ~3u)), tp.B);
    uint8_t *scell = (uint8_t *)h.rest;
    uint16_t *hsidx = (uint16_t *)(scell + ((max_staged + 16) & ~15u));
    uint16_t *stash = hsidx + ((max_home + 7u) & ~7u);                      // [stride][n_groups] in-range entries

    TileCtx tc;
    tile_setup<false>(tp, g, blockIdx.x, h, tc);
    {
        const uint32_t lane32 = threadIdx.x & 31u, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
        for (uint32_t hc = wid; hc < tc.n_hc; hc += nw) {
            const uint32_t p0 = h.hc_first[hc], p1 = h.hc_first[hc + 1], s0 = h.sstart[h.hc_sc[hc]];
            for (uint32_t p = p0 + lane32; p < p1; p += 32) hsidx[p] = (uint16_t)(s0 + (p - p0));
        }
        struct PV { double4 p, v; };
        tile_for_each_staged<PV>(
            tc, h, [&](uint32_t gi) { PV x; x.p = pos[gi]; x.v = vel[gi]; return x; },
            [&](uint32_t s, uint32_t sc, const PV &x) {
                const double *cg = h.cgeo + 6 * sc;
                ra[s] = make_double2(cg[3] + md_min_image(x.p.x - cg[0], g.L[0], g.h[0]),
                                     cg[4] + md_min_image(x.p.y - cg[1], g.L[1], g.h[1]));
                rb[s] = make_double2(cg[5] + md_min_image(x.p.z - cg[2], g.L[2], g.h[2]), x.v.x);
                rc[s] = make_double2(x.v.y, x.v.z);
                rt[s] = md_lane_to_tag(x.p.w);
            });
        if (threadIdx.x < N_DUMMY) {
            ra[tc.n_staged + threadIdx.x] = make_double2(1e150, 1e150);
            rb[tc.n_staged + threadIdx.x] = make_double2(1e150, 0.0);
        }
    }
    __syncthreads();

    const unsigned lane = threadIdx.x & (W - 1);
    const unsigned seg_mask = md_seg_mask<W>();
    const uint32_t n_groups = blockDim.x / W, grp = threadIdx.x / W;
    const uint32_t stride8 = tp.stride >> 3;
    const uint32_t sh = tp.shift;
    uint16_t *my_stash = stash + grp;

    for (uint32_t p = grp; p < tc.n_home; p += n_groups) {
        const uint32_t self = hsidx[p];
        const double2 ma = ra[self], mb = rb[self], mc = rc[self];
        const uint32_t ti = rt[self];
        const uint32_t nblk = ((nl_cnt[tc.g0 + p] & MD_NL_CNT_MASK) + 7u) >> 3;
        const uint4 *row = (const uint4 *)nl16 + (size_t)(tc.g0 + p) * stride8;
        // ---- phase 1: distance tests, in-range entries compacted into the group's list
        uint32_t n_in = 0;  // entries in the list so far (the same in all lanes of the group)
        for (uint32_t b0 = 0; b0 < nblk; b0 += W) {
            const uint32_t b = b0 + lane;
            uint32_t hits = 0;
            uint4 q = make_uint4(0, 0, 0, 0);
            if (b < nblk) {
                q = __ldg(row + b);
                const uint32_t qq[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const uint32_t j = ((qq[e >> 1] >> ((e & 1) * 16)) & 0xffffu) >> sh;
                    const double2 pa = ra[j];
                    const double pz = rb[j].x;
                    const double dx = ma.x - pa.x, dy = ma.y - pa.y, dz = mb.x - pz;
                    const double r2 = dx * dx + dy * dy + dz * dz;
                    bool in = r2 < dp.thr_in;
                    if (!in && r2 < dp.thr_out)
                        in = tile_exact_r2(pos, g, tc.g0 + p, tile_global_of_staged(h, tc.n_sc, j)) < dp.rc2_exact;
                    if (in && r2 > 0.0) hits |= 1u << e;
                }
            }
            // exclusive prefix of the hit counts over the W lanes of the group
            const uint32_t c = __popc(hits);
            uint32_t inc = c;
#pragma unroll
            for (int o = 1; o < W; o <<= 1) {
                const uint32_t u = __shfl_up_sync(seg_mask, inc, o, W);
                if ((int)lane >= o) inc += u;
            }
            uint32_t k = n_in + inc - c;
            n_in += __shfl_sync(seg_mask, inc, W - 1, W);
            const uint32_t qq[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                if ((hits >> e) & 1u) {
                    my_stash[k * n_groups] = (uint16_t)(((qq[e >> 1] >> ((e & 1) * 16)) & 0xffffu) >> sh);
                    ++k;
                }
            }
        }
        __syncwarp(seg_mask);
        // ---- phase 2: the heavy pair term, in-range pairs dealt out evenly to the W lanes
        const double vix = mb.y, viy = mc.x, viz = mc.y;
        double fx = 0.0, fy = 0.0, fz = 0.0, en = 0.0;
        for (uint32_t k = lane; k < n_in; k += W) {
            const uint32_t j = my_stash[k * n_groups];
            const double2 pa = ra[j], pb = rb[j], pc = rc[j];
            const double dx = ma.x - pa.x, dy = ma.y - pa.y, dz = mb.x - pb.x;
            const double r2 = dx * dx + dy * dy + dz * dz;
            const double rinv = md_rsqrt_nr1(r2);
            const double r = r2 * rinv;
            const double w = 1.0 - r * dp.inv_rc;
            const double rv = (dx * (vix - pb.y) + dy * (viy - pc.x) + dz * (viz - pc.y)) * rinv;
            const double theta = md_dpd_theta(ti, rt[j], dp.step, dp.seed);
            const double f = (dp.A * w - dp.gamma * w * w * rv + dp.sr * w * theta) * rinv;
            fx += f * dx; fy += f * dy; fz += f * dz;
            en += 0.25 * dp.A * dp.rc * w * w;
        }
        __syncwarp(seg_mask);
        fx = md_seg_sum<W>(fx, seg_mask);
        fy = md_seg_sum<W>(fy, seg_mask);
        fz = md_seg_sum<W>(fz, seg_mask);
        en = md_seg_sum<W>(en, seg_mask);
        if (lane == 0) force[tc.g0 + p] = make_double4(fx, fy, fz, en);
    }
}

// ===============================================================================================================
// decode the 16-bit tile list into the general 32-bit CSR (exports / parity read-back only).  The stored list is a
// guard-band superset; here every entry is tested with the exact fp64 expression (R2) on the positions the
// list was built from (pos_ref, the snapshot taken at the binning), so the exported list is the plain definition.
// FILL = false: exact row lengths into cnt32;  FILL = true: global slots into nl_idx at nl_off.
// ===============================================================================================================
template <bool FILL>
__global__ void k_tile_decode(TileParams tp, Geom g, const double *__restrict__ pos_ref,
                              const uint32_t *__restrict__ nl_cnt, const uint16_t *__restrict__ nl16, double rl2,
                              uint32_t *__restrict__ cnt32, const uint64_t *__restrict__ nl_off,
                              uint32_t *nl_idx)
{
    extern __shared__ __align__(16) char smem_raw[];
    const TileSmem h = tile_carve(smem_raw, tp.B);
    TileCtx tc;
    tile_setup<false>(tp, g, blockIdx.x, h, tc);
    const unsigned lane = threadIdx.x & 31u, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const unsigned lt = md_lanemask_lt();
    for (uint32_t p = wid; p < tc.n_home; p += nw) {
        const uint32_t gi = tc.g0 + p;
        const uint32_t rowg = gi;
        const uint32_t cnt = ((nl_cnt[rowg] & MD_NL_CNT_MASK) + 7u) & ~7u;  // stored rows are whole blocks of 8, dummies interspersed
        const uint16_t *row = nl16 + (size_t)rowg * tp.stride;
        const double xi = pos_ref[3ull * gi], yi = pos_ref[3ull * gi + 1], zi = pos_ref[3ull * gi + 2];
        uint32_t *out = FILL ? nl_idx + nl_off[gi] : nullptr;
        uint32_t n = 0;
        for (uint32_t k0 = 0; k0 < cnt; k0 += 32) {
            const uint32_t k = k0 + lane;
            bool keep = false;
            uint32_t gj = 0;
            if (k < cnt) {
                const uint32_t s = (uint32_t)row[k] >> tp.shift;
                if (s < tc.n_staged) {
                    gj = tile_global_of_staged(h, tc.n_sc, s);
                    const double dx = md_min_image(__dsub_rn(xi, pos_ref[3ull * gj]), g.L[0], g.h[0]);
                    const double dy = md_min_image(__dsub_rn(yi, pos_ref[3ull * gj + 1]), g.L[1], g.h[1]);
                    const double dz = md_min_image(__dsub_rn(zi, pos_ref[3ull * gj + 2]), g.L[2], g.h[2]);
                    keep = md_r2_exact(dx, dy, dz) < rl2;
                }
            }
            const unsigned bal = __ballot_sync(0xffffffffu, keep);
            if (FILL && keep) out[n + __popc(bal & lt)] = gj;
            n += __popc(bal);
        }
        if (!FILL && lane == 0) cnt32[gi] = n;
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
    tp.stride = c->nl_stride;
    tp.shift = c->nl_shift;
    tp.tile_cell_begin = c->tile_cell_begin;
    tp.tile_origin = c->tile_origin;
    tp.lin_of_rank = c->lin_of_rank;
    tp.rank_of_lin = c->rank_of_lin;
    tp.cell_start = c->cell_start;
    for (int a = 0; a < 3; ++a) tp.cw[a] = c->box[a] / (double)c->dims[a];
    // rows rotate so that the 8 lanes of a quarter-warp of the force kernel meet 8 different bank classes: with W >= 4
    // lanes per particle a quarter holds 2 particles x 4 blocks (rotation 0 / 4), with W = 2 it holds 4 particles x 2
    // blocks (rotation 0 / 2 / 4 / 6), with W = 1 eight particles x 1 block (rotation 0 .. 7).  Layout only: any
    // rotation is a correct list.
    tp.rot_mul = (uint32_t)c->nl_rotw;          // W = 1: rotation p & 7;  W = 2: 2 (p & 3);  W >= 4: 4 (p & 1)
    tp.rot_mask = 8u / (uint32_t)c->nl_rotw - 1u;
    tp.desc_words = (TILE_DESC_CTX + tile_desc_table_words(c->tile_B) + 3u) & ~3u;
    tp.desc = c->tile_desc_valid ? c->tile_desc : nullptr;
    return tp;
}

// bound on |r2_staged - r2_true| for staged coordinates of magnitude <= E per axis, separations <= R
// direct form (force kernels): r2 = dx^2 + dy^2 + dz^2 on rounded coordinates
static double guard_fp32(double E, double R)
{
    // a staged fp32 coordinate carries up to four roundings of magnitude <= E u: the cell-relative record, the fp32
    // offset of the cell image, their sum, the 1/sigma scaling (tile_stage_rel) -> 8 E u per separation component
    const double u = 5.9604644775390625e-08;  // 2^-24
    const double delta = 8.0 * E * u + u * R;
    return 1.5 * (2.0 * 1.7320508075688772 * R * delta + 3.0 * delta * delta + 4.0 * u * R * R);
}
static double guard_fp64(double E, double R)
{
    const double u = 1.1102230246251565e-16;  // 2^-53
    const double delta = 6.0 * E * u + u * R;
    return 4.0 * (2.0 * 1.7320508075688772 * R * delta + 3.0 * delta * delta + 4.0 * u * R * R);
}
// dot-product form (build kernel): t = |b|^2 - 2 a.b, compared with thr - |a|^2, all fp32.  Coordinates are rounded
// once (error E u each, i.e. <= 2 sqrt(3) R E u on r^2 as above); then |a|^2, |b|^2 (<= 3 E^2 each, 3 roundings), the
// three FFMA of the dot product (partial sums <= 9 E^2) and the final subtraction each add <= u times their magnitude:
// generously 40 E^2 u in total.
static double guard_dot_fp32(double E, double R)
{
    const double u = 5.9604644775390625e-08;
    return guard_fp32(E, R) + 40.0 * E * E * u;
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
    s += rec_bytes * (c->tile_max_staged + N_DUMMY);
    if (with_vel) s += sizeof(double4) * (c->tile_max_staged + N_DUMMY);
    s += (c->tile_max_staged + 16) & ~(size_t)15;  // staged-cell table of tile_stage
    return s;
}

int tile_measure(md_ctx *c)
{
    MD_CUDA_CHECK(c, cudaMemsetAsync(&c->d_flags->max_home, 0, 2 * sizeof(unsigned int), c->stream));
    c->tile_desc_valid = false;
    TileParams tp = make_tp(c);  // slow-path setup inside k_tile_header
    const uint64_t need = (uint64_t)c->n_tiles * tp.desc_words;
    if (need > c->tile_desc_len) {
        if (c->tile_desc) { md_free(c, c->tile_desc); c->tile_desc = nullptr; }
        c->tile_desc_len = 0;
        MD_TRY(md_alloc(c, (void **)&c->tile_desc, need * sizeof(uint32_t)));
        c->tile_desc_len = need;
    }
    const size_t smem = tile_header_bytes(c->tile_B);
    if (smem > 40 * 1024)
        MD_CUDA_CHECK(c, cudaFuncSetAttribute(k_tile_header, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k_tile_header<<<c->n_tiles, 128, smem, c->stream>>>(tp, c->g, c->tile_desc, &c->d_flags->max_home, &c->d_flags->max_staged);
    MD_LAUNCH_CHECK(c);
    c->tile_desc_valid = true;
    return MD_OK;
}

template <typename K>
static int set_smem(md_ctx *c, K kernel, size_t bytes)
{
    // (opt in well below the 48 KB default limit: it counts static + dynamic shared memory)
    if (bytes > 40 * 1024) MD_CUDA_CHECK(c, cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    return MD_OK;
}

static const size_t TILE_SMEM_LIMIT = 227 * 1024 - 1024;  // dynamic part: the kernels also hold a few hundred bytes of static shared memory

// entries are pre-shifted byte offsets when every staged index (and the dummy) fits in 12 bits
static uint32_t tile_shift(md_ctx *c) { return c->tile_max_staged + N_DUMMY <= 4096 ? 4u : 0u; }

// returns MD_OK and sets *fits = false if the largest tile does not fit in shared memory (caller falls back)

static int tile_build_mode()
{
    static const int build_mode = getenv("B200MD_BUILD") ? atoi(getenv("B200MD_BUILD")) : 8;
    return build_mode;
}
// k_tile_build8: 4 candidate phases per home particle; ballot variants: a full warp
int tile_build_lanes(md_ctx *) { return tile_build_mode() == 8 ? 4 : 32; }

int launch_tile_build(md_ctx *c, bool *fits)
{
    const uint32_t ms = c->tile_max_staged;
    const int block = std::min(c->cfg[MD_K_NLIST].block, TILE_MAX_BLOCK);
    const uint32_t nw = (uint32_t)block / 32;
    size_t smem = tile_smem_common(c, sizeof(float4), false);
    const bool b8 = tile_build_mode() == 8;
    const size_t rows = b8 ? BUILD8_P : BUILD_P;
    smem += sizeof(uint16_t) * (size_t)nw * rows * (c->nl_stride + RB_EXTRA + (b8 ? 8 : 0)) + sizeof(uint32_t) * nw * (b8 ? 4 : rows) * 24;  // row assembly
    *fits = smem <= TILE_SMEM_LIMIT && ms + N_DUMMY <= 65536 && c->tile_B <= 4;
    if (!*fits) return MD_OK;
    c->nl_shift = tile_shift(c);
    {   // the force kernel that will read the list: the last step description says which, else LJ
        const bool dpd = (c->force_hint & MD_F_DPD) != 0 && !(c->force_hint & MD_F_LJ);
        c->nl_rotw = tile_rot_class(c->cfg[dpd ? MD_K_DPD : MD_K_LJ].w);
    }
    const double R = c->r_list * 1.001, E = tile_extent(c), rl2 = c->r_list * c->r_list;
    MD_CUDA_CHECK(c, cudaMemsetAsync(&c->d_flags->nl_total, 0, sizeof(unsigned long long), c->stream));
    MD_CUDA_CHECK(c, cudaMemsetAsync(&c->d_flags->nl_overflow, 0, sizeof(unsigned int), c->stream));
    TileParams tp = make_tp(c);
    const double gd = guard_dot_fp32(E, R);
    // near section (MD_MIXED, particle rows): neighbours within r_near + r_buff at the build, r_near = MD_NEAR_SIGMAS sigma
    // of the LJ parameters last seen (R25); the force kernel checks that the section covers its own sigma
    float thr_near = 0.f;
    c->nl_near_r = 0.0;
    static const double near_sig = getenv("B200MD_NEAR") ? atof(getenv("B200MD_NEAR")) : MD_NEAR_SIGMAS;  // diagnostic
    if (b8 && c->precision == MD_MIXED && near_sig > 0.0) {
        c->nl_near_r = near_sig * c->lj_sigma_hint;
        const double rn = c->nl_near_r + c->r_buff;
        thr_near = (float)(rn * rn + gd);
    }
    if (b8) {
        MD_TRY(set_smem(c, k_tile_build8, smem));
        k_tile_build8<<<c->n_tiles, block, smem, c->stream>>>(tp, c->g, c->rel, c->pos, (float)(rl2 + gd), thr_near, ms, c->nl_cnt,
                                                             c->nl16, c->d_flags);
    } else {
        MD_TRY(set_smem(c, k_tile_build<BUILD_P>, smem));
        k_tile_build<BUILD_P><<<c->n_tiles, block, smem, c->stream>>>(tp, c->g, c->rel, c->pos, (float)(rl2 + gd), ms, c->nl_cnt,
                                                                     c->nl16, c->d_flags);
    }
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

template <int W, bool MIXED, int ACC, bool ENERGY>
static int launch_lj_pre(md_ctx *c, const TileParams &tp, const LJTile &p, int block, size_t smem)
{
    if (c->nl_shift) {
        MD_TRY(set_smem(c, k_tile_lj<W, MIXED, ACC, ENERGY, true>, smem));
        k_tile_lj<W, MIXED, ACC, ENERGY, true><<<c->n_tiles, block, smem, c->stream>>>(tp, c->g, c->pos, c->rel, c->nl_cnt, c->nl16, p,
                                                                                     c->tile_max_staged, c->force, md_gate(c));
    } else {
        MD_TRY(set_smem(c, k_tile_lj<W, MIXED, ACC, ENERGY, false>, smem));
        k_tile_lj<W, MIXED, ACC, ENERGY, false><<<c->n_tiles, block, smem, c->stream>>>(tp, c->g, c->pos, c->rel, c->nl_cnt, c->nl16, p,
                                                                                      c->tile_max_staged, c->force, md_gate(c));
    }
    return MD_OK;
}

template <int W, bool MIXED, int ACC>
static int launch_lj_energy(md_ctx *c, const TileParams &tp, const LJTile &p, int block, size_t smem, bool energy)
{
    if (energy) return launch_lj_pre<W, MIXED, ACC, true>(c, tp, p, block, smem);
    return launch_lj_pre<W, MIXED, ACC, false>(c, tp, p, block, smem);
}

int launch_tile_lj(md_ctx *c, double eps, double sigma, int shift, bool energy)
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
    p.near2 = MD_NEAR_SIGMAS * MD_NEAR_SIGMAS * p.sig2;
    const size_t smem = tile_smem_common(c, mixed ? sizeof(float4) : sizeof(double4), false);
    TileParams tp = make_tp(c);
    static const int lj3_mode = getenv("B200MD_LJ3") ? atoi(getenv("B200MD_LJ3")) : 2;
    if (!mixed && lj3_mode) {
        const size_t ns = c->tile_max_staged + N_DUMMY;
        const size_t smemd = 16 * ns + 8 * ((ns + 1) & ~(size_t)1) + tile_header_bytes(c->tile_B) +
                             ((c->tile_max_staged + 16) & ~(size_t)15) + ((2 * (size_t)c->tile_max_home + 15) & ~(size_t)15);
        if (smemd <= TILE_SMEM_LIMIT) {
            LJ3D q;
            q.rc2_exact = p.rc2_exact;
            q.inv_sigma = 1.0 / sigma;
            q.fscale = 48.0 * eps / sigma;
            q.rc2s = p.rc2_exact / p.sig2;
            q.guard = 2.0 * gd / p.sig2 + 8.0 * 1.1102230246251565e-16 * q.rc2s;
            q.eps4 = p.eps4;
            q.uc = p.uc;
#define LJ3D_LAUNCH(PRE_, EN_)                                                                                              \
    do {                                                                                                                   \
        MD_TRY(set_smem(c, (k_tile_lj3d<W_, PRE_, EN_>), smemd));                                                         \
        k_tile_lj3d<W_, PRE_, EN_><<<c->n_tiles, cf.block, smemd, c->stream>>>(tp, c->g, c->pos, c->nl_cnt, c->nl16, q,    \
                                                                                c->tile_max_staged, c->force, md_gate(c));             \
    } while (0)
            MD_DISPATCH_W(cf.w, {
                if (c->nl_shift) { if (energy) LJ3D_LAUNCH(true, true); else LJ3D_LAUNCH(true, false); }
                else { if (energy) LJ3D_LAUNCH(false, true); else LJ3D_LAUNCH(false, false); }
            });
#undef LJ3D_LAUNCH
            MD_LAUNCH_CHECK(c);
            return MD_OK;
        }
    }
    if (mixed && !energy && c->nl_shift && c->acc_block == 8 && lj3_mode && (c->nl_near_r >= MD_NEAR_SIGMAS * sigma * (1.0 - 1e-12) || getenv("B200MD_NEAR"))) {
        const size_t smem = tile_smem_common(c, sizeof(float4), false) + ((2 * (size_t)c->tile_max_home + 15) & ~(size_t)15);
        LJ3U q;
        q.rc2_exact = p.rc2_exact;
        q.sig2 = p.sig2;
        q.sig2f = (float)p.sig2;
        q.fscale = 48.0 * eps / p.sig2;
        q.rc2s = (float)p.rc2_exact;
        // guard of the far loop: the fp32 error bound of r^2 plus the rounding of rc^2 itself
        q.guard = (float)(1.0001 * (gd + 2.0 * 5.9604644775390625e-08 * p.rc2_exact));
        {   // near section: a rebuilt separation component is good to ~2.5 qr (two residuals and two offsets of half a quantum)
            const double dsep = 2.5 * c->g.qr + 1e-15 * E;
            q.guard64 = 4.0 * (2.0 * 1.7320508075688772 * R * dsep + 3.0 * dsep * dsep);
        }
        const int w = cf.w > 8 ? 8 : cf.w;
        cf.block = std::min(cf.block, MD_LJ3_MAX_BLOCK);  // k_tile_lj3 is compiled for 4 CTAs of 256 threads per SM (64 registers)
        if (w <= 1) {
            MD_TRY(set_smem(c, (k_tile_lj3<1, true>), smem));
            k_tile_lj3<1, true><<<c->n_tiles, cf.block, smem, c->stream>>>(tp, c->g, c->pos, c->rel, c->nl_cnt, c->nl16, q, c->tile_max_staged, c->force, md_gate(c));
        } else if (w == 2) {  // rows laid out with rotation 2 (p & 3) when the list was built for W = 2 (launch_tile_build)
            MD_TRY(set_smem(c, (k_tile_lj3<2, true>), smem));
            k_tile_lj3<2, true><<<c->n_tiles, cf.block, smem, c->stream>>>(tp, c->g, c->pos, c->rel, c->nl_cnt, c->nl16, q, c->tile_max_staged, c->force, md_gate(c));
        } else if (w == 4) {
            if (lj3_mode == 2) {
                MD_TRY(set_smem(c, k_tile_lj3<4, true>, smem));
                k_tile_lj3<4, true><<<c->n_tiles, cf.block, smem, c->stream>>>(tp, c->g, c->pos, c->rel, c->nl_cnt, c->nl16, q, c->tile_max_staged, c->force, md_gate(c));
            } else {
                MD_TRY(set_smem(c, k_tile_lj3<4, false>, smem));
                k_tile_lj3<4, false><<<c->n_tiles, cf.block, smem, c->stream>>>(tp, c->g, c->pos, c->rel, c->nl_cnt, c->nl16, q, c->tile_max_staged, c->force, md_gate(c));
            }
        } else {
            if (lj3_mode == 2) {
                MD_TRY(set_smem(c, k_tile_lj3<8, true>, smem));
                k_tile_lj3<8, true><<<c->n_tiles, cf.block, smem, c->stream>>>(tp, c->g, c->pos, c->rel, c->nl_cnt, c->nl16, q, c->tile_max_staged, c->force, md_gate(c));
            } else {
                MD_TRY(set_smem(c, k_tile_lj3<8, false>, smem));
                k_tile_lj3<8, false><<<c->n_tiles, cf.block, smem, c->stream>>>(tp, c->g, c->pos, c->rel, c->nl_cnt, c->nl16, q, c->tile_max_staged, c->force, md_gate(c));
            }
        }
        MD_LAUNCH_CHECK(c);
        return MD_OK;
    }
    MD_DISPATCH_W(cf.w, {
        if (mixed) {
            if (c->acc_block == 1) MD_TRY((launch_lj_energy<W_, true, 1>(c, tp, p, cf.block, smem, energy)));
            else MD_TRY((launch_lj_energy<W_, true, 8>(c, tp, p, cf.block, smem, energy)));
        } else {
            MD_TRY((launch_lj_energy<W_, false, 8>(c, tp, p, cf.block, smem, energy)));
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
    TileParams tp = make_tp(c);
    static const int dpd_mode = getenv("B200MD_DPD") ? atoi(getenv("B200MD_DPD")) : 2;
    if (dpd_mode == 2) {
        cf.block = std::min(cf.block, MD_DPD2_MAX_BLOCK);  // k_tile_dpd2 is compiled for 4 CTAs of 256 threads per SM (64 registers)
        const size_t ns = c->tile_max_staged + N_DUMMY;
        const int w = std::max(1, std::min(cf.w, 32));
        const size_t n_groups = (size_t)cf.block / w;
        const size_t smem2 = 48 * ns + 4 * ((ns + 3) & ~(size_t)3) + tile_header_bytes(c->tile_B) +
                             ((c->tile_max_staged + 16) & ~(size_t)15) + 2 * (((size_t)c->tile_max_home + 7) & ~(size_t)7) +
                             2 * n_groups * c->nl_stride;
        if (smem2 <= TILE_SMEM_LIMIT) {
            MD_DISPATCH_W(cf.w, {
                MD_TRY(set_smem(c, k_tile_dpd2<W_>, smem2));
                k_tile_dpd2<W_><<<c->n_tiles, cf.block, smem2, c->stream>>>(tp, c->g, c->pos, c->vel, c->nl_cnt, c->nl16, p,
                                                                         c->tile_max_staged, c->tile_max_home, c->force, md_gate(c));
            });
            MD_LAUNCH_CHECK(c);
            return MD_OK;
        }
    }
    const size_t smem = tile_smem_common(c, sizeof(double4), true);
    MD_DISPATCH_W(cf.w, {
        MD_TRY(set_smem(c, k_tile_dpd<W_>, smem));
        k_tile_dpd<W_><<<c->n_tiles, cf.block, smem, c->stream>>>(tp, c->g, c->pos, c->vel, c->nl_cnt, c->nl16, p,
                                                               c->tile_max_staged, c->force, md_gate(c));
    });
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

bool tile_forces_fit(md_ctx *c, bool dpd)
{
    const size_t rec = (!dpd && c->precision == MD_MIXED) ? sizeof(float4) : sizeof(double4);
    return tile_smem_common(c, rec, dpd) <= TILE_SMEM_LIMIT;
}

// pass 1 (fill = false): exact row lengths into cnt32; pass 2 (fill = true): slots into nl_idx at nl_off
int launch_tile_decode(md_ctx *c, bool fill, uint32_t *cnt32)
{
    const size_t smem = tile_header_bytes(c->tile_B);
    const double rl2 = c->r_list * c->r_list;
    if (fill)
        k_tile_decode<true><<<c->n_tiles, 256, smem, c->stream>>>(make_tp(c), c->g, c->pos_ref, c->nl_cnt, c->nl16, rl2,
                                                                 nullptr, c->nl_off, c->nl_idx);
    else
        k_tile_decode<false><<<c->n_tiles, 256, smem, c->stream>>>(make_tp(c), c->g, c->pos_ref, c->nl_cnt, c->nl16, rl2,
                                                                  cnt32, nullptr, nullptr);
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}
