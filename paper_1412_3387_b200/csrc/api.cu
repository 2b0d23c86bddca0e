// api.cu -- the extern "C" boundary of libb200md (include/b200md.h): context lifetime, host/device pointer
// marshalling, S7 step scheduler, S8 runtime tuner.  No arithmetic of the method lives here.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>

#include "md_device.cuh"

// =====================================================================================================
// memory helpers
// =====================================================================================================
int md_alloc(md_ctx *c, void **p, uint64_t bytes)
{
    *p = nullptr;
    if (bytes == 0) bytes = 16;
    if (c->ws_base) {
        // first fit in the caller's workspace; buffers above 1/32 of it (neighbour lists, exports, staging: the ones that
        // are re-carved when they grow) are taken from the TOP so that they do not fragment the long-lived small ones
        const uint64_t need = (bytes + 255) & ~255ull;
        const bool big = need > c->ws_bytes / 32;
        const size_t nb = c->ws_blocks.size();
        for (size_t k = 0; k < nb; ++k) {
            const size_t i = big ? nb - 1 - k : k;
            if (c->ws_blocks[i].used || c->ws_blocks[i].size < need) continue;
            size_t at = i;
            if (c->ws_blocks[i].size > need) {
                const uint64_t off = c->ws_blocks[i].off, size = c->ws_blocks[i].size;
                if (big) {  // [free rest][this allocation]
                    c->ws_blocks[i].size = size - need;
                    c->ws_blocks.insert(c->ws_blocks.begin() + i + 1, md_ctx::WsBlock{off + size - need, need, false});
                    at = i + 1;
                } else {    // [this allocation][free rest]
                    c->ws_blocks[i].size = need;
                    c->ws_blocks.insert(c->ws_blocks.begin() + i + 1, md_ctx::WsBlock{off + need, size - need, false});
                }
            }
            c->ws_blocks[at].used = true;
            *p = c->ws_base + c->ws_blocks[at].off;
            c->device_bytes += need;
            c->ws_peak = std::max(c->ws_peak, c->ws_blocks[at].off + need);
            return MD_OK;
        }
        c->err = "workspace too small: " + std::to_string(bytes) + " more bytes needed, " + std::to_string(c->device_bytes) +
                 " of " + std::to_string(c->ws_bytes) + " in use (size it with md_workspace_bytes)";
        return MD_ENOMEM;
    }
    cudaError_t e = cudaMalloc(p, bytes);
    if (e != cudaSuccess) {
        c->err = std::string("cudaMalloc(") + std::to_string(bytes) + "): " + cudaGetErrorString(e);
        cudaGetLastError();
        return e == cudaErrorMemoryAllocation ? MD_ENOMEM : MD_ECUDA;
    }
    c->allocs.push_back({*p, bytes});
    c->device_bytes += bytes;
    return MD_OK;
}

void md_free(md_ctx *c, void *p)
{
    if (!p) return;
    if (c->ws_base) {  // work already enqueued on the context's stream still owns the block in stream order
        const uint64_t off = (uint64_t)((char *)p - c->ws_base);
        for (size_t i = 0; i < c->ws_blocks.size(); ++i) {
            if (c->ws_blocks[i].off != off || !c->ws_blocks[i].used) continue;
            c->ws_blocks[i].used = false;
            c->device_bytes -= c->ws_blocks[i].size;
            if (i + 1 < c->ws_blocks.size() && !c->ws_blocks[i + 1].used) {
                c->ws_blocks[i].size += c->ws_blocks[i + 1].size;
                c->ws_blocks.erase(c->ws_blocks.begin() + i + 1);
            }
            if (i > 0 && !c->ws_blocks[i - 1].used) {
                c->ws_blocks[i - 1].size += c->ws_blocks[i].size;
                c->ws_blocks.erase(c->ws_blocks.begin() + i);
            }
            return;
        }
        return;
    }
    for (auto it = c->allocs.begin(); it != c->allocs.end(); ++it)
        if (it->first == p) {
            c->device_bytes -= it->second;
            c->allocs.erase(it);
            break;
        }
    cudaFree(p);
}

int md_sync(md_ctx *c)
{
    MD_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    return MD_OK;
}

int md_read_flags(md_ctx *c)
{
    MD_CUDA_CHECK(c, cudaMemcpyAsync(c->h_flags, c->d_flags, sizeof(DevFlags), cudaMemcpyDeviceToHost, c->stream));
    MD_TRY(md_sync(c));
    if (c->profiling) prof_resolve(c);
    return MD_OK;
}

static cudaEvent_t prof_event(md_ctx *c)
{
    if (!c->ev_pool.empty()) { cudaEvent_t e = c->ev_pool.back(); c->ev_pool.pop_back(); return e; }
    cudaEvent_t e = nullptr;
    cudaEventCreate(&e);
    return e;
}

ProfScope::ProfScope(md_ctx *ctx, int kernel) : c(ctx), k(kernel)
{
    if (!c->profiling) return;
    if (c->profiling == 2) {
        if (kernel != MD_K_LJ && kernel != MD_K_DPD) return;
        // MD_OPT_PROFILE_STRIDE: every S-th pair-force launch is bracketed (the events of every launch cost a 30 us step of
        // 4,000 particles a third of its time)
        if (c->prof_stride > 1 && (c->prof_count++ % c->prof_stride) != 0) return;
    }
    e0 = prof_event(c);
    e1 = prof_event(c);
    cudaEventRecord(e0, c->stream);
}

ProfScope::~ProfScope()
{
    if (!e0) return;
    cudaEventRecord(e1, c->stream);
    c->ev_pending.push_back({k, e0, e1});
}

void prof_resolve(md_ctx *c)
{
    for (auto &p : c->ev_pending) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, p.e0, p.e1) == cudaSuccess) {
            c->stats.stage_ms[p.k] += ms;
            c->stats.stage_launches[p.k]++;
        } else cudaGetLastError();
        c->ev_pool.push_back(p.e0);
        c->ev_pool.push_back(p.e1);
    }
    c->ev_pending.clear();
}

// folds the event pairs that have completed (no synchronisation), keeps the rest pending
void prof_resolve_ready(md_ctx *c)
{
    size_t keep = 0;
    for (size_t i = 0; i < c->ev_pending.size(); ++i) {
        auto p = c->ev_pending[i];
        if (cudaEventQuery(p.e1) == cudaSuccess) {
            float ms = 0.f;
            if (cudaEventElapsedTime(&ms, p.e0, p.e1) == cudaSuccess) {
                c->stats.stage_ms[p.k] += ms;
                c->stats.stage_launches[p.k]++;
            } else cudaGetLastError();
            c->ev_pool.push_back(p.e0);
            c->ev_pool.push_back(p.e1);
        } else {
            cudaGetLastError();
            c->ev_pending[keep++] = p;
        }
    }
    c->ev_pending.resize(keep);
}

extern "C" int md_set_profiling(md_ctx *c, int on)
{
    if (!c) return MD_EINVAL;
    MD_TRY(md_sync(c));
    prof_resolve(c);
    c->profiling = on == 2 ? 2 : (on != 0 ? 1 : 0);
    for (int k = 0; k < MD_N_KERNELS; ++k) { c->stats.stage_ms[k] = 0.0; c->stats.stage_launches[k] = 0; }
    return MD_OK;
}

static bool is_device_ptr(const void *p)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

// bump allocator over a growable staging buffer for host-pointer arguments; reset at the start of each API call
struct Stage {
    md_ctx *c;
    uint64_t used = 0;
    explicit Stage(md_ctx *ctx) : c(ctx) {}
    int reserve(uint64_t bytes)
    {
        if (bytes <= c->stage_bytes) return MD_OK;
        MD_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
        if (c->stage) md_free(c, c->stage);
        c->stage_bytes = bytes + (bytes >> 3) + 4096;
        return md_alloc(c, &c->stage, c->stage_bytes);
    }
    void *take(uint64_t bytes)
    {
        void *p = (char *)c->stage + used;
        used += (bytes + 255) & ~255ull;
        return p;
    }
};

static uint64_t pad256(uint64_t b) { return (b + 255) & ~255ull; }

// input: returns a device pointer holding `bytes` of *src (copying if src is a host pointer)
static int stage_in(md_ctx *c, Stage &st, const void *src, uint64_t bytes, const void **dev)
{
    if (!src) { *dev = nullptr; return MD_OK; }
    if (is_device_ptr(src)) { *dev = src; return MD_OK; }
    void *d = st.take(bytes);
    MD_CUDA_CHECK(c, cudaMemcpyAsync(d, src, bytes, cudaMemcpyHostToDevice, c->stream));
    *dev = d;
    return MD_OK;
}

// output: device pointer the kernel writes to; finish_out copies back if dst is a host pointer
struct OutBuf { void *dst; void *dev; uint64_t bytes; bool host; };
static OutBuf stage_out(Stage &st, void *dst, uint64_t bytes)
{
    OutBuf o{dst, nullptr, bytes, false};
    if (!dst) return o;
    if (is_device_ptr(dst)) { o.dev = dst; return o; }
    o.dev = st.take(bytes);
    o.host = true;
    return o;
}
static int finish_out(md_ctx *c, const OutBuf &o)
{
    if (o.dst && o.host) MD_CUDA_CHECK(c, cudaMemcpyAsync(o.dst, o.dev, o.bytes, cudaMemcpyDeviceToHost, c->stream));
    return MD_OK;
}
static uint64_t stage_need(const void *p, uint64_t bytes) { return (p && !is_device_ptr(p)) ? pad256(bytes) : 0; }

// =====================================================================================================
// cell storage order (host): rank_of_lin for Morton / Hilbert curves over the cell grid
// =====================================================================================================
static uint64_t morton3(uint32_t x, uint32_t y, uint32_t z)
{
    auto spread = [](uint64_t v) {
        v &= 0x1fffff;
        v = (v | v << 32) & 0x1f00000000ffffull;
        v = (v | v << 16) & 0x1f0000ff0000ffull;
        v = (v | v << 8) & 0x100f00f00f00f00full;
        v = (v | v << 4) & 0x10c30c30c30c30c3ull;
        v = (v | v << 2) & 0x1249249249249249ull;
        return v;
    };
    return spread(x) | spread(y) << 1 | spread(z) << 2;
}

// Hilbert index of a 3-D point with `bits` bits per axis (Skilling, "Programming the Hilbert curve", 2004:
// axes -> transposed index, then interleave)
static uint64_t hilbert3(uint32_t x, uint32_t y, uint32_t z, int bits)
{
    uint32_t X[3] = {x, y, z};
    const uint32_t M = 1u << (bits - 1);
    for (uint32_t Q = M; Q > 1; Q >>= 1) {
        const uint32_t P = Q - 1;
        for (int i = 0; i < 3; ++i) {
            if (X[i] & Q) X[0] ^= P;
            else { const uint32_t t = (X[0] ^ X[i]) & P; X[0] ^= t; X[i] ^= t; }
        }
    }
    for (int i = 1; i < 3; ++i) X[i] ^= X[i - 1];
    uint32_t t = 0;
    for (uint32_t Q = M; Q > 1; Q >>= 1)
        if (X[2] & Q) t ^= Q - 1;
    for (int i = 0; i < 3; ++i) X[i] ^= t;
    uint64_t h = 0;
    for (int b = bits - 1; b >= 0; --b)
        for (int i = 0; i < 3; ++i) h = (h << 1) | ((X[i] >> b) & 1u);
    return h;
}

// grid of the cell-relative fp32 records (Geom::q0): every staged coordinate of a tile -- at most (B/2 + 1) cell widths +
// r_buff from the brick centre -- must be an exact float multiple of q0, i.e. stay below 2^24 q0
static void set_record_grid(md_ctx *c, uint32_t B)
{
    double E = 0.0;
    for (int a = 0; a < 3; ++a) E = std::max(E, (0.5 * B + 1.0) * c->g.cw[a] + c->r_buff + 1e-6);
    c->g.q0 = ldexp(1.0, ilogb(E) + 1 - 24);
    c->g.q0i = 1.0 / c->g.q0;
    c->g.qr = c->g.q0 / 512.0;  // a power of two: residual arithmetic in the near section is exact (lj3_near)
    c->g.qri = 512.0 / c->g.q0;
}

static uint32_t choose_brick(md_ctx *c)
{
    if (c->tile_B_forced) return (uint32_t)c->tile_B_forced;
    const double ppc = (double)c->N / (double)c->n_cells;
    // aim at a few hundred home particles per tile, but keep at least ~2 tiles per SM
    uint32_t B = ppc >= 48.0 ? 1u : (ppc >= 4.0 ? 2u : 4u);
    while (B > 1 && (double)c->n_cells / (double)(B * B * B) < 300.0) B >>= 1;
    return B;
}

int build_cell_order(md_ctx *c)
{
    c->tile_desc_valid = false;
    for (uint32_t **p : {&c->rank_of_lin, &c->lin_of_rank, &c->tile_cell_begin, &c->tile_origin})
        if (*p) { md_free(c, *p); *p = nullptr; }
    c->use_tiles = false;
    c->n_tiles = 0;
    set_record_grid(c, c->order == MD_ORDER_MORTON ? choose_brick(c) : 1u);
    if (c->order == MD_ORDER_LEX) return MD_OK;
    const uint32_t nx = c->dims[0], ny = c->dims[1], nz = c->dims[2];
    int bits = 1;
    while ((1u << bits) < std::max(nx, std::max(ny, nz))) ++bits;
    std::vector<std::pair<uint64_t, uint32_t>> keys(c->n_cells);
    for (uint32_t z = 0; z < nz; ++z)
        for (uint32_t y = 0; y < ny; ++y)
            for (uint32_t x = 0; x < nx; ++x) {
                const uint32_t lin = x + nx * (y + ny * z);
                keys[lin] = {c->order == MD_ORDER_MORTON ? morton3(x, y, z) : hilbert3(x, y, z, bits), lin};
            }
    std::sort(keys.begin(), keys.end());
    std::vector<uint32_t> rank(c->n_cells), lin_of_rank(c->n_cells);
    for (uint32_t r = 0; r < c->n_cells; ++r) { rank[keys[r].second] = r; lin_of_rank[r] = keys[r].second; }
    MD_TRY(md_alloc(c, (void **)&c->rank_of_lin, sizeof(uint32_t) * c->n_cells));
    MD_CUDA_CHECK(c, cudaMemcpy(c->rank_of_lin, rank.data(), sizeof(uint32_t) * c->n_cells, cudaMemcpyHostToDevice));
    if (c->order != MD_ORDER_MORTON) return MD_OK;

    // tiles: bricks of B^3 cells = runs of equal (Morton key >> 3 log2 B), contiguous in rank order
    const uint32_t B = choose_brick(c);
    int lb = 0;
    while ((1u << lb) < B) ++lb;
    std::vector<uint32_t> begin, origin;
    uint64_t prev = ~0ull;
    for (uint32_t r = 0; r < c->n_cells; ++r) {
        const uint64_t brick = keys[r].first >> (3 * lb);
        if (brick != prev) {
            prev = brick;
            begin.push_back(r);
            const uint32_t lin = keys[r].second;
            const uint32_t x = lin % nx, y = (lin / nx) % ny, z = lin / (nx * ny);
            origin.push_back((x >> lb) << lb);
            origin.push_back((y >> lb) << lb);
            origin.push_back((z >> lb) << lb);
        }
    }
    c->n_tiles = (uint32_t)begin.size();
    begin.push_back(c->n_cells);
    c->tile_B = B;
    MD_TRY(md_alloc(c, (void **)&c->lin_of_rank, sizeof(uint32_t) * c->n_cells));
    MD_TRY(md_alloc(c, (void **)&c->tile_cell_begin, sizeof(uint32_t) * begin.size()));
    MD_TRY(md_alloc(c, (void **)&c->tile_origin, sizeof(uint32_t) * origin.size()));
    MD_CUDA_CHECK(c, cudaMemcpy(c->lin_of_rank, lin_of_rank.data(), sizeof(uint32_t) * c->n_cells, cudaMemcpyHostToDevice));
    MD_CUDA_CHECK(c, cudaMemcpy(c->tile_cell_begin, begin.data(), sizeof(uint32_t) * begin.size(), cudaMemcpyHostToDevice));
    MD_CUDA_CHECK(c, cudaMemcpy(c->tile_origin, origin.data(), sizeof(uint32_t) * origin.size(), cudaMemcpyHostToDevice));
    c->use_tiles = true;
    return MD_OK;
}

// =====================================================================================================
// lifetime
// =====================================================================================================
// cell grid and geometry record of a skin r_buff (md_create; md_tune_rbuff changes it on a live context)
static int set_geometry(md_ctx *c, double r_buff)
{
    const double r_list = c->rc + r_buff;
    uint64_t ncell = 1;
    uint32_t dims[3];
    for (int a = 0; a < 3; ++a) {
        const double n = floor(c->box[a] / r_list);
        if (!(c->box[a] > 0.0) || n < 3.0 || n > 2097151.0) {
            c->err = "box too small for the 27-cell stencil (need floor(L/(rc+r_buff)) >= 3 per axis)";
            return MD_EINVAL;
        }
        dims[a] = (uint32_t)n;
        ncell *= dims[a];
    }
    if (ncell >= 0xfffffff0ull) { c->err = "too many cells"; return MD_EINVAL; }
    c->r_buff = r_buff;
    c->r_list = r_list;
    for (int a = 0; a < 3; ++a) {
        c->dims[a] = dims[a];
        c->g.L[a] = c->box[a];
        c->g.h[a] = 0.5 * c->box[a];
        c->g.lo[a] = -0.5 * c->box[a];
        c->g.n[a] = dims[a];
        c->g.dn[a] = (double)dims[a];
        c->g.cw[a] = c->box[a] / (double)dims[a];
    }
    c->n_cells = (uint32_t)ncell;
    c->g.n_cells = c->n_cells;
    c->g.N = (uint32_t)c->N;
    set_record_grid(c, 1);
    return MD_OK;
}

static void set_default_cfg(md_ctx *c)
{
    for (int k = 0; k < MD_N_KERNELS; ++k) c->cfg[k] = LaunchCfg{128, 1, 0.f};
    c->cfg[MD_K_NLIST] = LaunchCfg{256, 4, 0.f};
    c->cfg[MD_K_LJ] = LaunchCfg{256, 2, 0.f};
    c->cfg[MD_K_DPD] = LaunchCfg{128, 4, 0.f};
    c->cfg[MD_K_BONDS] = LaunchCfg{128, 1, 0.f};
    c->cfg[MD_K_INTEGRATE] = LaunchCfg{256, 1, 0.f};
    c->cfg[MD_K_CELLS] = LaunchCfg{256, 1, 0.f};
}

static thread_local std::string g_create_err;

// the per-particle and per-cell arrays: allocated at the first md_configure / md_set_state, so that md_set_workspace can
// come between md_create and them
static int alloc_state(md_ctx *c)
{
    if (c->state_allocated) return MD_OK;
    const uint64_t N = c->N;
    int s = MD_OK;
    auto A = [&](void **p, uint64_t bytes) { if (s == MD_OK) s = md_alloc(c, p, bytes); };
    A((void **)&c->pos, N * sizeof(double4));
    A((void **)&c->pos_alt, N * sizeof(double4));
    A((void **)&c->vel, N * sizeof(double4));
    A((void **)&c->vel_alt, N * sizeof(double4));
    A((void **)&c->force, N * sizeof(double4));
    A((void **)&c->force_alt, N * sizeof(double4));
    A((void **)&c->image, 3 * N * sizeof(int));
    A((void **)&c->image_alt, 3 * N * sizeof(int));
    A((void **)&c->pos_ref, 3 * N * sizeof(double));
    A((void **)&c->rel, N * sizeof(float4));
    A((void **)&c->nvt_state, 4 * sizeof(double));
    A((void **)&c->tag, N * sizeof(uint32_t));
    A((void **)&c->tag_alt, N * sizeof(uint32_t));
    A((void **)&c->rtag, N * sizeof(uint32_t));
    A((void **)&c->cell_lin, N * sizeof(uint32_t));
    A((void **)&c->cell_rank_tmp, N * sizeof(uint32_t));
    A((void **)&c->perm, N * sizeof(uint32_t));
    A((void **)&c->perm_sorted, N * sizeof(uint32_t));
    A((void **)&c->cell_count, (uint64_t)c->n_cells * sizeof(uint32_t));
    A((void **)&c->cell_start, ((uint64_t)c->n_cells + 1) * sizeof(uint32_t));
    A((void **)&c->nl_cnt, N * sizeof(uint32_t));
    A((void **)&c->nl_off, (N + 1) * sizeof(uint64_t));
    A((void **)&c->d_flags, sizeof(DevFlags));
    if (s == MD_OK && cudaMallocHost((void **)&c->h_flags, sizeof(DevFlags)) != cudaSuccess) { c->err = "cudaMallocHost failed"; s = MD_ENOMEM; }
    if (s == MD_OK && cudaMemset(c->d_flags, 0, sizeof(DevFlags)) != cudaSuccess) s = MD_ECUDA;
    if (s == MD_OK && cudaMemset(c->force, 0, N * sizeof(double4)) != cudaSuccess) s = MD_ECUDA;
    if (s != MD_OK) return s;
    c->state_allocated = true;
    return MD_OK;
}


extern "C" int md_create(md_ctx **out, const double box[3], uint64_t N, double rc, double r_buff)
{
    if (!out) return MD_EINVAL;
    *out = nullptr;
    if (!box || N == 0 || N >= 0xfffffff0ull || !(rc > 0.0) || !(r_buff >= 0.0)) { g_create_err = "md_create: bad argument"; return MD_EINVAL; }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        g_create_err = "md_create: no CUDA device (this library has no CPU fallback)";
        return MD_ECUDA;
    }
    md_ctx *c = new md_ctx();
    memset(&c->stats, 0, sizeof(c->stats));
    c->N = N;
    c->rc = rc;
    c->precision = MD_FP64;
    c->order = MD_ORDER_LEX;
    c->sched = MD_SCHED_BATCH;
    c->stream = 0;
    c->log = getenv("B200MD_LOG") != nullptr;
    for (int a = 0; a < 3; ++a) c->box[a] = box[a];
    if (set_geometry(c, r_buff) != MD_OK) { g_create_err = c->err; delete c; return MD_EINVAL; }
    set_default_cfg(c);

    *out = c;
    return MD_OK;
}

extern "C" int md_configure(md_ctx *c, int precision, void *stream, int order, int sched)
{
    if (!c) return MD_EINVAL;
    if ((precision != MD_FP64 && precision != MD_MIXED) || order < 0 || order > MD_ORDER_HILBERT ||
        (sched != MD_SCHED_SYNC && sched != MD_SCHED_SPECULATIVE && sched != MD_SCHED_BATCH)) {
        c->err = "md_configure: bad argument";
        return MD_EINVAL;
    }
    MD_TRY(alloc_state(c));
    c->precision = precision;
    c->stream = (cudaStream_t)stream;
    c->sched = sched;
    if (order != c->order || (order != MD_ORDER_LEX && !c->rank_of_lin)) {
        c->order = order;
        MD_TRY(build_cell_order(c));
        c->cells_valid = c->nlist_valid = false;
    }
    return MD_OK;
}

// ---- caller-provided device memory ("PyTorch used only for device memory and streams") ---------------
extern "C" int md_set_workspace(md_ctx *c, void *workspace, uint64_t bytes)
{
    if (!c) return MD_EINVAL;
    if (c->state_allocated || c->device_bytes) { c->err = "md_set_workspace: call it right after md_create (device memory is already allocated)"; return MD_ESTATE; }
    if (!workspace || bytes < 4096 || !is_device_ptr(workspace)) { c->err = "md_set_workspace: a device pointer and its size are required"; return MD_EINVAL; }
    const uint64_t skew = (256 - ((uintptr_t)workspace & 255)) & 255;  // blocks are 256-byte aligned
    c->ws_base = (char *)workspace + skew;
    c->ws_bytes = (bytes - skew) & ~255ull;
    c->ws_blocks.assign(1, md_ctx::WsBlock{0, c->ws_bytes, false});
    c->ws_peak = 0;
    return MD_OK;
}

extern "C" int md_workspace_bytes(const double box[3], uint64_t N, double rc, double r_buff, int precision, uint64_t *bytes)
{
    if (!box || !bytes || N == 0 || !(rc > 0.0) || !(r_buff >= 0.0)) return MD_EINVAL;
    (void)precision;  // both modes keep the same arrays (the fp32 records exist in fp64 mode too)
    const double r_list = rc + r_buff;
    double ncell = 1.0, vol = 1.0;
    for (int a = 0; a < 3; ++a) {
        const double n = floor(box[a] / r_list);
        if (!(box[a] > 0.0) || n < 3.0) return MD_EINVAL;
        ncell *= n;
        vol *= box[a];
    }
    const double n = (double)N;
    const double nbar = n / vol * 4.18879020478639 * r_list * r_list * r_list;  // mean neighbours per particle
    double b = 0.0;
    b += n * (6 * 32 + 2 * 12 + 24 + 16 + 7 * 4 + 4 + 8);           // state, twins, records, tags, permutations, row lengths, offsets
    b += ncell * (4 * 4 + 320.0) + 65536.0;                          // cell tables, curve tables, per-tile headers
    b += (n + 1.0) * (1.5 * (1.35 * nbar + 24.0) + 32.0) * 2.0;      // 16-bit rows at the density-based stride, grown once by 1.5
    b += n * 4.0 + n * (nbar + 4.0) * 4.0 * 1.125 + 4096.0;          // the exact 32-bit list (general path; exports of a tile list)
    b += n * (4.0 + 8.0) + n * 20.0;                                 // export scratch; bond table for up to 2 bonds per particle
    b += 2.0 * 3.0 * 8.0 * n * 1.125 + 65536.0;                      // staging of host-pointer state arguments ...
    b += n * (nbar + 4.0) * 4.0 * 1.125;                             // ... or of an exported pair list (8 bytes per pair)
    b += 64.0 * 256.0 + 1048576.0;                                   // block rounding, small tables
    b *= 1.10;                                                       // first-fit fragmentation
    *bytes = (uint64_t)b;
    return MD_OK;
}

extern "C" int md_destroy(md_ctx *c)
{
    if (!c) return MD_EINVAL;
    cudaStreamSynchronize(c->stream);
    prof_resolve(c);
    for (cudaEvent_t e : c->ev_pool) cudaEventDestroy(e);
    for (auto &p : c->allocs) cudaFree(p.first);
    if (c->ev_flags) cudaEventDestroy(c->ev_flags);
    if (c->h_flags) cudaFreeHost(c->h_flags);
    cudaGetLastError();
    delete c;
    return MD_OK;
}

extern "C" const char *md_last_error(md_ctx *c) { return c ? c->err.c_str() : g_create_err.c_str(); }

// =====================================================================================================
// state
// =====================================================================================================
extern "C" int md_set_state(md_ctx *c, const double *pos, const double *vel, const double *mass, uint64_t step0)
{
    if (!c || !pos || !vel) { if (c) c->err = "md_set_state: pos and vel are required"; return MD_EINVAL; }
    MD_TRY(alloc_state(c));
    const uint64_t b3 = 3 * c->N * sizeof(double), b1 = c->N * sizeof(double);
    Stage st(c);
    MD_TRY(st.reserve(stage_need(pos, b3) + stage_need(vel, b3) + stage_need(mass, b1)));
    const void *dp, *dv, *dm;
    MD_TRY(stage_in(c, st, pos, b3, &dp));
    MD_TRY(stage_in(c, st, vel, b3, &dv));
    MD_TRY(stage_in(c, st, mass, b1, &dm));
    MD_TRY(launch_pack_state(c, (const double *)dp, (const double *)dv, (const double *)dm));
    MD_CUDA_CHECK(c, cudaMemsetAsync(c->nvt_state, 0, 4 * sizeof(double), c->stream));  // thermostat at rest (R30)
    MD_CUDA_CHECK(c, cudaMemsetAsync(c->force, 0, c->N * sizeof(double4), c->stream));
    MD_CUDA_CHECK(c, cudaMemsetAsync(c->d_flags, 0, sizeof(DevFlags), c->stream));
    c->have_state = true;
    c->cells_valid = c->nlist_valid = c->force_valid = false;
    c->step = step0;
    return MD_OK;
}

extern "C" int md_set_bonds(md_ctx *c, const uint32_t *ta, const uint32_t *tb, uint64_t nb)
{
    if (!c) return MD_EINVAL;
    if (nb > 0 && (!ta || !tb)) { c->err = "md_set_bonds: null tag array"; return MD_EINVAL; }
    if (nb >= 0x7fffffffull) { c->err = "md_set_bonds: too many bonds"; return MD_EINVAL; }
    MD_TRY(alloc_state(c));
    MD_TRY(md_sync(c));
    if (c->bond_off) { md_free(c, c->bond_off); c->bond_off = nullptr; }
    if (c->bond_partner) { md_free(c, c->bond_partner); c->bond_partner = nullptr; }
    c->n_bonds = nb;
    if (nb == 0) return MD_OK;
    MD_TRY(md_alloc(c, (void **)&c->bond_off, (c->N + 1) * sizeof(uint32_t)));
    MD_TRY(md_alloc(c, (void **)&c->bond_partner, 2 * nb * sizeof(uint32_t)));
    Stage st(c);
    const uint64_t bb = nb * sizeof(uint32_t);
    MD_TRY(st.reserve(stage_need(ta, bb) + stage_need(tb, bb)));
    const void *da, *db;
    MD_TRY(stage_in(c, st, ta, bb, &da));
    MD_TRY(stage_in(c, st, tb, bb, &db));
    // validate on the host side when the caller gave host pointers (cheap); device pointers are trusted
    if (!is_device_ptr(ta))
        for (uint64_t m = 0; m < nb; ++m)
            if (ta[m] >= c->N || tb[m] >= c->N || ta[m] == tb[m]) { c->err = "md_set_bonds: tag out of range or self bond"; c->n_bonds = 0; return MD_EINVAL; }
    MD_TRY(launch_bonds_build(c, (const uint32_t *)da, (const uint32_t *)db, nb));
    return md_sync(c);
}

extern "C" int md_get_state(md_ctx *c, double *pos, double *vel, int32_t *image)
{
    if (!c) return MD_EINVAL;
    if (!c->have_state) { c->err = "md_get_state: no state"; return MD_ESTATE; }
    const uint64_t b3 = 3 * c->N * sizeof(double), bi = 3 * c->N * sizeof(int32_t);
    Stage st(c);
    MD_TRY(st.reserve(stage_need(pos, b3) + stage_need(vel, b3) + stage_need(image, bi)));
    OutBuf op = stage_out(st, pos, b3), ov = stage_out(st, vel, b3), oi = stage_out(st, image, bi);
    MD_TRY(launch_unpack_state(c, (double *)op.dev, (double *)ov.dev, (int32_t *)oi.dev));
    MD_TRY(finish_out(c, op));
    MD_TRY(finish_out(c, ov));
    MD_TRY(finish_out(c, oi));
    if (op.host || ov.host || oi.host) MD_TRY(md_sync(c));
    return MD_OK;
}

static int eval_forces(md_ctx *c, const md_step_desc *w, uint64_t step, bool energy);

// md_step evaluates LJ forces without the per-particle energies.  When they are asked for, the same evaluation is
// repeated with the energy lane switched on INTO THE SCRATCH TWIN of the force array and only the energy lane is copied
// over: the forces that the next half-kick uses stay those of the step's own kernel, whether or not energies were read.
static int energies_on_demand(md_ctx *c)
{
    std::swap(c->force, c->force_alt);
    const int s = eval_forces(c, &c->last_desc, c->last_force_step, true);
    std::swap(c->force, c->force_alt);
    MD_TRY(s);
    MD_TRY(launch_copy_energy(c, c->force_alt));
    c->energy_valid = true;
    return MD_OK;
}

extern "C" int md_get_forces(md_ctx *c, double *force, double *energy)
{
    if (!c) return MD_EINVAL;
    if (!c->force_valid) { c->err = "md_get_forces: no force has been computed for the current positions"; return MD_ESTATE; }
    // md_step evaluates LJ forces without the per-particle energies; the forces are a pure function of the current
    // state, so the same evaluation is repeated with the energy lane switched on when it is asked for
    if (energy && !c->energy_valid && c->last_from_step) MD_TRY(energies_on_demand(c));
    const uint64_t b3 = 3 * c->N * sizeof(double), b1 = c->N * sizeof(double);
    Stage st(c);
    MD_TRY(st.reserve(stage_need(force, b3) + stage_need(energy, b1)));
    OutBuf of = stage_out(st, force, b3), oe = stage_out(st, energy, b1);
    MD_TRY(launch_unpack_forces(c, (double *)of.dev, (double *)oe.dev));
    MD_TRY(finish_out(c, of));
    MD_TRY(finish_out(c, oe));
    if (of.host || oe.host) MD_TRY(md_sync(c));
    return MD_OK;
}

// =====================================================================================================
// S1 / S2
// =====================================================================================================
static int do_build_cells(md_ctx *c)
{
    ProfScope ps(c, MD_K_CELLS);
    MD_TRY(launch_build_cells(c));
    c->tile_desc_valid = false;  // the per-tile header tables follow cell_start
    c->cells_valid = true;
    c->nlist_valid = false;
    c->steps_since_build = 0;
    c->last_d2 = 0.f;
    MD_CUDA_CHECK(c, cudaMemsetAsync(&c->d_flags->rebuild, 0, 2 * sizeof(int), c->stream));
    return MD_OK;
}

extern "C" int md_build_cells(md_ctx *c)
{
    if (!c) return MD_EINVAL;
    if (!c->have_state) { c->err = "md_build_cells: md_set_state first"; return MD_ESTATE; }
    return do_build_cells(c);
}

extern "C" int md_get_cells(md_ctx *c, uint32_t *cell_of, uint32_t dims[3])
{
    if (!c) return MD_EINVAL;
    if (dims) for (int a = 0; a < 3; ++a) dims[a] = c->dims[a];
    if (!cell_of) return MD_OK;
    if (!c->cells_valid) { c->err = "md_get_cells: md_build_cells first"; return MD_ESTATE; }
    const uint64_t b = c->N * sizeof(uint32_t);
    Stage st(c);
    MD_TRY(st.reserve(stage_need(cell_of, b)));
    OutBuf o = stage_out(st, cell_of, b);
    MD_TRY(launch_unpack_cells(c, (uint32_t *)o.dev));
    MD_TRY(finish_out(c, o));
    if (o.host) MD_TRY(md_sync(c));
    return MD_OK;
}

static int ensure_nl32(md_ctx *c, uint64_t total)
{
    if (total > c->nl_capacity) {
        if (c->nl_idx) { md_free(c, c->nl_idx); c->nl_idx = nullptr; }
        const uint64_t cap = total + total / 8 + 1024;
        c->nl_capacity = 0;
        MD_TRY(md_alloc(c, (void **)&c->nl_idx, cap * sizeof(uint32_t)));
        c->nl_capacity = cap;
    }
    return MD_OK;
}

static int build_nlist_general(md_ctx *c)
{
    MD_TRY(launch_nlist_count(c));
    MD_TRY(launch_exclusive_scan_u32(c, c->nl_cnt, c->N, nullptr, c->nl_off, true, &c->d_flags->nl_total));
    MD_TRY(md_read_flags(c));
    const uint64_t total = c->h_flags->nl_total;
    MD_TRY(ensure_nl32(c, total));
    c->nl_entries = total;
    MD_TRY(launch_nlist_fill(c));
    c->nl_is_tile = false;
    return MD_OK;
}

static uint32_t round16(double x) { return (uint32_t)((uint64_t)(x + 15.0) / 16 * 16); }

static int build_nlist_tiles(md_ctx *c, bool *done)
{
    *done = false;
    MD_TRY(tile_measure(c));
    MD_TRY(md_read_flags(c));
    c->tile_max_home = c->h_flags->max_home;
    c->tile_max_staged = c->h_flags->max_staged;
    if (c->nl_stride == 0) {
        // row stride from the mean density: 1.35 n + 24 covers the fluctuations of liquids and ideal gases at the
        // configured densities; a longer row is detected by the build kernel and the stride grows
        const double vol = c->box[0] * c->box[1] * c->box[2];
        const double rho = (double)c->N / vol;
        const double nbar = rho * 4.18879020478639 * c->r_list * c->r_list * c->r_list;
        if (c->nl16) { md_free(c, c->nl16); c->nl16 = nullptr; }
        c->nl_stride = round16(1.35 * nbar + 24.0);
    }
    for (int attempt = 0; attempt < 3; ++attempt) {
        if (!c->nl16) MD_TRY(md_alloc(c, (void **)&c->nl16, (c->N + 1) * (uint64_t)c->nl_stride * sizeof(uint16_t)));  // + one row: the force kernels
                                                                                      // request block `lane` of a row before they know its length
        bool fits = false;
        MD_TRY(launch_tile_build(c, &fits));
        if (!fits) return MD_OK;  // largest tile exceeds shared memory: general path
        MD_TRY(md_read_flags(c));
        if (c->h_flags->nl_overflow == 0) {
            c->nl_entries = c->h_flags->nl_total;
            c->nl_is_tile = true;
            c->nl32_decoded = false;
            *done = true;
            return MD_OK;
        }
        md_free(c, c->nl16);
        c->nl16 = nullptr;
        c->nl_stride = round16(1.25 * c->h_flags->nl_overflow + 16.0);
        if (c->log) fprintf(stderr, "[b200md] neighbour row stride grows to %u entries\n", c->nl_stride);
    }
    c->err = "neighbour list: row stride still too small after growing";
    return MD_ECUDA;
}

static int do_build_nlist(md_ctx *c)
{
    ProfScope ps(c, MD_K_NLIST);
    bool done = false;
    if (c->use_tiles) MD_TRY(build_nlist_tiles(c, &done));
    if (!done) MD_TRY(build_nlist_general(c));
    c->nlist_valid = true;
    c->stats.rebuilds++;
    c->stats.max_cell_count = c->h_flags->max_cell_count;
    return MD_OK;
}

// exports read the general 32-bit CSR; a tile list is decoded into it on demand (exact filter, see tiles.cu)
static int ensure_decoded(md_ctx *c)
{
    if (!c->nl_is_tile) { c->nl_cnt_exp = c->nl_cnt; return MD_OK; }
    if (c->nl32_decoded) return MD_OK;
    if (!c->nl_cnt32) MD_TRY(md_alloc(c, (void **)&c->nl_cnt32, c->N * sizeof(uint32_t)));
    MD_TRY(launch_tile_decode(c, false, c->nl_cnt32));
    MD_TRY(launch_exclusive_scan_u32(c, c->nl_cnt32, c->N, nullptr, c->nl_off, false, &c->d_flags->nl_total));
    MD_TRY(md_read_flags(c));
    c->nl_exact_entries = c->h_flags->nl_total;
    MD_TRY(ensure_nl32(c, c->h_flags->nl_total));
    MD_TRY(launch_tile_decode(c, true, nullptr));
    c->nl_cnt_exp = c->nl_cnt32;
    c->nl32_decoded = true;
    return MD_OK;
}

extern "C" int md_build_nlist(md_ctx *c)
{
    if (!c) return MD_EINVAL;
    if (!c->have_state) { c->err = "md_build_nlist: md_set_state first"; return MD_ESTATE; }
    // bins taken before an integration step are stale: the list kernels assume positions as binned (image shifts per
    // cell, cell-relative records), so the binning is repeated whenever half 1 has run since
    if (!c->cells_valid || c->steps_since_build > 0) MD_TRY(do_build_cells(c));
    return do_build_nlist(c);
}

extern "C" int md_get_nlist(md_ctx *c, uint64_t *n_pairs, uint32_t *pairs, uint64_t cap)
{
    if (!c || !n_pairs) return MD_EINVAL;
    if (!c->nlist_valid) { c->err = "md_get_nlist: md_build_nlist first"; return MD_ESTATE; }
    MD_TRY(ensure_decoded(c));
    uint32_t *cnt = nullptr;
    uint64_t *off = nullptr;
    MD_TRY(md_alloc(c, (void **)&cnt, c->N * sizeof(uint32_t)));
    MD_TRY(md_alloc(c, (void **)&off, (c->N + 1) * sizeof(uint64_t)));
    int s = launch_export_pairs_count(c, cnt);
    if (s == MD_OK) s = launch_exclusive_scan_u32(c, cnt, c->N, nullptr, off, false, &c->d_flags->nl_total);
    if (s == MD_OK) s = md_read_flags(c);
    const uint64_t total = c->h_flags->nl_total;
    if (s == MD_OK) *n_pairs = total;
    if (s == MD_OK && pairs) {
        if (cap < total) { c->err = "md_get_nlist: cap too small"; s = MD_EINVAL; }
        else {
            const uint64_t b = 2 * total * sizeof(uint32_t);
            Stage st(c);
            s = st.reserve(stage_need(pairs, b));
            if (s == MD_OK) {
                OutBuf o = stage_out(st, pairs, b);
                s = launch_export_pairs_fill(c, off, (uint32_t *)o.dev);
                if (s == MD_OK) s = finish_out(c, o);
            }
        }
    }
    if (s == MD_OK) s = md_sync(c); else cudaStreamSynchronize(c->stream);
    md_free(c, cnt);
    md_free(c, off);
    return s;
}

extern "C" int md_get_nlist_rows(md_ctx *c, const uint32_t *probe_tags, uint32_t n_probe, uint32_t *counts,
                                 uint32_t *nbr_tags, uint32_t row_stride)
{
    if (!c || !probe_tags || !counts || (!nbr_tags && row_stride)) return MD_EINVAL;
    if (!c->nlist_valid) { c->err = "md_get_nlist_rows: md_build_nlist first"; return MD_ESTATE; }
    MD_TRY(ensure_decoded(c));
    const uint64_t bp = (uint64_t)n_probe * sizeof(uint32_t), bn = (uint64_t)n_probe * row_stride * sizeof(uint32_t);
    Stage st(c);
    MD_TRY(st.reserve(stage_need(probe_tags, bp) + stage_need(counts, bp) + stage_need(nbr_tags, bn)));
    const void *dp;
    MD_TRY(stage_in(c, st, probe_tags, bp, &dp));
    OutBuf oc = stage_out(st, counts, bp), on = stage_out(st, nbr_tags, bn);
    if (on.dev) MD_CUDA_CHECK(c, cudaMemsetAsync(on.dev, 0xff, bn, c->stream));
    MD_TRY(launch_export_rows(c, (const uint32_t *)dp, n_probe, (uint32_t *)oc.dev, (uint32_t *)on.dev, row_stride));
    MD_TRY(finish_out(c, oc));
    MD_TRY(finish_out(c, on));
    if (oc.host || on.host) MD_TRY(md_sync(c));
    return MD_OK;
}

// =====================================================================================================
// S4 / S5 / S6 single calls
// =====================================================================================================
// pair kernels: tile path when the current list is a tile list, else the general list kernels
static int ensure_decoded(md_ctx *c);
static int pair_lj(md_ctx *c, double eps, double sigma, int shift, bool energy)
{
    // a tile list whose largest tile fits the build kernel but not this force kernel's records goes through the decoded list
    if (c->nl_is_tile && tile_forces_fit(c, false))
        return launch_tile_lj(c, eps, sigma, shift, energy);
    MD_TRY(ensure_decoded(c));
    return launch_forces_lj(c, eps, sigma, shift);
}
static int pair_dpd(md_ctx *c, double A, double gamma, double kT, double dt, uint64_t step, uint64_t seed)
{
    if (c->nl_is_tile && tile_forces_fit(c, true)) return launch_tile_dpd(c, A, gamma, kT, dt, step, seed);
    MD_TRY(ensure_decoded(c));
    return launch_forces_dpd(c, A, gamma, kT, dt, step, seed);
}

static int need_nlist(md_ctx *c, const char *who)
{
    if (!c->nlist_valid) { c->err = std::string(who) + ": no valid neighbour list (md_build_nlist first)"; return MD_ESTATE; }
    return MD_OK;
}

extern "C" int md_forces_lj(md_ctx *c, double eps, double sigma, int shift)
{
    if (!c) return MD_EINVAL;
    MD_TRY(need_nlist(c, "md_forces_lj"));
    c->lj_sigma_hint = sigma;
    ProfScope ps(c, MD_K_LJ);
    MD_TRY(pair_lj(c, eps, sigma, shift, true));
    c->force_valid = c->energy_valid = true;
    c->last_from_step = false;
    return MD_OK;
}

extern "C" int md_forces_dpd(md_ctx *c, double A, double gamma, double kT, double dt, uint64_t step, uint64_t seed)
{
    if (!c) return MD_EINVAL;
    if (!(dt > 0.0)) { c->err = "md_forces_dpd: dt must be positive"; return MD_EINVAL; }
    MD_TRY(need_nlist(c, "md_forces_dpd"));
    ProfScope ps(c, MD_K_DPD);
    MD_TRY(pair_dpd(c, A, gamma, kT, dt, step, seed));
    c->force_valid = c->energy_valid = true;
    c->last_from_step = false;
    return MD_OK;
}

extern "C" int md_forces_bonds(md_ctx *c, double k, double r0)
{
    if (!c) return MD_EINVAL;
    if (!c->have_state) { c->err = "md_forces_bonds: md_set_state first"; return MD_ESTATE; }
    if (c->n_bonds == 0) { c->force_valid = true; return MD_OK; }
    ProfScope ps(c, MD_K_BONDS);
    MD_TRY(launch_forces_bonds(c, k, r0));
    c->force_valid = true;
    return MD_OK;
}

extern "C" int md_forces_fene(md_ctx *c, double k, double r0)
{
    if (!c) return MD_EINVAL;
    if (!c->have_state) { c->err = "md_forces_fene: md_set_state first"; return MD_ESTATE; }
    if (c->n_bonds == 0) { c->force_valid = true; return MD_OK; }
    ProfScope ps(c, MD_K_BONDS);
    MD_TRY(launch_forces_bonds(c, k, r0, MD_BOND_FENE));
    c->force_valid = true;
    return MD_OK;
}

extern "C" int md_set_bond_table(md_ctx *c, double r_min, double r_max, const double *U, const double *F, uint64_t m)
{
    if (!c) return MD_EINVAL;
    MD_TRY(alloc_state(c));
    MD_TRY(md_sync(c));
    if (c->btab_uf) { md_free(c, c->btab_uf); c->btab_uf = nullptr; }
    c->btab_m = 0;
    if (m == 0) return MD_OK;
    if (!U || !F || m < 2 || m >= 0x7fffffffull || !(r_min >= 0.0) || !(r_min < r_max)) {
        c->err = "md_set_bond_table: need U, F, 2 <= m < 2^31 and 0 <= r_min < r_max";
        return MD_EINVAL;
    }
    MD_TRY(md_alloc(c, (void **)&c->btab_uf, 2 * m * sizeof(double)));
    Stage st(c);
    const uint64_t bb = m * sizeof(double);
    MD_TRY(st.reserve(stage_need(U, bb) + stage_need(F, bb)));
    const void *du, *df;
    MD_TRY(stage_in(c, st, U, bb, &du));
    MD_TRY(stage_in(c, st, F, bb, &df));
    MD_TRY(launch_table_pack(c, (const double *)du, (const double *)df, (uint32_t)m, c->btab_uf));
    c->btab_m = (uint32_t)m;
    c->btab_rmin = r_min;
    c->btab_rmax = r_max;
    return md_sync(c);
}

extern "C" int md_forces_bond_table(md_ctx *c)
{
    if (!c) return MD_EINVAL;
    if (!c->have_state) { c->err = "md_forces_bond_table: md_set_state first"; return MD_ESTATE; }
    if (c->btab_m == 0) { c->err = "md_forces_bond_table: md_set_bond_table first"; return MD_ESTATE; }
    if (c->n_bonds == 0) { c->force_valid = true; return MD_OK; }
    ProfScope ps(c, MD_K_BONDS);
    MD_TRY(launch_forces_bonds(c, 0.0, 0.0, MD_BOND_TABLE));
    c->force_valid = true;
    return MD_OK;
}

extern "C" int md_set_pair_table(md_ctx *c, double r_min, double r_max, const double *U, const double *F, uint64_t m)
{
    if (!c) return MD_EINVAL;
    MD_TRY(alloc_state(c));
    MD_TRY(md_sync(c));
    if (c->tab_uf) { md_free(c, c->tab_uf); c->tab_uf = nullptr; }
    c->tab_m = 0;
    if (m == 0) return MD_OK;
    if (!U || !F || m < 2 || m >= 0x7fffffffull || !(r_min >= 0.0) || !(r_min < r_max) || !(r_max <= c->rc)) {
        c->err = "md_set_pair_table: need U, F, 2 <= m < 2^31 and 0 <= r_min < r_max <= r_cut";
        return MD_EINVAL;
    }
    MD_TRY(md_alloc(c, (void **)&c->tab_uf, 2 * m * sizeof(double)));
    Stage st(c);
    const uint64_t bb = m * sizeof(double);
    MD_TRY(st.reserve(stage_need(U, bb) + stage_need(F, bb)));
    const void *du, *df;
    MD_TRY(stage_in(c, st, U, bb, &du));
    MD_TRY(stage_in(c, st, F, bb, &df));
    MD_TRY(launch_table_pack(c, (const double *)du, (const double *)df, (uint32_t)m, c->tab_uf));
    c->tab_m = (uint32_t)m;
    c->tab_rmin = r_min;
    c->tab_rmax = r_max;
    return md_sync(c);
}

extern "C" int md_forces_pair(md_ctx *c, int kind, const double p[4], int shift)
{
    if (!c || (!p && kind != MD_PAIR_TABLE) || kind < MD_PAIR_LJ || kind > MD_PAIR_TABLE) { if (c) c->err = "md_forces_pair: bad argument"; return MD_EINVAL; }
    if (kind == MD_PAIR_TABLE && c->tab_m == 0) { c->err = "md_forces_pair: md_set_pair_table first"; return MD_ESTATE; }
    MD_TRY(need_nlist(c, "md_forces_pair"));
    ProfScope ps(c, MD_K_LJ);
    MD_TRY(ensure_decoded(c));
    MD_TRY(launch_forces_pair(c, kind, p, shift));
    c->force_valid = c->energy_valid = true;
    c->last_from_step = false;
    return MD_OK;
}

extern "C" int md_set_angles(md_ctx *c, const uint32_t *ta, const uint32_t *tb, const uint32_t *tc, uint64_t na)
{
    if (!c) return MD_EINVAL;
    if (na > 0 && (!ta || !tb || !tc)) { c->err = "md_set_angles: null tag array"; return MD_EINVAL; }
    if (na >= 0x3fffffffull) { c->err = "md_set_angles: too many angles"; return MD_EINVAL; }
    MD_TRY(alloc_state(c));
    MD_TRY(md_sync(c));
    for (uint32_t **q : {&c->angle_off, &c->angle_ent, &c->angle_abc})
        if (*q) { md_free(c, *q); *q = nullptr; }
    c->n_angles = na;
    if (na == 0) return MD_OK;
    if (!is_device_ptr(ta))
        for (uint64_t m = 0; m < na; ++m)
            if (ta[m] >= c->N || tb[m] >= c->N || tc[m] >= c->N || ta[m] == tb[m] || tb[m] == tc[m] || ta[m] == tc[m]) {
                c->err = "md_set_angles: tag out of range or repeated in a triplet";
                c->n_angles = 0;
                return MD_EINVAL;
            }
    MD_TRY(md_alloc(c, (void **)&c->angle_off, (c->N + 1) * sizeof(uint32_t)));
    MD_TRY(md_alloc(c, (void **)&c->angle_ent, 3 * na * sizeof(uint32_t)));
    MD_TRY(md_alloc(c, (void **)&c->angle_abc, 3 * na * sizeof(uint32_t)));
    Stage st(c);
    const uint64_t bb = na * sizeof(uint32_t);
    MD_TRY(st.reserve(stage_need(ta, bb) + stage_need(tb, bb) + stage_need(tc, bb)));
    const void *da, *db, *dc;
    MD_TRY(stage_in(c, st, ta, bb, &da));
    MD_TRY(stage_in(c, st, tb, bb, &db));
    MD_TRY(stage_in(c, st, tc, bb, &dc));
    MD_TRY(launch_angles_build(c, (const uint32_t *)da, (const uint32_t *)db, (const uint32_t *)dc, na));
    return md_sync(c);
}

extern "C" int md_forces_angles(md_ctx *c, double k, double theta0)
{
    if (!c) return MD_EINVAL;
    if (!c->have_state) { c->err = "md_forces_angles: md_set_state first"; return MD_ESTATE; }
    if (c->n_angles == 0) { c->force_valid = true; return MD_OK; }
    ProfScope ps(c, MD_K_BONDS);
    MD_TRY(launch_forces_angles(c, k, theta0));
    c->force_valid = true;
    return MD_OK;
}

extern "C" int md_set_dihedrals(md_ctx *c, const uint32_t *ta, const uint32_t *tb, const uint32_t *tc, const uint32_t *td,
                                uint64_t nd)
{
    if (!c) return MD_EINVAL;
    if (nd > 0 && (!ta || !tb || !tc || !td)) { c->err = "md_set_dihedrals: null tag array"; return MD_EINVAL; }
    if (nd >= 0x3fffffffull) { c->err = "md_set_dihedrals: too many dihedrals"; return MD_EINVAL; }
    MD_TRY(alloc_state(c));
    MD_TRY(md_sync(c));
    for (uint32_t **q : {&c->dih_off, &c->dih_ent, &c->dih_abcd})
        if (*q) { md_free(c, *q); *q = nullptr; }
    c->n_dihedrals = nd;
    if (nd == 0) return MD_OK;
    if (!is_device_ptr(ta))
        for (uint64_t m = 0; m < nd; ++m) {
            const uint32_t q[4] = {ta[m], tb[m], tc[m], td[m]};
            bool bad = false;
            for (int x = 0; x < 4; ++x) {
                bad |= q[x] >= c->N;
                for (int y = x + 1; y < 4; ++y) bad |= q[x] == q[y];
            }
            if (bad) {
                c->err = "md_set_dihedrals: tag out of range or repeated in a quadruplet";
                c->n_dihedrals = 0;
                return MD_EINVAL;
            }
        }
    MD_TRY(md_alloc(c, (void **)&c->dih_off, (c->N + 1) * sizeof(uint32_t)));
    MD_TRY(md_alloc(c, (void **)&c->dih_ent, 4 * nd * sizeof(uint32_t)));
    MD_TRY(md_alloc(c, (void **)&c->dih_abcd, 4 * nd * sizeof(uint32_t)));
    Stage st(c);
    const uint64_t bb = nd * sizeof(uint32_t);
    MD_TRY(st.reserve(stage_need(ta, bb) + stage_need(tb, bb) + stage_need(tc, bb) + stage_need(td, bb)));
    const void *da, *db, *dc, *dd;
    MD_TRY(stage_in(c, st, ta, bb, &da));
    MD_TRY(stage_in(c, st, tb, bb, &db));
    MD_TRY(stage_in(c, st, tc, bb, &dc));
    MD_TRY(stage_in(c, st, td, bb, &dd));
    MD_TRY(launch_dihedrals_build(c, (const uint32_t *)da, (const uint32_t *)db, (const uint32_t *)dc, (const uint32_t *)dd, nd));
    return md_sync(c);
}

extern "C" int md_forces_dihedrals(md_ctx *c, double k, int sign, int n)
{
    if (!c) return MD_EINVAL;
    if ((sign != 1 && sign != -1) || n < 1) { c->err = "md_forces_dihedrals: sign must be +1 or -1 and n >= 1"; return MD_EINVAL; }
    if (!c->have_state) { c->err = "md_forces_dihedrals: md_set_state first"; return MD_ESTATE; }
    if (c->n_dihedrals == 0) { c->force_valid = true; return MD_OK; }
    ProfScope ps(c, MD_K_BONDS);
    MD_TRY(launch_forces_dihedrals(c, k, sign, n));
    c->force_valid = true;
    return MD_OK;
}

extern "C" int md_forces_langevin(md_ctx *c, double gamma, double kT, double dt, uint64_t step, uint64_t seed)
{
    if (!c) return MD_EINVAL;
    if (!(gamma >= 0.0) || !(kT >= 0.0) || !(dt > 0.0)) { c->err = "md_forces_langevin: gamma >= 0, kT >= 0, dt > 0 required"; return MD_EINVAL; }
    if (!c->have_state) { c->err = "md_forces_langevin: md_set_state first"; return MD_ESTATE; }
    ProfScope ps(c, MD_K_BONDS);
    MD_TRY(launch_forces_langevin(c, gamma, kT, dt, step, seed));
    c->force_valid = true;
    return MD_OK;
}

extern "C" int md_integrate_nve(md_ctx *c, double dt, int half)
{
    if (!c) return MD_EINVAL;
    if (!c->have_state) { c->err = "md_integrate_nve: md_set_state first"; return MD_ESTATE; }
    if (half == 1) {
        if (!c->cells_valid) MD_TRY(do_build_cells(c));  // the displacement check needs the reference snapshot
        ProfScope ps(c, MD_K_INTEGRATE);
        MD_TRY(launch_half1(c, dt, false));
        c->steps_since_build++;
        c->force_valid = false;
        return MD_OK;
    }
    if (half == 2) { ProfScope ps(c, MD_K_INTEGRATE); return launch_half2(c, dt); }
    c->err = "md_integrate_nve: half must be 1 or 2";
    return MD_EINVAL;
}

extern "C" int md_integrate_nvt(md_ctx *c, double dt, int half, double kT, double tau)
{
    if (!c) return MD_EINVAL;
    if (!c->have_state) { c->err = "md_integrate_nvt: md_set_state first"; return MD_ESTATE; }
    if (!(kT > 0.0) || !(tau > 0.0)) { c->err = "md_integrate_nvt: kT and tau must be positive"; return MD_EINVAL; }
    if (half == 1) {
        if (!c->cells_valid) MD_TRY(do_build_cells(c));
        ProfScope ps(c, MD_K_INTEGRATE);
        MD_TRY(launch_half1(c, dt, false, true));
        MD_TRY(launch_nvt_thermostat(c, dt, kT, tau));
        c->steps_since_build++;
        c->force_valid = false;
        return MD_OK;
    }
    if (half == 2) { ProfScope ps(c, MD_K_INTEGRATE); return launch_half2(c, dt, true); }
    c->err = "md_integrate_nvt: half must be 1 or 2";
    return MD_EINVAL;
}

extern "C" int md_mtk_thermostat_half(md_ctx *c, double dt, double kT, double tau)
{
    if (!c) return MD_EINVAL;
    if (!c->have_state) { c->err = "md_mtk_thermostat_half: md_set_state first"; return MD_ESTATE; }
    if (!(dt > 0.0) || !(kT > 0.0) || !(tau > 0.0)) { c->err = "md_mtk_thermostat_half: dt, kT and tau must be positive"; return MD_EINVAL; }
    ProfScope ps(c, MD_K_INTEGRATE);
    return launch_mtk_thermostat(c, dt, kT, tau, 1);
}

extern "C" int md_set_thermostat(md_ctx *c, double xi, double eta)
{
    if (!c) return MD_EINVAL;
    if (!c->have_state) { c->err = "md_set_thermostat: md_set_state first"; return MD_ESTATE; }
    const double v[2] = {xi, eta};
    MD_CUDA_CHECK(c, cudaMemcpyAsync(c->nvt_state, v, sizeof(v), cudaMemcpyHostToDevice, c->stream));
    return md_sync(c);
}

extern "C" int md_get_thermostat(md_ctx *c, double *xi, double *eta)
{
    if (!c || !xi || !eta) return MD_EINVAL;
    if (!c->have_state) { c->err = "md_get_thermostat: md_set_state first"; return MD_ESTATE; }
    double v[2];
    MD_CUDA_CHECK(c, cudaMemcpyAsync(v, c->nvt_state, sizeof(v), cudaMemcpyDeviceToHost, c->stream));
    MD_TRY(md_sync(c));
    *xi = v[0];
    *eta = v[1];
    return MD_OK;
}

extern "C" int md_needs_rebuild(md_ctx *c, int *flag)
{
    if (!c || !flag) return MD_EINVAL;
    MD_TRY(md_read_flags(c));
    *flag = c->h_flags->rebuild;
    return MD_OK;
}

// =====================================================================================================
// S7 step scheduler
// =====================================================================================================
static int eval_forces(md_ctx *c, const md_step_desc *w, uint64_t step, bool energy)
{
    bool any = false;
    if (w->flags & MD_F_LJ) {
        ProfScope ps(c, MD_K_LJ);
        MD_TRY(pair_lj(c, w->lj_epsilon, w->lj_sigma, w->lj_energy_shift, energy));
        any = true;
    }
    if (w->flags & MD_F_DPD) {
        if (any) { c->err = "md_step: LJ and DPD pair terms are mutually exclusive (each overwrites the force)"; return MD_EINVAL; }
        ProfScope ps(c, MD_K_DPD);
        MD_TRY(pair_dpd(c, w->dpd_A, w->dpd_gamma, w->dpd_kT, w->dt, step, w->dpd_seed));
        any = true;
    }
    if (w->flags & MD_F_PAIR) {
        if (any) { c->err = "md_step: the pair terms (LJ, DPD, MD_F_PAIR) are mutually exclusive (each overwrites the force)"; return MD_EINVAL; }
        if (w->pair_kind < MD_PAIR_LJ || w->pair_kind > MD_PAIR_TABLE) { c->err = "md_step: unknown pair_kind"; return MD_EINVAL; }
        if (w->pair_kind == MD_PAIR_TABLE && c->tab_m == 0) { c->err = "md_step: md_set_pair_table first"; return MD_ESTATE; }
        ProfScope ps(c, MD_K_LJ);
        MD_TRY(ensure_decoded(c));
        MD_TRY(launch_forces_pair(c, w->pair_kind, w->pair_p, w->lj_energy_shift));
        any = true;
    }
    if (!any) MD_TRY(launch_zero_force(c));
    if ((w->flags & MD_F_BONDS) && c->n_bonds) {
        if (w->bond_kind < MD_BOND_HARMONIC || w->bond_kind > MD_BOND_TABLE) { c->err = "md_step: unknown bond_kind"; return MD_EINVAL; }
        if (w->bond_kind == MD_BOND_TABLE && c->btab_m == 0) { c->err = "md_step: md_set_bond_table first"; return MD_ESTATE; }
        ProfScope ps(c, MD_K_BONDS);
        MD_TRY(launch_forces_bonds(c, w->bond_k, w->bond_r0, w->bond_kind));
    }
    if ((w->flags & MD_F_ANGLES) && c->n_angles) {
        ProfScope ps(c, MD_K_BONDS);
        MD_TRY(launch_forces_angles(c, w->angle_k, w->angle_theta0));
    }
    if ((w->flags & MD_F_DIHEDRALS) && c->n_dihedrals) {
        if ((w->dihedral_sign != 1 && w->dihedral_sign != -1) || w->dihedral_n < 1) {
            c->err = "md_step: dihedral_sign must be +1 or -1 and dihedral_n >= 1";
            return MD_EINVAL;
        }
        ProfScope ps(c, MD_K_BONDS);
        MD_TRY(launch_forces_dihedrals(c, w->dihedral_k, w->dihedral_sign, w->dihedral_n));
    }
    if (w->flags & MD_F_LANGEVIN) {
        if (!(w->langevin_gamma >= 0.0) || !(w->langevin_kT >= 0.0)) { c->err = "md_step: langevin_gamma >= 0 and langevin_kT >= 0 required"; return MD_EINVAL; }
        if (w->flags & MD_F_NVT) { c->err = "md_step: MD_F_LANGEVIN and MD_F_NVT are mutually exclusive"; return MD_EINVAL; }
        ProfScope ps(c, MD_K_BONDS);
        MD_TRY(launch_forces_langevin(c, w->langevin_gamma, w->langevin_kT, w->dt, step, w->langevin_seed));
    }
    c->force_valid = true;
    // only the tile LJ kernel skips the per-particle energies
    c->energy_valid = energy || !((w->flags & MD_F_LJ) && c->nl_is_tile);
    c->last_desc = *w;
    c->last_force_step = step;
    c->last_from_step = true;
    return MD_OK;
}

static int tune_all(md_ctx *c, const md_step_desc *w, int mode);

static int rebuild(md_ctx *c)
{
    MD_TRY(do_build_cells(c));
    return do_build_nlist(c);
}

// MD_SCHED_BATCH: no host round trip per step.  The kernels of a whole batch of steps are enqueued before the host looks at
// the rebuild flag; each is gated on DevFlags::rebuild_at (md_internal.h: Gate).  When half 1 of the batch's step m fires
// the displacement criterion it writes m; the force kernel of step m and everything enqueued after it find their gate
// closed and return at once, so the state stays exactly as that half 1 left it.  The host reads the flag once per batch,
// rebuilds, and resumes with the forces of step m: the same sequence of kernels on the same data as the other schedulers
// (bit-identical results).  The batch length follows the predicted distance to the next rebuild (largest displacement seen
// and its growth per step): a wrong prediction costs empty launches, never correctness.  PAPER.md:122 overlaps the check
// with a speculative force evaluation; PAPER.md:120, :163 are the launch overheads this removes at small N.
static int md_step_batch(md_ctx *c, const md_step_desc *w, uint64_t n_steps, bool nvt, bool mtk)
{
    // half 1 of the first step, not gated; its flag is read before anything else is enqueued
    {
        ProfScope ps(c, MD_K_INTEGRATE);
        c->gate_s = c->gate_set = c->gate_nvt = 0;
        if (mtk) MD_TRY(launch_mtk_thermostat(c, w->dt, w->nvt_kT, w->nvt_tau, 1));  // R39: leading T(dt/2) of the first step
        MD_TRY(launch_half1(c, w->dt, false, nvt));
        if (nvt) MD_TRY(launch_nvt_thermostat(c, w->dt, w->nvt_kT, w->nvt_tau));
    }
    c->steps_since_build++;
    MD_TRY(md_read_flags(c));
    bool flagged = c->h_flags->rebuild != 0;
    uint64_t done = 0;
    while (done < n_steps) {
        if (flagged) {
            if (c->h_flags->dangerous) c->stats.dangerous_builds++;
            MD_TRY(rebuild(c));
            if (c->retune_period && c->stats.rebuilds - c->rebuilds_at_tune >= c->retune_period) MD_TRY(tune_all(c, w, 2));
        } else {
            float d2;
            memcpy(&d2, &c->h_flags->max_d2[c->d2_slot], sizeof(float));
            c->last_d2 = d2;
            if (c->steps_since_build > 0) c->d2_rate = sqrt((double)d2) / (double)c->steps_since_build;
        }
        // batch length: the steps the largest displacement still has to the threshold at its observed growth
        uint64_t K = n_steps - done;
        {
            const double room = 0.5 * c->r_buff - sqrt((double)c->last_d2);
            const double rate = c->d2_rate > 0.0 ? c->d2_rate : 0.0;
            uint64_t pred = rate > 0.0 ? (uint64_t)std::max(1.0, floor(room / rate)) : (c->steps_since_build == 0 ? 2 : 4);
            K = std::min<uint64_t>(K, std::min<uint64_t>(std::max<uint64_t>(pred, 1), 64));
        }
        MD_CUDA_CHECK(c, cudaMemsetAsync(&c->d_flags->rebuild_at, 0, sizeof(unsigned int), c->stream));
        for (uint64_t j = 1; j <= K; ++j) {
            c->gate_s = (unsigned int)j;
            MD_TRY(eval_forces(c, w, c->step + j, false));  // R15: hash counter = index of the step being completed
            ProfScope ps(c, MD_K_INTEGRATE);
            if (done + j < n_steps && mtk) {
                // R39: half 2 of step j, its trailing T(dt/2) and the leading one of step j + 1 (one reduction: the second
                // factor's K is s^2 K), all part of step j; then the plain half 1 of step j + 1
                MD_TRY(launch_half2(c, w->dt, false));
                MD_TRY(launch_mtk_thermostat(c, w->dt, w->nvt_kT, w->nvt_tau, 2));
                c->gate_s = c->gate_set = (unsigned int)(j + 1);
                MD_TRY(launch_half1(c, w->dt, false, false));
                c->gate_s = (unsigned int)j;
            } else if (done + j < n_steps) {
                c->gate_set = c->gate_nvt = (unsigned int)(j + 1);
                MD_TRY(launch_half1(c, w->dt, true, nvt));   // half 2 of step j + half 1 of step j + 1
                if (nvt) { c->gate_nvt = (unsigned int)j; MD_TRY(launch_nvt_thermostat(c, w->dt, w->nvt_kT, w->nvt_tau)); }
            } else {
                MD_TRY(launch_half2(c, w->dt, nvt));
                if (mtk) MD_TRY(launch_mtk_thermostat(c, w->dt, w->nvt_kT, w->nvt_tau, 1));
            }
        }
        c->gate_s = c->gate_set = c->gate_nvt = 0;
        MD_TRY(md_read_flags(c));
        const uint64_t m = c->h_flags->rebuild_at;        // 0: every enqueued step ran; else steps 1 .. m-1 ran, half 1 of m fired
        const uint64_t ran = m == 0 ? K : m - 1;
        flagged = m != 0;
        done += ran;
        c->step += ran;
        c->stats.steps += ran;
        // half-1 steps since the binning: `ran` full steps' worth, plus the trailing half 1 of the next step if it ran
        c->steps_since_build += m == 0 ? (done < n_steps ? K : K - 1) : ran;
        if (m != 0) c->force_valid = false;
        if (c->profiling) prof_resolve_ready(c);
    }
    c->force_valid = true;
    return MD_OK;
}

// Step loop.  The displacement criterion is decided on the device by half 1; the host needs the flag to
// know whether to enqueue a rebuild.  As in the paper (forces are computed speculatively while the
// criterion is being checked) the force kernels are enqueued BEFORE the host waits for the flag whenever a rebuild
// is not expected at this step, so the device never idles on the round trip; if the flag then says "rebuild", the
// speculative forces are discarded and evaluated again on the new list.  Whether a rebuild is expected is predicted
// from the largest displacement of the previous step and its observed growth per step; a wrong prediction costs time
// only, never correctness (the flag is always read before the forces are used).  Inside the loop the second
// half-kick of a step and the first of the next are one launch (bit-identical to the two separate kernels).
extern "C" int md_step(md_ctx *c, const md_step_desc *w, uint64_t n_steps)
{
    if (!c || !w) return MD_EINVAL;
    if (!c->have_state) { c->err = "md_step: md_set_state first"; return MD_ESTATE; }
    if (!(w->dt > 0.0)) { c->err = "md_step: dt must be positive"; return MD_EINVAL; }
    if (n_steps == 0) return MD_OK;
    const bool nvt = (w->flags & MD_F_NVT) != 0, mtk = (w->flags & MD_F_MTK) != 0;
    if ((nvt || mtk) && (!(w->nvt_kT > 0.0) || !(w->nvt_tau > 0.0))) { c->err = "md_step: nvt_kT and nvt_tau must be positive"; return MD_EINVAL; }
    if (mtk && (w->flags & (MD_F_NVT | MD_F_LANGEVIN))) { c->err = "md_step: MD_F_MTK excludes MD_F_NVT and MD_F_LANGEVIN"; return MD_EINVAL; }
    c->force_hint = w->flags;
    if (w->flags & MD_F_LJ) {
        // the near sections of a mixed-precision tile list are sized for sigma (R25): a list built for a smaller one is rebuilt
        if (c->nlist_valid && c->nl_is_tile && c->precision == MD_MIXED && c->nl_near_r < MD_NEAR_SIGMAS * w->lj_sigma * (1.0 - 1e-12) &&
            c->steps_since_build == 0)
            c->nlist_valid = false;
        c->lj_sigma_hint = w->lj_sigma;
    }
    if (!c->nlist_valid) MD_TRY(rebuild(c));
    if (!c->force_valid) MD_TRY(eval_forces(c, w, c->step, false));  // R16: F(t0) before the first half-kick
    if (c->sched == MD_SCHED_BATCH) return md_step_batch(c, w, n_steps, nvt, mtk);
    if (!c->ev_flags) MD_CUDA_CHECK(c, cudaEventCreateWithFlags(&c->ev_flags, cudaEventDisableTiming));
    for (uint64_t s = 0; s < n_steps; ++s) {
        if (s == 0) {
            ProfScope ps(c, MD_K_INTEGRATE);
            if (mtk) MD_TRY(launch_mtk_thermostat(c, w->dt, w->nvt_kT, w->nvt_tau, 1));
            MD_TRY(launch_half1(c, w->dt, false, nvt));
            if (nvt) MD_TRY(launch_nvt_thermostat(c, w->dt, w->nvt_kT, w->nvt_tau));
        }
        c->steps_since_build++;
        MD_CUDA_CHECK(c, cudaMemcpyAsync(c->h_flags, c->d_flags, sizeof(DevFlags), cudaMemcpyDeviceToHost, c->stream));
        MD_CUDA_CHECK(c, cudaEventRecord(c->ev_flags, c->stream));
        // predicted largest displacement of this step: last one seen + the observed growth per step (with margin)
        const double d_prev = sqrt((double)c->last_d2);
        const bool speculate = c->sched != MD_SCHED_SYNC && d_prev + 1.5 * c->d2_rate < 0.5 * c->r_buff;
        if (speculate) {
            MD_TRY(eval_forces(c, w, c->step + 1, false));  // R15: hash counter = index of the step being completed
            c->stats.speculative_forces++;
        }
        MD_CUDA_CHECK(c, cudaEventSynchronize(c->ev_flags));
        if (c->profiling) prof_resolve_ready(c);
        {
            float d2;
            memcpy(&d2, &c->h_flags->max_d2[c->d2_slot], sizeof(float));
            c->last_d2 = d2;
            const double d = sqrt((double)d2);
            if (c->steps_since_build > 0) c->d2_rate = d / (double)c->steps_since_build;
        }
        if (c->h_flags->rebuild) {
            if (c->h_flags->dangerous) c->stats.dangerous_builds++;
            if (speculate) c->stats.wasted_forces++;
            MD_TRY(rebuild(c));
            // periodic re-scan: density and temperature drift move the optimum
            if (c->retune_period && c->stats.rebuilds - c->rebuilds_at_tune >= c->retune_period) MD_TRY(tune_all(c, w, 2));
            MD_TRY(eval_forces(c, w, c->step + 1, false));
        } else if (!speculate) {
            MD_TRY(eval_forces(c, w, c->step + 1, false));
        }
        {
            ProfScope ps(c, MD_K_INTEGRATE);
            if (s + 1 < n_steps && mtk) {
                MD_TRY(launch_half2(c, w->dt, false));
                MD_TRY(launch_mtk_thermostat(c, w->dt, w->nvt_kT, w->nvt_tau, 2));  // trailing T of this step + leading T of the next
                MD_TRY(launch_half1(c, w->dt, false, false));
            } else if (s + 1 < n_steps) {
                MD_TRY(launch_half1(c, w->dt, true, nvt));  // half 2 of this step + half 1 of the next
                if (nvt) MD_TRY(launch_nvt_thermostat(c, w->dt, w->nvt_kT, w->nvt_tau));
            } else {
                MD_TRY(launch_half2(c, w->dt, nvt));
                if (mtk) MD_TRY(launch_mtk_thermostat(c, w->dt, w->nvt_kT, w->nvt_tau, 1));
            }
        }
        c->step++;
        c->stats.steps++;
    }
    c->force_valid = true;
    return MD_OK;
}

// =====================================================================================================
// S8 runtime tuner: sweep block size x w, median of 5 timed launches, keep the fastest
// =====================================================================================================
template <typename F>
static int time_median5(md_ctx *c, F &&fn, float *us)
{
    cudaEvent_t e0, e1;
    MD_CUDA_CHECK(c, cudaEventCreate(&e0));
    MD_CUDA_CHECK(c, cudaEventCreate(&e1));
    float t[5];
    int s = fn();  // warm-up (also absorbs first-launch module load)
    for (int r = 0; r < 5 && s == MD_OK; ++r) {
        cudaEventRecord(e0, c->stream);
        s = fn();
        cudaEventRecord(e1, c->stream);
        cudaEventSynchronize(e1);
        cudaEventElapsedTime(&t[r], e0, e1);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (s != MD_OK) return s;
    std::sort(t, t + 5);
    *us = t[2] * 1000.f;
    return MD_OK;
}

// largest block size the kernel behind MD_K_* can be launched with in the current configuration (the __launch_bounds__
// of the variant the launcher picks): the tuner sweeps launchable sizes only and md_get_stats reports the launched one
int md_block_limit(const md_ctx *c, int kernel)
{
    const bool tile = c->nlist_valid ? c->nl_is_tile : c->use_tiles;
    switch (kernel) {
    case MD_K_NLIST: return tile ? MD_TILE_MAX_BLOCK : 1024;
    case MD_K_LJ: return !tile ? 1024 : (c->precision == MD_MIXED ? MD_LJ3_MAX_BLOCK : MD_TILE_MAX_BLOCK);
    case MD_K_DPD: return tile ? MD_DPD2_MAX_BLOCK : 1024;
    case MD_K_INTEGRATE: return MD_HALF1_MAX_BLOCK;
    default: return 1024;
    }
}

// mode 0: pruned grid, 1: every multiple of 32, 2: local re-scan around the current setting (periodic re-tune)
template <typename F>
static int tune_kernel(md_ctx *c, int kernel, const char *name, bool sweep_w, int w_max, int mode, F &&fn)
{
    static const int pruned[] = {32, 64, 96, 128, 192, 256, 384, 512, 768, 1024};
    const int n_pruned = (int)(sizeof(pruned) / sizeof(int));
    const int limit = md_block_limit(c, kernel);
    const LaunchCfg cur = c->cfg[kernel];
    std::vector<int> blocks, ws;
    if (mode == 1) { for (int b = 32; b <= limit; b += 32) blocks.push_back(b); }
    else if (mode == 2) {
        int at = 0;
        for (int i = 0; i < n_pruned; ++i) if (pruned[i] <= std::min(cur.block, limit)) at = i;
        for (int i = std::max(0, at - 1); i <= std::min(n_pruned - 1, at + 1); ++i) if (pruned[i] <= limit) blocks.push_back(pruned[i]);
    } else { for (int i = 0; i < n_pruned; ++i) if (pruned[i] <= limit) blocks.push_back(pruned[i]); }
    if (!sweep_w) ws.push_back(cur.w);
    else if (mode == 2) { for (int w = std::max(1, cur.w / 2); w <= std::min(w_max, cur.w * 2); w *= 2) ws.push_back(w); }
    else { for (int w = 1; w <= w_max; w *= 2) ws.push_back(w); }
    LaunchCfg best = cur;
    best.block = std::min(best.block, limit);
    best.us = 1e30f;
    for (int w : ws)
        for (int b : blocks) {
            c->cfg[kernel].block = b;
            c->cfg[kernel].w = w;
            float us;
            c->tune_skip = false;
            MD_TRY(time_median5(c, fn, &us));
            if (c->tune_skip) continue;
            if (c->log) fprintf(stderr, "[b200md tuner] %-10s block=%4d w=%2d  %9.1f us\n", name, b, w, us);
            if (us < best.us) best = LaunchCfg{b, w, us};
        }
    if (best.us > 1e29f) best.us = 0.f;  // nothing launchable was timed: keep the setting
    c->cfg[kernel] = best;
    if (c->log) fprintf(stderr, "[b200md tuner] %-10s -> block=%d w=%d (%.1f us)\n", name, best.block, best.w, best.us);
    return MD_OK;
}

static int tune_all(md_ctx *c, const md_step_desc *w, int mode)
{
    c->force_hint = w->flags;
    if (w->flags & MD_F_LJ) c->lj_sigma_hint = w->lj_sigma;
    const uint64_t rebuilds0 = c->stats.rebuilds + (c->nlist_valid ? 0 : 1);  // the replays are not rebuilds of the run
    // the kernels are pure functions of the live state, so they can be replayed without advancing the simulation
    // (every kernel is tuned).  Binning: only when no step has been taken since the last one (a replay
    // re-takes the reference snapshot of the displacement check, which must not move in time).
    if (c->cells_valid && c->steps_since_build == 0) {
        MD_TRY(tune_kernel(c, MD_K_CELLS, "cells", false, 1, mode, [&]() { return launch_build_cells(c); }));
        c->tile_desc_valid = false;
        c->nlist_valid = false;
        MD_CUDA_CHECK(c, cudaMemsetAsync(&c->d_flags->rebuild, 0, 2 * sizeof(int), c->stream));
    }
    if (!c->nlist_valid) MD_TRY(rebuild(c));
    if (c->nl_is_tile) {
        // tile build: the lanes per particle are fixed by the kernel (4 candidate phases, or a full warp with the ballot
        // variant); only the block size is swept
        MD_TRY(tune_kernel(c, MD_K_NLIST, "nlist/tile", false, 1, mode, [&]() {
            bool fits = false;
            const int st = launch_tile_build(c, &fits);
            if (!fits) c->tune_skip = true;  // this block size does not fit in shared memory
            return st;
        }));
        c->cfg[MD_K_NLIST].w = tile_build_lanes(c);
    } else {
        MD_TRY(tune_kernel(c, MD_K_NLIST, "nlist", true, 32, mode, [&]() {
            MD_TRY(launch_nlist_count(c));
            return launch_nlist_fill(c);
        }));
    }
    if (w->flags & MD_F_LJ)
        MD_TRY(tune_kernel(c, MD_K_LJ, c->nl_is_tile ? "lj/tile" : "lj", true, c->nl_is_tile && c->precision == MD_MIXED ? 8 : 32, mode, [&]() {
            // the row rotation of the tile list follows W (1, 2 or more lanes per particle): time each W on its own layout
            if (c->nl_is_tile && c->nl_rotw != tile_rot_class(c->cfg[MD_K_LJ].w)) MD_TRY(do_build_nlist(c));
            return pair_lj(c, w->lj_epsilon, w->lj_sigma, w->lj_energy_shift, false);
        }));
    if (w->flags & MD_F_DPD)
        MD_TRY(tune_kernel(c, MD_K_DPD, c->nl_is_tile ? "dpd/tile" : "dpd", true, 32, mode, [&]() {
            if (c->nl_is_tile && c->nl_rotw != tile_rot_class(c->cfg[MD_K_DPD].w)) MD_TRY(do_build_nlist(c));
            return pair_dpd(c, w->dpd_A, w->dpd_gamma, w->dpd_kT, w->dt, c->step, w->dpd_seed);
        }));
    if ((w->flags & MD_F_BONDS) && c->n_bonds)
        MD_TRY(tune_kernel(c, MD_K_BONDS, "bonds", false, 1, mode, [&]() { return launch_forces_bonds(c, w->bond_k, w->bond_r0); }));
    // half 1 with dt = 0 is the identity on positions and velocities (x + 0 v, v + 0 F/m) with the full memory traffic
    MD_TRY(tune_kernel(c, MD_K_INTEGRATE, "integrate", false, 1, mode, [&]() { return launch_half1(c, 0.0, false, false); }));
    // the list the run starts with has the layout of the chosen W
    if (c->nl_is_tile) {
        const bool dpd = (w->flags & MD_F_DPD) != 0 && !(w->flags & MD_F_LJ);
        if (c->nl_rotw != tile_rot_class(c->cfg[dpd ? MD_K_DPD : MD_K_LJ].w)) MD_TRY(do_build_nlist(c));
    }
    c->force_valid = false;  // the replays overwrote the force array with a partial evaluation
    c->tuned = true;
    c->stats.tuner_runs++;
    c->stats.rebuilds = rebuilds0;
    c->rebuilds_at_tune = c->stats.rebuilds;
    return MD_OK;
}

extern "C" int md_tune(md_ctx *c, const md_step_desc *w, int full)
{
    if (!c || !w) return MD_EINVAL;
    if (!c->have_state) { c->err = "md_tune: md_set_state first"; return MD_ESTATE; }
    if (!c->cells_valid) MD_TRY(do_build_cells(c));
    return tune_all(c, w, full ? 1 : 0);
}

// ---- the skin that gives the most time steps per second -------------------
static int set_rbuff(md_ctx *c, double r_buff)
{
    MD_TRY(md_sync(c));
    MD_TRY(set_geometry(c, r_buff));
    md_free(c, c->cell_count);
    md_free(c, c->cell_start);
    c->cell_count = c->cell_start = nullptr;
    MD_TRY(md_alloc(c, (void **)&c->cell_count, (uint64_t)c->n_cells * sizeof(uint32_t)));
    MD_TRY(md_alloc(c, (void **)&c->cell_start, ((uint64_t)c->n_cells + 1) * sizeof(uint32_t)));
    MD_TRY(build_cell_order(c));
    if (c->nl16) { md_free(c, c->nl16); c->nl16 = nullptr; }
    c->nl_stride = 0;
    c->cells_valid = c->nlist_valid = false;
    return MD_OK;
}

extern "C" int md_tune_rbuff(md_ctx *c, const md_step_desc *w, const double *candidates, uint32_t n_candidates,
                             uint64_t burst_steps, double *chosen)
{
    if (!c || !w) return MD_EINVAL;
    if (!c->have_state) { c->err = "md_tune_rbuff: md_set_state first"; return MD_ESTATE; }
    if (burst_steps == 0) burst_steps = 200;
    std::vector<double> cand;
    if (candidates && n_candidates) cand.assign(candidates, candidates + n_candidates);
    else for (double f : {0.5, 0.75, 1.0, 1.25, 1.5, 1.75, 2.0}) cand.push_back(f * (c->r_buff > 0.0 ? c->r_buff : 0.1 * c->rc));
    // the live state, saved in slot order (a consistent set of arrays) and restored after every burst
    const uint64_t N = c->N;
    struct Save { void *src; uint64_t bytes; void *copy; };
    std::vector<Save> sv = {{c->pos, N * sizeof(double4), nullptr},   {c->vel, N * sizeof(double4), nullptr},
                            {c->force, N * sizeof(double4), nullptr}, {c->image, 3 * N * sizeof(int), nullptr},
                            {c->tag, N * sizeof(uint32_t), nullptr},  {c->rtag, N * sizeof(uint32_t), nullptr},
                            {c->nvt_state, 4 * sizeof(double), nullptr}};
    int s = MD_OK;
    for (auto &v : sv) {
        if (s == MD_OK) s = md_alloc(c, &v.copy, v.bytes);
        if (s == MD_OK && cudaMemcpyAsync(v.copy, v.src, v.bytes, cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess) s = MD_ECUDA;
    }
    const uint64_t step0 = c->step;
    const bool fvalid = c->force_valid, evalid = c->energy_valid;
    const md_stats stats0 = c->stats;
    const double r0 = c->r_buff;
    auto restore = [&]() -> int {
        // the binning swaps the array twins: copy into whatever the context points at now
        void *dst[7] = {c->pos, c->vel, c->force, c->image, c->tag, c->rtag, c->nvt_state};
        for (size_t i = 0; i < sv.size(); ++i)
            MD_CUDA_CHECK(c, cudaMemcpyAsync(dst[i], sv[i].copy, sv[i].bytes, cudaMemcpyDeviceToDevice, c->stream));
        c->step = step0;
        c->force_valid = fvalid;
        c->energy_valid = evalid;
        c->cells_valid = c->nlist_valid = false;
        c->last_d2 = 0.f;
        c->d2_rate = 0.0;
        return MD_OK;
    };
    double best_r = r0, best_tps = 0.0;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (s == MD_OK && (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess)) s = MD_ECUDA;
    for (size_t k = 0; k < cand.size() && s == MD_OK; ++k) {
        if (!(cand[k] >= 0.0) || set_rbuff(c, cand[k]) != MD_OK) continue;  // skins the box cannot hold are skipped
        s = md_step(c, w, std::max<uint64_t>(10, burst_steps / 10));        // first list build + a few rebuilds, untimed
        if (s == MD_OK) {
            cudaEventRecord(e0, c->stream);
            s = md_step(c, w, burst_steps);
            cudaEventRecord(e1, c->stream);
        }
        if (s == MD_ENOMEM) {  // a skin whose list does not fit the caller's workspace is not a candidate
            if (c->log) fprintf(stderr, "[b200md tuner] r_buff=%.4f  skipped: %s\n", cand[k], c->err.c_str());
            cudaStreamSynchronize(c->stream);
            s = restore();
            continue;
        }
        if (s != MD_OK) break;
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double tps = 1e3 * (double)burst_steps / ms;
        if (c->log) fprintf(stderr, "[b200md tuner] r_buff=%.4f  %10.1f steps/s\n", cand[k], tps);
        if (tps > best_tps) { best_tps = tps; best_r = cand[k]; }
        s = restore();
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    int s2 = set_rbuff(c, best_r);   // (also when a burst failed: back to a valid configuration and the saved state)
    if (s2 == MD_OK) s2 = restore();
    if (s2 == MD_OK) s2 = md_sync(c);
    for (auto &v : sv) if (v.copy) md_free(c, v.copy);
    const uint64_t launches = c->stats.launches;
    c->stats = stats0;               // the bursts are not steps or rebuilds of the run
    c->stats.launches = launches;
    c->stats.r_buff = c->r_buff;
    c->stats.rbuff_tuned_tps = best_tps;
    if (c->log) fprintf(stderr, "[b200md tuner] r_buff -> %.4f (%.1f steps/s)\n", best_r, best_tps);
    if (chosen) *chosen = best_r;
    return s != MD_OK ? s : s2;
}

extern "C" int md_set_option(md_ctx *c, int option, int64_t value)
{
    if (!c) return MD_EINVAL;
    switch (option) {
    case MD_OPT_TILE_BRICK:
        if (value != 0 && value != 1 && value != 2 && value != 4) { c->err = "md_set_option: brick must be 0 (auto), 1, 2 or 4"; return MD_EINVAL; }
        c->tile_B_forced = (int)value;
        MD_TRY(md_sync(c));
        MD_TRY(build_cell_order(c));
        c->cells_valid = c->nlist_valid = false;
        return MD_OK;
    case MD_OPT_ACC_BLOCK:
        if (value != 1 && value != 8) { c->err = "md_set_option: accumulation block must be 1 or 8"; return MD_EINVAL; }
        c->acc_block = (int)value;
        return MD_OK;
    case MD_OPT_PROFILE_STRIDE:
        if (value < 1) { c->err = "md_set_option: profile stride must be >= 1"; return MD_EINVAL; }
        c->prof_stride = (uint64_t)value;
        c->prof_count = 0;
        return MD_OK;
    case MD_OPT_RETUNE_PERIOD:
        if (value < 0) { c->err = "md_set_option: re-tune period must be >= 0"; return MD_EINVAL; }
        c->retune_period = (uint64_t)value;
        return MD_OK;
    default:
        c->err = "md_set_option: unknown option";
        return MD_EINVAL;
    }
}

extern "C" int md_set_launch(md_ctx *c, int kernel, int block, int w)
{
    if (!c || kernel < 0 || kernel >= MD_N_KERNELS || block < 32 || block > 1024 || (block % 32) || w < 1 || w > 32 ||
        (w & (w - 1))) {
        if (c) c->err = "md_set_launch: bad argument";
        return MD_EINVAL;
    }
    c->cfg[kernel].block = block;
    c->cfg[kernel].w = w;
    c->cfg[kernel].us = 0.f;
    return MD_OK;
}

extern "C" int md_get_stats(md_ctx *c, md_stats *out)
{
    if (!c || !out) return MD_EINVAL;
    MD_TRY(md_sync(c));
    prof_resolve(c);
    c->stats.nlist_entries = c->nl_entries;
    c->stats.nlist_capacity = c->nl_capacity;
    c->stats.device_bytes = c->device_bytes;
    c->stats.mean_neighbors = c->N ? (double)c->nl_entries / (double)c->N : 0.0;
    for (int a = 0; a < 3; ++a) c->stats.dims[a] = c->dims[a];
    c->stats.r_buff = c->r_buff;
    for (int k = 0; k < MD_N_KERNELS; ++k) {
        c->stats.block[k] = std::min(c->cfg[k].block, md_block_limit(c, k));  // the launched size
        c->stats.w[k] = c->cfg[k].w;
        c->stats.tuned_us[k] = c->cfg[k].us;
    }
    *out = c->stats;
    return MD_OK;
}

extern "C" int md_thermo(md_ctx *c, md_thermo_t *out)
{
    if (!c || !out) return MD_EINVAL;
    if (!c->have_state) { c->err = "md_thermo: md_set_state first"; return MD_ESTATE; }
    if (!c->force_valid) { c->err = "md_thermo: no force has been computed for the current positions"; return MD_ESTATE; }
    if (!c->energy_valid && c->last_from_step) MD_TRY(energies_on_demand(c));
    double r[5];
    MD_TRY(launch_thermo(c, r));
    out->kinetic = r[0];
    out->potential = r[1];
    out->momentum[0] = r[2]; out->momentum[1] = r[3]; out->momentum[2] = r[4];
    out->temperature = c->N > 1 ? 2.0 * r[0] / (3.0 * (double)c->N - 3.0) : 0.0;
    return MD_OK;
}

extern "C" int md_pressure(md_ctx *c, const md_step_desc *w, md_pressure_t *out)
{
    if (!c || !w || !out) return MD_EINVAL;
    if (!c->have_state) { c->err = "md_pressure: md_set_state first"; return MD_ESTATE; }
    if ((w->flags & MD_F_BONDS) && c->n_bonds) {
        if (w->bond_kind < MD_BOND_HARMONIC || w->bond_kind > MD_BOND_TABLE) { c->err = "md_pressure: unknown bond_kind"; return MD_EINVAL; }
        if (w->bond_kind == MD_BOND_TABLE && c->btab_m == 0) { c->err = "md_pressure: md_set_bond_table first"; return MD_ESTATE; }
    }
    if (w->flags & MD_F_PAIR) {
        if (w->pair_kind < MD_PAIR_LJ || w->pair_kind > MD_PAIR_TABLE) { c->err = "md_pressure: unknown pair_kind"; return MD_EINVAL; }
        if (w->pair_kind == MD_PAIR_TABLE && c->tab_m == 0) { c->err = "md_pressure: md_set_pair_table first"; return MD_ESTATE; }
    }
    if ((w->flags & (MD_F_LJ | MD_F_DPD | MD_F_PAIR)) && (!c->nlist_valid || c->steps_since_build > 0)) {
        // the pair virial needs a list of the current positions only if the old one may have lost pairs: between
        // rebuilds the list still covers every pair within rc, so a valid list is enough
        if (!c->nlist_valid) MD_TRY(rebuild(c));
    }
    if (w->flags & (MD_F_LJ | MD_F_DPD | MD_F_PAIR)) MD_TRY(ensure_decoded(c));
    MD_TRY(launch_virial(c, w, c->step, out->virial));
    double r[5];
    MD_TRY(launch_thermo(c, r));
    out->kinetic = r[0];
    out->volume = c->box[0] * c->box[1] * c->box[2];
    out->pressure = (2.0 * r[0] + out->virial[0] + out->virial[1] + out->virial[2]) / (3.0 * out->volume);
    return MD_OK;
}

extern "C" int md_struct_size(int which)
{
    switch (which) {
    case 0: return (int)sizeof(md_step_desc);
    case 1: return (int)sizeof(md_stats);
    case 2: return (int)sizeof(md_thermo_t);
    case 3: return (int)sizeof(md_pressure_t);
    default: return -1;
    }
}

extern "C" int md_debug_philox(md_ctx *c, const uint32_t *ctr, const uint32_t *key, uint32_t *out, uint64_t n)
{
    if (!c || !ctr || !key || !out) return MD_EINVAL;
    Stage st(c);
    MD_TRY(st.reserve(stage_need(ctr, 16 * n) + stage_need(key, 8 * n) + stage_need(out, 16 * n)));
    const void *dc, *dk;
    MD_TRY(stage_in(c, st, ctr, 16 * n, &dc));
    MD_TRY(stage_in(c, st, key, 8 * n, &dk));
    OutBuf o = stage_out(st, out, 16 * n);
    MD_TRY(launch_debug_philox(c, (const uint32_t *)dc, (const uint32_t *)dk, (uint32_t *)o.dev, n));
    MD_TRY(finish_out(c, o));
    if (o.host) MD_TRY(md_sync(c));
    return MD_OK;
}
