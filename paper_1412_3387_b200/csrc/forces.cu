// forces.cu -- S4a LJ, S4b DPD pair forces over the neighbour list, S5 harmonic bonds.
//
// "the work for particle i is parallelized over its neighbors, processing w elements of its neighbor
// list in parallel, again in a strided fashion ... an intra-warp floating point reduction is applied to total up
// the particle force, which then is written to global memory."  Full (double-sided) list, so every particle's force
// is produced by its own W threads and written once: no atomics.
#include "md_device.cuh"

// ------------------------------------------------------------------------------------------------------------
// LJ 12-6, truncated at rc (R1).  MIXED: the pair polynomial runs in fp32 on the fp32-rounded
// separation, the r < rc decision is taken on the fp64 r^2 (R26), contributions are widened and summed in fp64.
// ------------------------------------------------------------------------------------------------------------
struct LJParams {
    double rc2, sig2, eps24, eps4, uc;  // uc = U(rc) if shifted else 0
    double near2;                       // MD_MIXED: pairs closer than this are evaluated in fp64 (R25)
};

template <int W, bool MIXED>
__global__ void __launch_bounds__(1024) k_forces_lj(const double4 *__restrict__ pos, const uint32_t *__restrict__ nl_cnt,
                                                    const uint64_t *__restrict__ nl_off,
                                                    const uint32_t *__restrict__ nl_idx, Geom g, LJParams p,
                                                    double4 *__restrict__ force, Gate gate)
{
    if (md_gate_closed(gate)) return;
    const uint32_t i = (uint32_t)(((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) / W);
    const unsigned lane = threadIdx.x & (W - 1);
    const unsigned seg_mask = md_seg_mask<W>();
    if (i >= g.N) return;
    const double4 pi = pos[i];
    const uint32_t n = nl_cnt[i];
    const uint32_t *row = nl_idx + nl_off[i];
    double fx = 0.0, fy = 0.0, fz = 0.0, en = 0.0;
    for (uint32_t k = lane; k < n; k += W) {
        const uint32_t j = row[k];
        const double4 pj = pos[j];
        const double dx = md_min_image(pi.x - pj.x, g.L[0], g.h[0]);
        const double dy = md_min_image(pi.y - pj.y, g.L[1], g.h[1]);
        const double dz = md_min_image(pi.z - pj.z, g.L[2], g.h[2]);
        const double r2 = md_r2_exact(dx, dy, dz);
        if (r2 < p.rc2) {
            if (MIXED && r2 >= p.near2) {  // (the first shell stays fp64: DESIGN.md R25)
                const float fdx = (float)dx, fdy = (float)dy, fdz = (float)dz;
                const float fr2 = fdx * fdx + fdy * fdy + fdz * fdz;
                const float rinv2 = 1.0f / fr2;
                const float s2 = (float)p.sig2 * rinv2;
                const float s6 = s2 * s2 * s2;
                const float f = (float)p.eps24 * s6 * (2.0f * s6 - 1.0f) * rinv2;
                fx += (double)(f * fdx);
                fy += (double)(f * fdy);
                fz += (double)(f * fdz);
                en += (double)(0.5f * ((float)p.eps4 * s6 * (s6 - 1.0f) - (float)p.uc));
            } else {
                const double rinv2 = 1.0 / r2;
                const double s2 = p.sig2 * rinv2;
                const double s6 = s2 * s2 * s2;
                const double f = p.eps24 * s6 * (2.0 * s6 - 1.0) * rinv2;
                fx += f * dx;
                fy += f * dy;
                fz += f * dz;
                en += 0.5 * (p.eps4 * s6 * (s6 - 1.0) - p.uc);
            }
        }
    }
    fx = md_seg_sum<W>(fx, seg_mask);
    fy = md_seg_sum<W>(fy, seg_mask);
    fz = md_seg_sum<W>(fz, seg_mask);
    en = md_seg_sum<W>(en, seg_mask);
    if (lane == 0) force[i] = make_double4(fx, fy, fz, en);
}

int launch_forces_lj(md_ctx *c, double eps, double sigma, int shift)
{
    const LaunchCfg &cf = c->cfg[MD_K_LJ];
    LJParams p;
    p.rc2 = c->rc * c->rc;
    p.sig2 = sigma * sigma;
    p.eps24 = 24.0 * eps;
    p.eps4 = 4.0 * eps;
    p.uc = 0.0;
    p.near2 = MD_NEAR_SIGMAS * MD_NEAR_SIGMAS * p.sig2;
    if (shift) {
        const double s2 = p.sig2 / p.rc2, s6 = s2 * s2 * s2;
        p.uc = 4.0 * eps * (s6 * s6 - s6);
    }
    const unsigned grid = md_grid(c->N * (uint64_t)cf.w, cf.block);
    const bool mixed = c->precision == MD_MIXED;
    MD_DISPATCH_W(cf.w, {
        if (mixed)
            k_forces_lj<W_, true><<<grid, cf.block, 0, c->stream>>>(c->pos, c->nl_cnt_exp, c->nl_off, c->nl_idx, c->g, p, c->force, md_gate(c));
        else
            k_forces_lj<W_, false><<<grid, cf.block, 0, c->stream>>>(c->pos, c->nl_cnt_exp, c->nl_off, c->nl_idx, c->g, p, c->force, md_gate(c));
    });
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

// ------------------------------------------------------------------------------------------------------------
// DPD (R9, R13-R15): conservative + drag + pairwise random force; fp64; needs neighbour velocities
// and tags.
// ------------------------------------------------------------------------------------------------------------
struct DPDParams {
    double rc2, inv_rc, A, gamma, sr;  // sr = sqrt(2 gamma kT) / sqrt(dt)
    uint64_t step, seed;
};

template <int W>
__global__ void __launch_bounds__(1024) k_forces_dpd(const double4 *__restrict__ pos, const double4 *__restrict__ vel,
                                                     const uint32_t *__restrict__ nl_cnt,
                                                     const uint64_t *__restrict__ nl_off,
                                                     const uint32_t *__restrict__ nl_idx, Geom g, DPDParams p,
                                                     double4 *__restrict__ force, Gate gate)
{
    if (md_gate_closed(gate)) return;
    const uint32_t i = (uint32_t)(((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) / W);
    const unsigned lane = threadIdx.x & (W - 1);
    const unsigned seg_mask = md_seg_mask<W>();
    if (i >= g.N) return;
    const double4 pi = pos[i];
    const double4 vi = vel[i];
    const uint32_t ti = md_lane_to_tag(pi.w);
    const uint32_t n = nl_cnt[i];
    const uint32_t *row = nl_idx + nl_off[i];
    double fx = 0.0, fy = 0.0, fz = 0.0, en = 0.0;
    for (uint32_t k = lane; k < n; k += W) {
        const uint32_t j = row[k];
        const double4 pj = pos[j];
        const double dx = md_min_image(pi.x - pj.x, g.L[0], g.h[0]);
        const double dy = md_min_image(pi.y - pj.y, g.L[1], g.h[1]);
        const double dz = md_min_image(pi.z - pj.z, g.L[2], g.h[2]);
        const double r2 = md_r2_exact(dx, dy, dz);
        if (r2 < p.rc2 && r2 > 0.0) {
            const double4 vj = vel[j];
            const double rinv = rsqrt(r2);
            const double r = r2 * rinv;
            const double w = 1.0 - r * p.inv_rc;
            const double rv = (dx * (vi.x - vj.x) + dy * (vi.y - vj.y) + dz * (vi.z - vj.z)) * rinv;
            const double theta = md_dpd_theta(ti, md_lane_to_tag(pj.w), p.step, p.seed);
            const double f = (p.A * w - p.gamma * w * w * rv + p.sr * w * theta) * rinv;
            fx += f * dx;
            fy += f * dy;
            fz += f * dz;
            en += 0.25 * p.A * w * w / p.inv_rc;  // half of U = A rc w^2 / 2
        }
    }
    fx = md_seg_sum<W>(fx, seg_mask);
    fy = md_seg_sum<W>(fy, seg_mask);
    fz = md_seg_sum<W>(fz, seg_mask);
    en = md_seg_sum<W>(en, seg_mask);
    if (lane == 0) force[i] = make_double4(fx, fy, fz, en);
}

int launch_forces_dpd(md_ctx *c, double A, double gamma, double kT, double dt, uint64_t step, uint64_t seed)
{
    const LaunchCfg &cf = c->cfg[MD_K_DPD];
    DPDParams p;
    p.rc2 = c->rc * c->rc;
    p.inv_rc = 1.0 / c->rc;
    p.A = A;
    p.gamma = gamma;
    p.sr = sqrt(2.0 * gamma * kT) / sqrt(dt);
    p.step = step;
    p.seed = seed;
    const unsigned grid = md_grid(c->N * (uint64_t)cf.w, cf.block);
    MD_DISPATCH_W(cf.w, {
        k_forces_dpd<W_><<<grid, cf.block, 0, c->stream>>>(c->pos, c->vel, c->nl_cnt_exp, c->nl_off, c->nl_idx, c->g, p, c->force, md_gate(c));
    });
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

// ------------------------------------------------------------------------------------------------------------
// harmonic (R19), FENE (R33) and tabulated (R38) bonds: every particle sums its own bonds (CSR by tag, partners ascending),
// no atomics.  Tabulated: kb = r_min, r0 = h (node spacing), tab = (U_k, F_k) pairs, tab_m nodes, r_hi = r_max.
// ------------------------------------------------------------------------------------------------------------
__global__ void k_forces_bonds(const double4 *__restrict__ pos, const uint32_t *__restrict__ tag,
                               const uint32_t *__restrict__ rtag, const uint32_t *__restrict__ bond_off,
                               const uint32_t *__restrict__ bond_partner, Geom g, double kb, double r0, int kind,
                               const double2 *__restrict__ tab, uint32_t tab_m, double r_hi,
                               double4 *__restrict__ force, Gate gate)
{
    if (md_gate_closed(gate)) return;
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.N) return;
    const uint32_t t = tag[i];
    const uint32_t b = bond_off[t], e = bond_off[t + 1];
    if (b == e) return;
    const double4 pi = pos[i];
    double fx = 0.0, fy = 0.0, fz = 0.0, en = 0.0;
    for (uint32_t m = b; m < e; ++m) {
        const double4 pj = pos[rtag[bond_partner[m]]];
        const double dx = md_min_image(pi.x - pj.x, g.L[0], g.h[0]);
        const double dy = md_min_image(pi.y - pj.y, g.L[1], g.h[1]);
        const double dz = md_min_image(pi.z - pj.z, g.L[2], g.h[2]);
        const double r2 = dx * dx + dy * dy + dz * dz;
        if (r2 > 0.0) {
            double f, u;
            if (kind == MD_BOND_HARMONIC) {
                const double r = sqrt(r2);
                f = -kb * (r - r0) / r;
                u = 0.5 * kb * (r - r0) * (r - r0);
            } else if (kind == MD_BOND_FENE) {  // DESIGN.md R33: NaN once the bond is stretched to r0
                const double x = r2 / (r0 * r0);
                f = x < 1.0 ? -kb / (1.0 - x) : nan("");
                u = x < 1.0 ? -0.5 * kb * r0 * r0 * log(1.0 - x) : nan("");
            } else {  // tabulated (R38): linear interpolation between two nodes; NaN once the bond has left the table
                const double r = sqrt(r2);
                if (r < kb || !(r < r_hi)) {
                    f = nan(""); u = nan("");
                } else {
                    const double sx = __ddiv_rn(__dsub_rn(r, kb), r0);
                    uint32_t k = (uint32_t)floor(sx);
                    k = min(k, tab_m - 2u);
                    const double t = __dsub_rn(sx, (double)k);
                    const double2 a = __ldg(tab + k), b2 = __ldg(tab + k + 1);
                    u = a.x + t * (b2.x - a.x);
                    f = (a.y + t * (b2.y - a.y)) / r;
                }
            }
            fx += f * dx;
            fy += f * dy;
            fz += f * dz;
            en += 0.5 * u;
        }
    }
    double4 f = force[i];
    f.x += fx; f.y += fy; f.z += fz; f.w += en;
    force[i] = f;
}

int launch_forces_bonds(md_ctx *c, double k, double r0, int kind)
{
    const LaunchCfg &cf = c->cfg[MD_K_BONDS];
    const double2 *tab = nullptr;
    uint32_t tab_m = 0;
    double r_hi = 0.0;
    if (kind == MD_BOND_TABLE) {  // parameters of md_set_bond_table (the caller has checked that one is set)
        tab = (const double2 *)c->btab_uf;
        tab_m = c->btab_m;
        k = c->btab_rmin;
        r0 = (c->btab_rmax - c->btab_rmin) / (double)(c->btab_m - 1);
        r_hi = c->btab_rmax;
    }
    k_forces_bonds<<<md_grid(c->N, cf.block), cf.block, 0, c->stream>>>(c->pos, c->tag, c->rtag, c->bond_off,
                                                                       c->bond_partner, c->g, k, r0, kind, tab, tab_m, r_hi,
                                                                       c->force, md_gate(c));
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

// forces of a step without a pair term start from zero (gated like a force kernel: MD_SCHED_BATCH)
__global__ void k_zero_force(double4 *__restrict__ force, uint32_t N, Gate gate)
{
    if (md_gate_closed(gate)) return;
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) force[i] = make_double4(0.0, 0.0, 0.0, 0.0);
}

int launch_zero_force(md_ctx *c)
{
    k_zero_force<<<md_grid(c->N, 256), 256, 0, c->stream>>>(c->force, (uint32_t)c->N, md_gate(c));
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

// energies on demand (md_get_forces / md_thermo after md_step): only the energy lane of a re-evaluation is kept
__global__ void k_copy_energy(double4 *__restrict__ force, const double4 *__restrict__ src, uint32_t N)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) force[i].w = src[i].w;
}

int launch_copy_energy(md_ctx *c, const double4 *src)
{
    k_copy_energy<<<md_grid(c->N, 256), 256, 0, c->stream>>>(c->force, src, (uint32_t)c->N);
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

// ------------------------------------------------------------------------------------------------------------
// test hook: the device hash, as the DPD kernel calls it
// ------------------------------------------------------------------------------------------------------------
__global__ void k_debug_philox(const uint32_t *ctr, const uint32_t *key, uint32_t *out, uint64_t n)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint4 r = md_philox4x32_10(make_uint4(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3]),
                                     make_uint2(key[2 * i], key[2 * i + 1]));
    out[4 * i] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
}

int launch_debug_philox(md_ctx *c, const uint32_t *ctr, const uint32_t *key, uint32_t *out, uint64_t n)
{
    k_debug_philox<<<md_grid(n, 128), 128, 0, c->stream>>>(ctr, key, out, n);
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}
