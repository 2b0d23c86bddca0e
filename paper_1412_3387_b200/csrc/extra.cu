// extra.cu -- SURVEY.md 8(f) rows 1 and 3 on the device: further short-range pair potentials (Yukawa, Gaussian, Morse,
// tabulated) on the W-threads-per-particle force kernel, harmonic angles and periodic dihedrals (per-particle CSR, no
// atomics), the Langevin thermostat as a one-body force, and the virial of every force term for the pressure (NPT / NPH
// of PAPER.md:63 need it).  The paper names these and prints no formula: DESIGN.md R31-R37.  fp64 throughout; the pair kernels read the exact 32-bit neighbour list (a tile list is decoded first).
#include "md_device.cuh"

// ------------------------------------------------------------------------------------------------------------
// R31, R37: f = -(dU/dr)/r and U of one pair; POT: MD_PAIR_LJ / YUKAWA / GAUSSIAN / MORSE / TABLE
// ------------------------------------------------------------------------------------------------------------
struct PairParams {
    double rc2, p0, p1, p2, uc;  // uc = U(rc) if the energy is shifted, else 0
    // MD_PAIR_TABLE (R37): (U_k, F_k) at r_min + k h; rc2 = r_max^2, p0 = r_min, p1 = h
    const double2 *tab;
    uint32_t tab_m;
};

template <int POT>
__device__ __forceinline__ double pair_eval(double r2, const PairParams &p, double &u)
{
    if (POT == MD_PAIR_LJ) {
        const double s2 = p.p1 * p.p1 / r2, s6 = s2 * s2 * s2;
        u = 4.0 * p.p0 * s6 * (s6 - 1.0);
        return 24.0 * p.p0 * s6 * (2.0 * s6 - 1.0) / r2;
    } else if (POT == MD_PAIR_YUKAWA) {
        const double r = sqrt(r2), e = p.p0 * exp(-p.p1 * r);
        u = e / r;
        return e * (p.p1 * r + 1.0) / (r2 * r);
    } else if (POT == MD_PAIR_GAUSSIAN) {
        const double e = p.p0 * exp(-r2 / (2.0 * p.p1 * p.p1));
        u = e;
        return e / (p.p1 * p.p1);
    } else if (POT == MD_PAIR_MORSE) {
        const double r = sqrt(r2), e1 = exp(-p.p1 * (r - p.p2)), e2 = e1 * e1;
        u = p.p0 * (e2 - 2.0 * e1);
        return 2.0 * p.p1 * p.p0 * (e2 - e1) / r;
    } else {  // MD_PAIR_TABLE: linear interpolation of U and F between the two nodes around r; nothing below r_min
        const double r = sqrt(r2);
        u = 0.0;
        if (r < p.p0) return 0.0;
        const double s = __ddiv_rn(__dsub_rn(r, p.p0), p.p1);
        uint32_t k = (uint32_t)floor(s);
        k = min(k, p.tab_m - 2u);
        const double t = __dsub_rn(s, (double)k);
        const double2 a = __ldg(p.tab + k), b = __ldg(p.tab + k + 1);
        u = a.x + t * (b.x - a.x);
        return (a.y + t * (b.y - a.y)) / r;
    }
}

static double pair_host_u(int kind, double r2, double p0, double p1, double p2)
{
    const double r = sqrt(r2);
    switch (kind) {
    case MD_PAIR_LJ: { const double s2 = p1 * p1 / r2, s6 = s2 * s2 * s2; return 4.0 * p0 * s6 * (s6 - 1.0); }
    case MD_PAIR_YUKAWA: return p0 * exp(-p1 * r) / r;
    case MD_PAIR_GAUSSIAN: return p0 * exp(-r2 / (2.0 * p1 * p1));
    default: { const double e1 = exp(-p1 * (r - p2)); return p0 * (e1 * e1 - 2.0 * e1); }
    }
}

// W threads stride over the row of particle i, shuffle reduction, one write per particle
template <int W, int POT>
__global__ void __launch_bounds__(1024) k_forces_pair(const double4 *__restrict__ pos, const uint32_t *__restrict__ nl_cnt,
                                                      const uint64_t *__restrict__ nl_off,
                                                      const uint32_t *__restrict__ nl_idx, Geom g, PairParams p,
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
        const double4 pj = pos[row[k]];
        const double dx = md_min_image(pi.x - pj.x, g.L[0], g.h[0]);
        const double dy = md_min_image(pi.y - pj.y, g.L[1], g.h[1]);
        const double dz = md_min_image(pi.z - pj.z, g.L[2], g.h[2]);
        const double r2 = md_r2_exact(dx, dy, dz);
        if (r2 < p.rc2 && r2 > 0.0) {
            double u;
            const double f = pair_eval<POT>(r2, p, u);
            fx += f * dx; fy += f * dy; fz += f * dz;
            en += 0.5 * (u - p.uc);
        }
    }
    fx = md_seg_sum<W>(fx, seg_mask);
    fy = md_seg_sum<W>(fy, seg_mask);
    fz = md_seg_sum<W>(fz, seg_mask);
    en = md_seg_sum<W>(en, seg_mask);
    if (lane == 0) force[i] = make_double4(fx, fy, fz, en);
}

static PairParams make_pair_params(md_ctx *c, int kind, const double prm[4], int shift)
{
    PairParams p;
    p.tab = nullptr;
    p.tab_m = 0;
    if (kind == MD_PAIR_TABLE) {
        p.rc2 = c->tab_rmax * c->tab_rmax;
        p.p0 = c->tab_rmin;
        p.p1 = (c->tab_rmax - c->tab_rmin) / (double)(c->tab_m - 1);
        p.p2 = 0.0;
        p.uc = 0.0;
        p.tab = (const double2 *)c->tab_uf;
        p.tab_m = c->tab_m;
        return p;
    }
    p.rc2 = c->rc * c->rc;
    p.p0 = prm[0]; p.p1 = prm[1]; p.p2 = prm[2];
    p.uc = shift ? pair_host_u(kind, p.rc2, p.p0, p.p1, p.p2) : 0.0;
    return p;
}

__global__ void k_table_pack(const double *__restrict__ U, const double *__restrict__ F, uint32_t m, double2 *__restrict__ tab)
{
    const uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < m) tab[k] = make_double2(U[k], F[k]);
}

int launch_table_pack(md_ctx *c, const double *U, const double *F, uint32_t m, double *dst_uf)
{
    k_table_pack<<<md_grid(m, 256), 256, 0, c->stream>>>(U, F, m, (double2 *)dst_uf);
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

int launch_forces_pair(md_ctx *c, int kind, const double prm[4], int shift)
{
    const LaunchCfg &cf = c->cfg[MD_K_LJ];
    const PairParams p = make_pair_params(c, kind, prm, shift);
    const int w = cf.w > 8 ? 8 : cf.w;
    const unsigned grid = md_grid(c->N * (uint64_t)w, cf.block);
#define PAIR_LAUNCH(W_)                                                                                                          \
    switch (kind) {                                                                                                              \
    case MD_PAIR_LJ: k_forces_pair<W_, MD_PAIR_LJ><<<grid, cf.block, 0, c->stream>>>(c->pos, c->nl_cnt_exp, c->nl_off, c->nl_idx, c->g, p, c->force, md_gate(c)); break; \
    case MD_PAIR_YUKAWA: k_forces_pair<W_, MD_PAIR_YUKAWA><<<grid, cf.block, 0, c->stream>>>(c->pos, c->nl_cnt_exp, c->nl_off, c->nl_idx, c->g, p, c->force, md_gate(c)); break; \
    case MD_PAIR_GAUSSIAN: k_forces_pair<W_, MD_PAIR_GAUSSIAN><<<grid, cf.block, 0, c->stream>>>(c->pos, c->nl_cnt_exp, c->nl_off, c->nl_idx, c->g, p, c->force, md_gate(c)); break; \
    case MD_PAIR_TABLE: k_forces_pair<W_, MD_PAIR_TABLE><<<grid, cf.block, 0, c->stream>>>(c->pos, c->nl_cnt_exp, c->nl_off, c->nl_idx, c->g, p, c->force, md_gate(c)); break; \
    default: k_forces_pair<W_, MD_PAIR_MORSE><<<grid, cf.block, 0, c->stream>>>(c->pos, c->nl_cnt_exp, c->nl_off, c->nl_idx, c->g, p, c->force, md_gate(c)); break; \
    }
    switch (w) {
    case 1: PAIR_LAUNCH(1); break;
    case 2: PAIR_LAUNCH(2); break;
    case 4: PAIR_LAUNCH(4); break;
    default: PAIR_LAUNCH(8); break;
    }
#undef PAIR_LAUNCH
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

// ------------------------------------------------------------------------------------------------------------
// R34 harmonic angles.  CSR by TAG built on the device: entry = 4 * angle index + role (0 = a, 1 = vertex b, 2 = c),
// rows sorted ascending so that a particle sums its terms in an order that does not depend on atomic arrival.
// ------------------------------------------------------------------------------------------------------------
__global__ void k_angle_count(const uint32_t *__restrict__ ta, const uint32_t *__restrict__ tb,
                              const uint32_t *__restrict__ tc, uint64_t na, uint32_t *cnt)
{
    const uint64_t m = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= na) return;
    atomicAdd(&cnt[ta[m]], 1u);
    atomicAdd(&cnt[tb[m]], 1u);
    atomicAdd(&cnt[tc[m]], 1u);
}

__global__ void k_angle_fill(const uint32_t *__restrict__ ta, const uint32_t *__restrict__ tb,
                             const uint32_t *__restrict__ tc, uint64_t na, const uint32_t *__restrict__ off,
                             uint32_t *fill, uint32_t *ent, uint32_t *abc)
{
    const uint64_t m = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= na) return;
    const uint32_t a = ta[m], b = tb[m], cc = tc[m];
    abc[3 * m] = a; abc[3 * m + 1] = b; abc[3 * m + 2] = cc;
    ent[off[a] + atomicAdd(&fill[a], 1u)] = 4u * (uint32_t)m;
    ent[off[b] + atomicAdd(&fill[b], 1u)] = 4u * (uint32_t)m + 1u;
    ent[off[cc] + atomicAdd(&fill[cc], 1u)] = 4u * (uint32_t)m + 2u;
}

__global__ void k_sort_rows_u32(const uint32_t *__restrict__ off, uint32_t N, uint32_t *v)
{
    const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= N) return;
    const uint32_t b = off[t], e = off[t + 1];
    for (uint32_t i = b + 1; i < e; ++i) {  // insertion sort, rows are tiny
        const uint32_t x = v[i];
        uint32_t j = i;
        while (j > b && v[j - 1] > x) { v[j] = v[j - 1]; --j; }
        v[j] = x;
    }
}

int launch_angles_build(md_ctx *c, const uint32_t *ta, const uint32_t *tb, const uint32_t *tc, uint64_t na)
{
    cudaStream_t st = c->stream;
    const uint32_t N = (uint32_t)c->N;
    uint32_t *cnt = c->perm;  // scratch (N uint32), only valid to borrow outside a binning
    MD_CUDA_CHECK(c, cudaMemsetAsync(cnt, 0, sizeof(uint32_t) * N, st));
    k_angle_count<<<md_grid(na, 256), 256, 0, st>>>(ta, tb, tc, na, cnt);
    MD_LAUNCH_CHECK(c);
    MD_TRY(launch_exclusive_scan_u32(c, cnt, N, c->angle_off, nullptr, false, nullptr));
    MD_CUDA_CHECK(c, cudaMemsetAsync(cnt, 0, sizeof(uint32_t) * N, st));
    k_angle_fill<<<md_grid(na, 256), 256, 0, st>>>(ta, tb, tc, na, c->angle_off, cnt, c->angle_ent, c->angle_abc);
    MD_LAUNCH_CHECK(c);
    k_sort_rows_u32<<<md_grid(N, 256), 256, 0, st>>>(c->angle_off, N, c->angle_ent);
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

// force on the particle with role `role` of the angle (a, b, c) and (for the virial) its arm relative to the vertex
__device__ __forceinline__ bool angle_term(const double4 *__restrict__ pos, const uint32_t *__restrict__ rtag,
                                           const uint32_t *__restrict__ abc, uint32_t m, uint32_t role, const Geom &g,
                                           double k, double theta0, double F[3], double arm[3], double &u)
{
    const double4 xa = pos[rtag[abc[3 * m]]], xb = pos[rtag[abc[3 * m + 1]]], xc = pos[rtag[abc[3 * m + 2]]];
    const double r1[3] = {md_min_image(xa.x - xb.x, g.L[0], g.h[0]), md_min_image(xa.y - xb.y, g.L[1], g.h[1]),
                          md_min_image(xa.z - xb.z, g.L[2], g.h[2])};
    const double r2[3] = {md_min_image(xc.x - xb.x, g.L[0], g.h[0]), md_min_image(xc.y - xb.y, g.L[1], g.h[1]),
                          md_min_image(xc.z - xb.z, g.L[2], g.h[2])};
    const double l1s = r1[0] * r1[0] + r1[1] * r1[1] + r1[2] * r1[2], l2s = r2[0] * r2[0] + r2[1] * r2[1] + r2[2] * r2[2];
    if (!(l1s > 0.0) || !(l2s > 0.0)) return false;
    const double l12 = sqrt(l1s) * sqrt(l2s);
    double cs = (r1[0] * r2[0] + r1[1] * r2[1] + r1[2] * r2[2]) / l12;
    cs = fmin(1.0, fmax(-1.0, cs));
    const double sn = sqrt(1.0 - cs * cs);
    if (sn < 1e-12) return false;
    const double th = acos(cs), gg = k * (th - theta0) / sn;
    u = 0.5 * k * (th - theta0) * (th - theta0) / 3.0;
    double Fa[3], Fc[3];
#pragma unroll
    for (int x = 0; x < 3; ++x) {
        Fa[x] = gg * (r2[x] / l12 - cs * r1[x] / l1s);
        Fc[x] = gg * (r1[x] / l12 - cs * r2[x] / l2s);
    }
#pragma unroll
    for (int x = 0; x < 3; ++x) {
        F[x] = role == 0 ? Fa[x] : (role == 2 ? Fc[x] : -(Fa[x] + Fc[x]));
        arm[x] = role == 0 ? r1[x] : (role == 2 ? r2[x] : 0.0);
    }
    return true;
}

__global__ void k_forces_angles(const double4 *__restrict__ pos, const uint32_t *__restrict__ tag,
                                const uint32_t *__restrict__ rtag, const uint32_t *__restrict__ off,
                                const uint32_t *__restrict__ ent, const uint32_t *__restrict__ abc, Geom g, double k,
                                double theta0, double4 *__restrict__ force, Gate gate)
{
    if (md_gate_closed(gate)) return;
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.N) return;
    const uint32_t t = tag[i];
    const uint32_t b = off[t], e = off[t + 1];
    if (b == e) return;
    double fx = 0.0, fy = 0.0, fz = 0.0, en = 0.0;
    for (uint32_t q = b; q < e; ++q) {
        double F[3], arm[3], u;
        if (angle_term(pos, rtag, abc, ent[q] >> 2, ent[q] & 3u, g, k, theta0, F, arm, u)) {
            fx += F[0]; fy += F[1]; fz += F[2]; en += u;
        }
    }
    double4 f = force[i];
    f.x += fx; f.y += fy; f.z += fz; f.w += en;
    force[i] = f;
}

int launch_forces_angles(md_ctx *c, double k, double theta0)
{
    const LaunchCfg &cf = c->cfg[MD_K_BONDS];
    k_forces_angles<<<md_grid(c->N, cf.block), cf.block, 0, c->stream>>>(c->pos, c->tag, c->rtag, c->angle_off, c->angle_ent,
                                                                        c->angle_abc, c->g, k, theta0, c->force, md_gate(c));
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

// ------------------------------------------------------------------------------------------------------------
// R35 periodic dihedrals U = k/2 (1 + s cos(n phi)).  Same storage as the angles: CSR by TAG, entry = 4 * dihedral
// index + role (0 = a, 1 = b, 2 = c, 3 = d), rows sorted; every particle sums the terms it takes part in.
// ------------------------------------------------------------------------------------------------------------
__global__ void k_dih_count(const uint32_t *__restrict__ ta, const uint32_t *__restrict__ tb, const uint32_t *__restrict__ tc,
                            const uint32_t *__restrict__ td, uint64_t nd, uint32_t *cnt)
{
    const uint64_t m = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= nd) return;
    atomicAdd(&cnt[ta[m]], 1u);
    atomicAdd(&cnt[tb[m]], 1u);
    atomicAdd(&cnt[tc[m]], 1u);
    atomicAdd(&cnt[td[m]], 1u);
}

__global__ void k_dih_fill(const uint32_t *__restrict__ ta, const uint32_t *__restrict__ tb, const uint32_t *__restrict__ tc,
                           const uint32_t *__restrict__ td, uint64_t nd, const uint32_t *__restrict__ off, uint32_t *fill,
                           uint32_t *ent, uint4 *abcd)
{
    const uint64_t m = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= nd) return;
    const uint4 q = make_uint4(ta[m], tb[m], tc[m], td[m]);
    abcd[m] = q;
    ent[off[q.x] + atomicAdd(&fill[q.x], 1u)] = 4u * (uint32_t)m;
    ent[off[q.y] + atomicAdd(&fill[q.y], 1u)] = 4u * (uint32_t)m + 1u;
    ent[off[q.z] + atomicAdd(&fill[q.z], 1u)] = 4u * (uint32_t)m + 2u;
    ent[off[q.w] + atomicAdd(&fill[q.w], 1u)] = 4u * (uint32_t)m + 3u;
}

int launch_dihedrals_build(md_ctx *c, const uint32_t *ta, const uint32_t *tb, const uint32_t *tc, const uint32_t *td, uint64_t nd)
{
    cudaStream_t st = c->stream;
    const uint32_t N = (uint32_t)c->N;
    uint32_t *cnt = c->perm;  // scratch (N uint32), only valid to borrow outside a binning
    MD_CUDA_CHECK(c, cudaMemsetAsync(cnt, 0, sizeof(uint32_t) * N, st));
    k_dih_count<<<md_grid(nd, 256), 256, 0, st>>>(ta, tb, tc, td, nd, cnt);
    MD_LAUNCH_CHECK(c);
    MD_TRY(launch_exclusive_scan_u32(c, cnt, N, c->dih_off, nullptr, false, nullptr));
    MD_CUDA_CHECK(c, cudaMemsetAsync(cnt, 0, sizeof(uint32_t) * N, st));
    k_dih_fill<<<md_grid(nd, 256), 256, 0, st>>>(ta, tb, tc, td, nd, c->dih_off, cnt, c->dih_ent, (uint4 *)c->dih_abcd);
    MD_LAUNCH_CHECK(c);
    k_sort_rows_u32<<<md_grid(N, 256), 256, 0, st>>>(c->dih_off, N, c->dih_ent);
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

__device__ __forceinline__ void md_cross(const double u[3], const double v[3], double w[3])
{
    w[0] = u[1] * v[2] - u[2] * v[1];
    w[1] = u[2] * v[0] - u[0] * v[2];
    w[2] = u[0] * v[1] - u[1] * v[0];
}

__device__ __forceinline__ double md_dot(const double u[3], const double v[3]) { return u[0] * v[0] + u[1] * v[1] + u[2] * v[2]; }

struct DihParams {
    double k, s;  // U = k/2 (1 + s cos(n phi))
    int n;
};

// force on the particle with role `role` of the dihedral (a, b, c, d) and (for the virial) its arm relative to b.
// F = x_a - x_b, G = x_b - x_c, H = x_d - x_c, A = F x G, B = H x G, phi = atan2((B x A).G / |G|, A.B)
// (only cos(n phi) and sin(n phi) are needed); gradients of phi after Blondel & Karplus; force = -dU/dphi grad phi, dU/dphi = -k/2 s n sin(n phi).
__device__ __forceinline__ bool dihedral_term(const double4 *__restrict__ pos, const uint32_t *__restrict__ rtag,
                                              const uint4 *__restrict__ abcd, uint32_t m, uint32_t role, const Geom &g,
                                              const DihParams &dp, double Fo[3], double arm[3], double &u)
{
    const uint4 q = abcd[m];
    const double4 xa = pos[rtag[q.x]], xb = pos[rtag[q.y]], xc = pos[rtag[q.z]], xd = pos[rtag[q.w]];
    const double F[3] = {md_min_image(xa.x - xb.x, g.L[0], g.h[0]), md_min_image(xa.y - xb.y, g.L[1], g.h[1]),
                         md_min_image(xa.z - xb.z, g.L[2], g.h[2])};
    const double G[3] = {md_min_image(xb.x - xc.x, g.L[0], g.h[0]), md_min_image(xb.y - xc.y, g.L[1], g.h[1]),
                         md_min_image(xb.z - xc.z, g.L[2], g.h[2])};
    const double H[3] = {md_min_image(xd.x - xc.x, g.L[0], g.h[0]), md_min_image(xd.y - xc.y, g.L[1], g.h[1]),
                         md_min_image(xd.z - xc.z, g.L[2], g.h[2])};
    double A[3], B[3], C[3];
    md_cross(F, G, A);
    md_cross(H, G, B);
    const double g2 = md_dot(G, G), a2 = md_dot(A, A), b2 = md_dot(B, B);
    if (!(g2 > 0.0) || a2 < 1e-24 * g2 * g2 || b2 < 1e-24 * g2 * g2) return false;
    const double gl = sqrt(g2);
    md_cross(B, A, C);
    // cos(n phi), sin(n phi) from cos phi = A.B / (|A| |B|), sin phi = (B x A).G / (|G| |A| |B|) by the angle-addition
    // recurrence (n is a small integer): no atan2 / sincos in the kernel
    const double iab = rsqrt(a2 * b2);
    const double c1 = md_dot(A, B) * iab, s1 = md_dot(C, G) / gl * iab;
    double cs = c1, sn = s1;
    for (int m = 1; m < dp.n; ++m) {
        const double t = cs * c1 - sn * s1;
        sn = sn * c1 + cs * s1;
        cs = t;
    }
    const double dU = -0.5 * dp.k * dp.s * (double)dp.n * sn;
    u = 0.125 * dp.k * (1.0 + dp.s * cs);
    const double fg = md_dot(F, G), hg = md_dot(H, G);
    const double ca = gl / a2, cb = gl / b2, ea = fg / (a2 * gl), eb = hg / (b2 * gl);
#pragma unroll
    for (int x = 0; x < 3; ++x) {
        double gr;  // d phi / d x_role
        if (role == 0) gr = -ca * A[x];
        else if (role == 1) gr = ca * A[x] + ea * A[x] - eb * B[x];
        else if (role == 2) gr = -cb * B[x] - ea * A[x] + eb * B[x];
        else gr = cb * B[x];
        Fo[x] = -dU * gr;
        arm[x] = role == 0 ? F[x] : (role == 2 ? -G[x] : (role == 3 ? H[x] - G[x] : 0.0));
    }
    return true;
}

__global__ void k_forces_dihedrals(const double4 *__restrict__ pos, const uint32_t *__restrict__ tag,
                                   const uint32_t *__restrict__ rtag, const uint32_t *__restrict__ off,
                                   const uint32_t *__restrict__ ent, const uint4 *__restrict__ abcd, Geom g, DihParams dp,
                                   double4 *__restrict__ force, Gate gate)
{
    if (md_gate_closed(gate)) return;
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.N) return;
    const uint32_t t = tag[i];
    const uint32_t b = off[t], e = off[t + 1];
    if (b == e) return;
    double fx = 0.0, fy = 0.0, fz = 0.0, en = 0.0;
    for (uint32_t q = b; q < e; ++q) {
        double F[3], arm[3], u;
        if (dihedral_term(pos, rtag, abcd, ent[q] >> 2, ent[q] & 3u, g, dp, F, arm, u)) {
            fx += F[0]; fy += F[1]; fz += F[2]; en += u;
        }
    }
    double4 f = force[i];
    f.x += fx; f.y += fy; f.z += fz; f.w += en;
    force[i] = f;
}

int launch_forces_dihedrals(md_ctx *c, double k, int sign, int n)
{
    const LaunchCfg &cf = c->cfg[MD_K_BONDS];
    const DihParams dp = {k, (double)sign, n};
    k_forces_dihedrals<<<md_grid(c->N, cf.block), cf.block, 0, c->stream>>>(c->pos, c->tag, c->rtag, c->dih_off, c->dih_ent,
                                                                           (const uint4 *)c->dih_abcd, c->g, dp, c->force,
                                                                           md_gate(c));
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

// ------------------------------------------------------------------------------------------------------------
// R36 Langevin thermostat: F_i += -gamma v_i + sqrt(6 gamma kT / dt) (u_x, u_y, u_z), u_k = 2 (X_k + 0.5) 2^-32 - 1 from
// Philox4x32-10 with counter (tag, 0xffffffff, step lo, step hi), key (seed lo, seed hi).  One thread per particle, one
// Philox block per particle and step; the operations are written in the oracle's order (no contraction): fp64 results
// identical up to the order of the additions into the force that is already there.
// ------------------------------------------------------------------------------------------------------------
__global__ void k_forces_langevin(const double4 *__restrict__ vel, const uint32_t *__restrict__ tag, uint32_t N, double gamma,
                                  double amp, uint64_t step, uint64_t seed, double4 *__restrict__ force, Gate gate)
{
    if (md_gate_closed(gate)) return;
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const uint4 x = md_philox4x32_10(make_uint4(tag[i], 0xffffffffu, (uint32_t)step, (uint32_t)(step >> 32)),
                                     make_uint2((uint32_t)seed, (uint32_t)(seed >> 32)));
    const double4 v = vel[i];
    double4 f = force[i];
    const double ux = __dsub_rn(__dmul_rn(2.0, __dmul_rn(__dadd_rn((double)x.x, 0.5), 1.0 / 4294967296.0)), 1.0);
    const double uy = __dsub_rn(__dmul_rn(2.0, __dmul_rn(__dadd_rn((double)x.y, 0.5), 1.0 / 4294967296.0)), 1.0);
    const double uz = __dsub_rn(__dmul_rn(2.0, __dmul_rn(__dadd_rn((double)x.z, 0.5), 1.0 / 4294967296.0)), 1.0);
    f.x = __dadd_rn(f.x, __dadd_rn(__dmul_rn(-gamma, v.x), __dmul_rn(amp, ux)));
    f.y = __dadd_rn(f.y, __dadd_rn(__dmul_rn(-gamma, v.y), __dmul_rn(amp, uy)));
    f.z = __dadd_rn(f.z, __dadd_rn(__dmul_rn(-gamma, v.z), __dmul_rn(amp, uz)));
    force[i] = f;
}

int launch_forces_langevin(md_ctx *c, double gamma, double kT, double dt, uint64_t step, uint64_t seed)
{
    const LaunchCfg &cf = c->cfg[MD_K_BONDS];
    k_forces_langevin<<<md_grid(c->N, cf.block), cf.block, 0, c->stream>>>(c->vel, c->tag, (uint32_t)c->N, gamma,
                                                                          sqrt(6.0 * gamma * kT / dt), step, seed, c->force,
                                                                          md_gate(c));
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

// ------------------------------------------------------------------------------------------------------------
// R32 virial W = sum over pairs of d (x) F (+ bonds, + angles and dihedrals: arm (x) F per end), order xx yy zz xy xz yz.  Every
// particle sums HALF of each of its pair and bond terms (the list is double-sided) and its own arm of each angle; a
// block sums a contiguous range of slots (shared-memory tree), one block sums the partials: fixed order, bit-reproducible.
// ------------------------------------------------------------------------------------------------------------
constexpr int VIR_BLOCK = 256;
constexpr uint32_t VIR_PER_BLOCK = 2048;
constexpr int VIR_NONE = 100, VIR_DPD = 101;

struct VirialTerms {
    PairParams pair;
    double dpd_inv_rc, dpd_A, dpd_gamma, dpd_sr;
    uint64_t dpd_step, dpd_seed;
    int bond_kind;  // -1: none
    double bond_k, bond_r0;
    const double2 *btab;  // MD_BOND_TABLE: bond_k = r_min, bond_r0 = h, btab_hi = r_max
    uint32_t btab_m;
    double btab_hi;
    int angles;
    double angle_k, angle_theta0;
    int dihedrals;
    DihParams dih;
};

__device__ __forceinline__ void vir_add(double w[6], double s, const double d[3], const double F[3])
{
    w[0] += s * d[0] * F[0]; w[1] += s * d[1] * F[1]; w[2] += s * d[2] * F[2];
    w[3] += s * d[0] * F[1]; w[4] += s * d[0] * F[2]; w[5] += s * d[1] * F[2];
}

template <int POT>
__global__ void __launch_bounds__(VIR_BLOCK) k_virial(const double4 *__restrict__ pos, const double4 *__restrict__ vel,
                                                      const uint32_t *__restrict__ tag, const uint32_t *__restrict__ rtag,
                                                      const uint32_t *__restrict__ nl_cnt, const uint64_t *__restrict__ nl_off,
                                                      const uint32_t *__restrict__ nl_idx,
                                                      const uint32_t *__restrict__ bond_off, const uint32_t *__restrict__ bond_partner,
                                                      const uint32_t *__restrict__ angle_off, const uint32_t *__restrict__ angle_ent,
                                                      const uint32_t *__restrict__ angle_abc, const uint32_t *__restrict__ dih_off,
                                                      const uint32_t *__restrict__ dih_ent, const uint4 *__restrict__ dih_abcd,
                                                      Geom g, VirialTerms vt,
                                                      double *__restrict__ partial /* [gridDim.x][6] */)
{
    __shared__ double sm[6 * VIR_BLOCK];
    const uint32_t b0 = blockIdx.x * VIR_PER_BLOCK, b1 = min(g.N, b0 + VIR_PER_BLOCK);
    double w[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    for (uint32_t i = b0 + threadIdx.x; i < b1; i += VIR_BLOCK) {
        const double4 pi = pos[i];
        if (POT != VIR_NONE) {
            const uint32_t n = nl_cnt[i];
            const uint32_t *row = nl_idx + nl_off[i];
            const double4 vi = POT == VIR_DPD ? vel[i] : make_double4(0, 0, 0, 0);
            for (uint32_t k = 0; k < n; ++k) {
                const uint32_t j = row[k];
                const double4 pj = pos[j];
                const double d[3] = {md_min_image(pi.x - pj.x, g.L[0], g.h[0]), md_min_image(pi.y - pj.y, g.L[1], g.h[1]),
                                     md_min_image(pi.z - pj.z, g.L[2], g.h[2])};
                const double r2 = md_r2_exact(d[0], d[1], d[2]);
                if (r2 < vt.pair.rc2 && r2 > 0.0) {
                    double f;
                    if (POT == VIR_DPD) {
                        const double4 vj = vel[j];
                        const double r = sqrt(r2), rinv = 1.0 / r, ww = 1.0 - r * vt.dpd_inv_rc;
                        const double rv = (d[0] * (vi.x - vj.x) + d[1] * (vi.y - vj.y) + d[2] * (vi.z - vj.z)) * rinv;
                        const double theta = md_dpd_theta(md_lane_to_tag(pi.w), md_lane_to_tag(pj.w), vt.dpd_step, vt.dpd_seed);
                        f = (vt.dpd_A * ww - vt.dpd_gamma * ww * ww * rv + vt.dpd_sr * ww * theta) * rinv;
                    } else {
                        double u;
                        f = pair_eval<(POT >= VIR_NONE ? 0 : POT)>(r2, vt.pair, u);
                    }
                    const double F[3] = {f * d[0], f * d[1], f * d[2]};
                    vir_add(w, 0.5, d, F);
                }
            }
        }
        const uint32_t t = tag[i];
        if (vt.bond_kind >= 0) {
            for (uint32_t m = bond_off[t]; m < bond_off[t + 1]; ++m) {
                const double4 pj = pos[rtag[bond_partner[m]]];
                const double d[3] = {md_min_image(pi.x - pj.x, g.L[0], g.h[0]), md_min_image(pi.y - pj.y, g.L[1], g.h[1]),
                                     md_min_image(pi.z - pj.z, g.L[2], g.h[2])};
                const double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
                if (r2 > 0.0) {
                    double f;
                    if (vt.bond_kind == MD_BOND_HARMONIC) { const double r = sqrt(r2); f = -vt.bond_k * (r - vt.bond_r0) / r; }
                    else if (vt.bond_kind == MD_BOND_FENE) f = -vt.bond_k / (1.0 - r2 / (vt.bond_r0 * vt.bond_r0));
                    else {
                        const double r = sqrt(r2);
                        if (r < vt.bond_k || !(r < vt.btab_hi)) f = nan("");
                        else {
                            const double sx = __ddiv_rn(__dsub_rn(r, vt.bond_k), vt.bond_r0);
                            uint32_t kk = (uint32_t)floor(sx);
                            kk = min(kk, vt.btab_m - 2u);
                            const double tt = __dsub_rn(sx, (double)kk);
                            const double2 a = __ldg(vt.btab + kk), b2 = __ldg(vt.btab + kk + 1);
                            f = (a.y + tt * (b2.y - a.y)) / r;
                        }
                    }
                    const double F[3] = {f * d[0], f * d[1], f * d[2]};
                    vir_add(w, 0.5, d, F);
                }
            }
        }
        if (vt.angles) {
            for (uint32_t q = angle_off[t]; q < angle_off[t + 1]; ++q) {
                double F[3], arm[3], u;
                if (angle_term(pos, rtag, angle_abc, angle_ent[q] >> 2, angle_ent[q] & 3u, g, vt.angle_k, vt.angle_theta0, F, arm, u))
                    vir_add(w, 1.0, arm, F);
            }
        }
        if (vt.dihedrals) {
            for (uint32_t q = dih_off[t]; q < dih_off[t + 1]; ++q) {
                double F[3], arm[3], u;
                if (dihedral_term(pos, rtag, dih_abcd, dih_ent[q] >> 2, dih_ent[q] & 3u, g, vt.dih, F, arm, u))
                    vir_add(w, 1.0, arm, F);
            }
        }
    }
#pragma unroll
    for (int k = 0; k < 6; ++k) sm[k * VIR_BLOCK + threadIdx.x] = w[k];
    __syncthreads();
    for (int o = VIR_BLOCK / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) {
#pragma unroll
            for (int k = 0; k < 6; ++k) sm[k * VIR_BLOCK + threadIdx.x] += sm[k * VIR_BLOCK + threadIdx.x + o];
        }
        __syncthreads();
    }
    if (threadIdx.x < 6) partial[6ull * blockIdx.x + threadIdx.x] = sm[threadIdx.x * VIR_BLOCK];
}

__global__ void __launch_bounds__(VIR_BLOCK) k_virial_final(const double *__restrict__ partial, uint32_t n_partial,
                                                            double *__restrict__ out /* [6] */)
{
    __shared__ double sm[6 * VIR_BLOCK];
    double w[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    for (uint32_t b = threadIdx.x; b < n_partial; b += VIR_BLOCK) {
#pragma unroll
        for (int k = 0; k < 6; ++k) w[k] += partial[6ull * b + k];
    }
#pragma unroll
    for (int k = 0; k < 6; ++k) sm[k * VIR_BLOCK + threadIdx.x] = w[k];
    __syncthreads();
    for (int o = VIR_BLOCK / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) {
#pragma unroll
            for (int k = 0; k < 6; ++k) sm[k * VIR_BLOCK + threadIdx.x] += sm[k * VIR_BLOCK + threadIdx.x + o];
        }
        __syncthreads();
    }
    if (threadIdx.x < 6) out[threadIdx.x] = sm[threadIdx.x * VIR_BLOCK];
}

// what: the interaction set (MD_F_LJ | MD_F_PAIR | MD_F_DPD, MD_F_BONDS, MD_F_ANGLES, MD_F_DIHEDRALS); the pair part reads the exact
// 32-bit list (the caller has decoded a tile list).  out6_host: 6 doubles on the host; synchronises.
int launch_virial(md_ctx *c, const md_step_desc *w, uint64_t step, double *out6_host)
{
    const uint32_t N = (uint32_t)c->N;
    const uint32_t nb = (N + VIR_PER_BLOCK - 1) / VIR_PER_BLOCK;
    double *buf = nullptr;
    MD_TRY(md_alloc(c, (void **)&buf, (6ull * nb + 8) * sizeof(double)));
    VirialTerms vt;
    memset(&vt, 0, sizeof(vt));
    int pot = VIR_NONE;
    if (w->flags & MD_F_LJ) {
        const double prm[4] = {w->lj_epsilon, w->lj_sigma, 0.0, 0.0};
        vt.pair = make_pair_params(c, MD_PAIR_LJ, prm, 0);
        pot = MD_PAIR_LJ;
    } else if (w->flags & MD_F_PAIR) {
        vt.pair = make_pair_params(c, w->pair_kind, w->pair_p, 0);
        pot = w->pair_kind;
    } else if (w->flags & MD_F_DPD) {
        vt.pair.rc2 = c->rc * c->rc;
        vt.dpd_inv_rc = 1.0 / c->rc;
        vt.dpd_A = w->dpd_A;
        vt.dpd_gamma = w->dpd_gamma;
        vt.dpd_sr = sqrt(2.0 * w->dpd_gamma * w->dpd_kT) / sqrt(w->dt);
        vt.dpd_step = step;
        vt.dpd_seed = w->dpd_seed;
        pot = VIR_DPD;
    }
    vt.bond_kind = ((w->flags & MD_F_BONDS) && c->n_bonds) ? w->bond_kind : -1;
    vt.bond_k = w->bond_k;
    vt.bond_r0 = w->bond_r0;
    if (vt.bond_kind == MD_BOND_TABLE) {
        vt.btab = (const double2 *)c->btab_uf;
        vt.btab_m = c->btab_m;
        vt.bond_k = c->btab_rmin;
        vt.bond_r0 = (c->btab_rmax - c->btab_rmin) / (double)(c->btab_m - 1);
        vt.btab_hi = c->btab_rmax;
    }
    vt.angles = ((w->flags & MD_F_ANGLES) && c->n_angles) ? 1 : 0;
    vt.angle_k = w->angle_k;
    vt.angle_theta0 = w->angle_theta0;
    vt.dihedrals = ((w->flags & MD_F_DIHEDRALS) && c->n_dihedrals) ? 1 : 0;
    vt.dih = DihParams{w->dihedral_k, (double)w->dihedral_sign, w->dihedral_n};
#define VIR_LAUNCH(P_)                                                                                                    \
    k_virial<P_><<<nb, VIR_BLOCK, 0, c->stream>>>(c->pos, c->vel, c->tag, c->rtag, c->nl_cnt_exp, c->nl_off, c->nl_idx,  \
                                                  c->bond_off, c->bond_partner, c->angle_off, c->angle_ent, c->angle_abc, \
                                                  c->dih_off, c->dih_ent, (const uint4 *)c->dih_abcd, c->g, vt, buf)
    switch (pot) {
    case MD_PAIR_LJ: VIR_LAUNCH(MD_PAIR_LJ); break;
    case MD_PAIR_YUKAWA: VIR_LAUNCH(MD_PAIR_YUKAWA); break;
    case MD_PAIR_GAUSSIAN: VIR_LAUNCH(MD_PAIR_GAUSSIAN); break;
    case MD_PAIR_MORSE: VIR_LAUNCH(MD_PAIR_MORSE); break;
    case MD_PAIR_TABLE: VIR_LAUNCH(MD_PAIR_TABLE); break;
    case VIR_DPD: VIR_LAUNCH(VIR_DPD); break;
    default: VIR_LAUNCH(VIR_NONE); break;
    }
#undef VIR_LAUNCH
    MD_LAUNCH_CHECK(c);
    k_virial_final<<<1, VIR_BLOCK, 0, c->stream>>>(buf, nb, buf + 6ull * nb);
    MD_LAUNCH_CHECK(c);
    MD_CUDA_CHECK(c, cudaMemcpyAsync(out6_host, buf + 6ull * nb, 6 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    const int s = md_sync(c);
    md_free(c, buf);
    return s;
}
