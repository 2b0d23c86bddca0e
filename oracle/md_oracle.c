/*
 * md_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, single-threaded, fp64, obviously-correct statement of what the MD hot path of
 * Glaser et al., "Strong scaling of general-purpose molecular dynamics simulations on GPUs"
 * (arXiv:1412.3387; /root/reference/PAPER.md) computes on one GPU.  It shares NO code with the CUDA
 * path under paper_1412_3387_b200/csrc/ (no headers, helpers, tables or constants) and neither side
 * includes or imports the other.  Only tests/, __graft_entry__.smoke() and the cpu_baseline /
 * --impl reference legs of bench.py may load this library.
 *
 * No cells, no neighbour lists, no blocking, no reordering: every quantity is its plain definition
 * over all pairs of particles, O(N^2), in tag order (tag == array index).
 * Build: gcc -O2 -ffp-contract=off -fno-fast-math (see oracle/build.py) so that the decision
 * arithmetic (r^2 < r_list^2, cell index) is plain IEEE-754 double without FMA contraction.
 *
 * The paper prints no formula for LJ, DPD, harmonic bonds or velocity-Verlet (it names them,
 * PAPER.md:63, and cites refs [1], [41], [42]); the forms below are the textbook definitions as read
 * in DESIGN.md "Readings" (R1..R27), each function says which.
 *
 * Pins (tests/test_oracle_*.py, all run without a GPU):
 *   orc_philox4x32_10     known-answer vectors (tests/golden/philox4x32_10_kat.txt)
 *   orc_forces_lj         F(2^(1/6) sigma)=0, U=-eps; closed-form U(rc); F=-dU/dr; FCC shell sums; sum F = 0
 *   orc_neighbor_pairs    scipy cKDTree(boxsize) pairs; vectorised numpy brute force; FCC shell counts
 *   orc_cell_assign       geometric containment; exact-face inputs; histogram = N
 *   orc_needs_rebuild     free-flight closed form
 *   orc_forces_dpd        conservative energy U=A rc (1-r/rc)^2/2 derivative; one-step drag decay;
 *                         theta symmetry/moments; sum F = 0
 *   orc_forces_bonds      two-body closed form; F=-dU/dr; sum F = 0
 *   orc_vv_half1/2        free flight with wraps; discrete harmonic frequency; time reversal; dt^2 scaling;
 *                         NVE drift bound
 *   orc_probe_*           equal to the corresponding rows of the full O(N^2) routines
 * No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------------------------------------
 * O8 minimum image ("the usual minimum image convention"; R8):
 * positions are wrapped into [-L/2, L/2), so one correction per axis suffices.
 * ---------------------------------------------------------------------------------------------- */
static double minimg(double d, double L)
{
    double h = 0.5 * L;
    if (d >= h) d -= L;
    else if (d < -h) d += L;
    return d;
}

/* squared minimum-image distance, evaluated as (dx*dx + dy*dy) + dz*dz, no FMA (R2) */
static double dist2(const double *xa, const double *xb, const double box[3], double d[3])
{
    d[0] = minimg(xa[0] - xb[0], box[0]);
    d[1] = minimg(xa[1] - xb[1], box[1]);
    d[2] = minimg(xa[2] - xb[2], box[2]);
    return (d[0] * d[0] + d[1] * d[1]) + d[2] * d[2];
}

/* ------------------------------------------------------------------------------------------------
 * Wrap positions into the box once (md_set_state does the same; R4).  image may be NULL.
 * ---------------------------------------------------------------------------------------------- */
void orc_wrap(double *pos, int32_t *image, uint64_t N, const double box[3])
{
    for (uint64_t i = 0; i < N; ++i)
        for (int a = 0; a < 3; ++a) {
            double L = box[a], h = 0.5 * L, x = pos[3 * i + a];
            int32_t im = 0;
            while (x >= h) { x -= L; ++im; }
            while (x < -h) { x += L; --im; }
            pos[3 * i + a] = x;
            if (image) image[3 * i + a] += im;
        }
}

/* ------------------------------------------------------------------------------------------------
 * O1 cell assignment ("Look up cell neighbors", Fig. 4 step 1; the cell width must be
 * >= r_cut + r_buff so that the 27-cell stencil holds every list neighbour).
 *   n_c = max(1, floor(L / r_list));  f = (x - lo)/L, lo = -L/2;  c = (int)(f * n_c), c == n_c -> n_c-1
 *   id  = cx + n_cx (cy + n_cy cz)
 * ---------------------------------------------------------------------------------------------- */
void orc_cell_dims(const double box[3], double r_list, uint32_t dims[3])
{
    for (int a = 0; a < 3; ++a) {
        double n = floor(box[a] / r_list);
        if (n < 1.0) n = 1.0;
        dims[a] = (uint32_t)n;
    }
}

void orc_cell_assign(const double *pos, uint64_t N, const double box[3], double r_list,
                     uint32_t *cell_of, uint32_t dims[3])
{
    orc_cell_dims(box, r_list, dims);
    for (uint64_t i = 0; i < N; ++i) {
        uint32_t c[3];
        for (int a = 0; a < 3; ++a) {
            double lo = -0.5 * box[a];
            double f = (pos[3 * i + a] - lo) / box[a];
            int64_t k = (int64_t)(f * (double)dims[a]);
            if (k >= (int64_t)dims[a]) k = (int64_t)dims[a] - 1;
            if (k < 0) k = 0;
            c[a] = (uint32_t)k;
        }
        cell_of[i] = c[0] + dims[0] * (c[1] + dims[1] * c[2]);
    }
}

/* ------------------------------------------------------------------------------------------------
 * O2 neighbour set at build time (Fig. 4 step 3 "r < r_cut", with the list radius
 * r_list = r_cut + r_buff of PAPER.md:79): all unordered tag pairs {a<b} with
 * |minimg(x_a - x_b)|^2 < r_list^2 (strict).  Emitted in (a, b) lexicographic order.
 * pairs may be NULL (count only).  Returns the number of pairs found (may exceed cap; only the
 * first cap pairs are stored).
 * ---------------------------------------------------------------------------------------------- */
uint64_t orc_neighbor_pairs(const double *pos, uint64_t N, const double box[3], double r_list,
                            uint32_t *pairs, uint64_t cap)
{
    double rl2 = r_list * r_list, d[3];
    uint64_t n = 0;
    for (uint64_t a = 0; a < N; ++a)
        for (uint64_t b = a + 1; b < N; ++b)
            if (dist2(pos + 3 * a, pos + 3 * b, box, d) < rl2) {
                if (pairs && n < cap) { pairs[2 * n] = (uint32_t)a; pairs[2 * n + 1] = (uint32_t)b; }
                ++n;
            }
    return n;
}

/* ------------------------------------------------------------------------------------------------
 * O3 rebuild trigger ("Neighbor list builds occur when particles move more than half of the buffer
 * length"): 1 iff some i has |minimg(x_i - xref_i)|^2 > (r_buff/2)^2 (strict).
 * ---------------------------------------------------------------------------------------------- */
int orc_needs_rebuild(const double *pos, const double *pos_ref, uint64_t N, const double box[3], double r_buff)
{
    double t = 0.5 * r_buff, t2 = t * t, d[3];
    for (uint64_t i = 0; i < N; ++i)
        if (dist2(pos + 3 * i, pos_ref + 3 * i, box, d) > t2) return 1;
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * O4 truncated Lennard-Jones 12-6 (named PAPER.md:63, :210, :300; formula = textbook, R1):
 *   pair with r^2 < rc^2:  s2 = sigma^2/r^2, s6 = s2^3, s12 = s6^2
 *   f = 24 eps (2 s12 - s6) / r^2 ;  F_a += f d, F_b -= f d, d = minimg(x_a - x_b)
 *   U = 4 eps (s12 - s6) - shift * U_c,  U_c = 4 eps ((sigma/rc)^12 - (sigma/rc)^6); half to each.
 * force (N*3) and energy (N, may be NULL) are OVERWRITTEN.
 * ---------------------------------------------------------------------------------------------- */
static double lj_pair(double r2, double eps, double sigma, double *u)
{
    double s2 = sigma * sigma / r2, s6 = s2 * s2 * s2, s12 = s6 * s6;
    *u = 4.0 * eps * (s12 - s6);
    return 24.0 * eps * (2.0 * s12 - s6) / r2;
}

void orc_forces_lj(const double *pos, uint64_t N, const double box[3], double rc, double eps, double sigma,
                   int energy_shift, double *force, double *energy)
{
    double rc2 = rc * rc, uc = 0.0, d[3], u;
    if (energy_shift) (void)lj_pair(rc2, eps, sigma, &uc);
    memset(force, 0, sizeof(double) * 3 * N);
    if (energy) memset(energy, 0, sizeof(double) * N);
    for (uint64_t a = 0; a < N; ++a)
        for (uint64_t b = a + 1; b < N; ++b) {
            double r2 = dist2(pos + 3 * a, pos + 3 * b, box, d);
            if (r2 < rc2) {
                double f = lj_pair(r2, eps, sigma, &u);
                for (int k = 0; k < 3; ++k) { force[3 * a + k] += f * d[k]; force[3 * b + k] -= f * d[k]; }
                if (energy) { energy[a] += 0.5 * (u - uc); energy[b] += 0.5 * (u - uc); }
            }
        }
}

/* ------------------------------------------------------------------------------------------------
 * Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), the counter-based hash behind the per-pair DPD
 * random number ("per-particle-pair random number generators [41]", the paper names no
 * hash; R14).  Written from the published round function:
 *   (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)), 10 rounds,
 *   key += (W0, W1) between rounds.
 * ---------------------------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* theta_ab: uniform on (-sqrt3, sqrt3), unit variance (R13), keyed on
 * (min tag, max tag, step, seed): counter = (min, max, step lo, step hi), key = (seed lo, seed hi);
 * u = (X0 + 0.5) 2^-32 is exact in fp64. */
double orc_dpd_theta(uint32_t tag_a, uint32_t tag_b, uint64_t step, uint64_t seed)
{
    uint32_t ctr[4], key[2], out[4];
    ctr[0] = tag_a < tag_b ? tag_a : tag_b;
    ctr[1] = tag_a < tag_b ? tag_b : tag_a;
    ctr[2] = (uint32_t)(step & 0xffffffffu);
    ctr[3] = (uint32_t)(step >> 32);
    key[0] = (uint32_t)(seed & 0xffffffffu);
    key[1] = (uint32_t)(seed >> 32);
    orc_philox4x32_10(ctr, key, out);
    double u = ((double)out[0] + 0.5) * (1.0 / 4294967296.0);
    return sqrt(3.0) * (2.0 * u - 1.0);
}

/* ------------------------------------------------------------------------------------------------
 * O5 DPD pair force (named PAPER.md:63; drag needs neighbour velocities and the random term needs
 * global particle IDs; formula = Groot-Warren, R9):
 *   pair with 0 < r < rc:  w = 1 - r/rc, rhat = d/r, d = minimg(x_a - x_b)
 *   F = [A w - gamma w^2 (rhat . (v_a - v_b)) + sqrt(2 gamma kT) w theta_ab / sqrt(dt)] rhat
 *   on a, -F on b.  force is OVERWRITTEN.
 * ---------------------------------------------------------------------------------------------- */
static double dpd_pair(const double d[3], double r2, const double *va, const double *vb, double rc, double A,
                       double gamma, double kT, double dt, uint32_t ta, uint32_t tb, uint64_t step,
                       uint64_t seed, double rhat[3])
{
    double r = sqrt(r2), w = 1.0 - r / rc;
    rhat[0] = d[0] / r; rhat[1] = d[1] / r; rhat[2] = d[2] / r;
    double rv = rhat[0] * (va[0] - vb[0]) + rhat[1] * (va[1] - vb[1]) + rhat[2] * (va[2] - vb[2]);
    double theta = orc_dpd_theta(ta, tb, step, seed);
    return A * w - gamma * w * w * rv + sqrt(2.0 * gamma * kT) * w * theta / sqrt(dt);
}

void orc_forces_dpd(const double *pos, const double *vel, uint64_t N, const double box[3], double rc, double A,
                    double gamma, double kT, double dt, uint64_t step, uint64_t seed, double *force)
{
    double rc2 = rc * rc, d[3], rhat[3];
    memset(force, 0, sizeof(double) * 3 * N);
    for (uint64_t a = 0; a < N; ++a)
        for (uint64_t b = a + 1; b < N; ++b) {
            double r2 = dist2(pos + 3 * a, pos + 3 * b, box, d);
            if (r2 < rc2 && r2 > 0.0) {
                double f = dpd_pair(d, r2, vel + 3 * a, vel + 3 * b, rc, A, gamma, kT, dt, (uint32_t)a,
                                    (uint32_t)b, step, seed, rhat);
                for (int k = 0; k < 3; ++k) { force[3 * a + k] += f * rhat[k]; force[3 * b + k] -= f * rhat[k]; }
            }
        }
}

/* ------------------------------------------------------------------------------------------------
 * O6 harmonic bonds (named PAPER.md:63; a bond is an unordered pair of particle IDs, PAPER.md:147;
 * U = k/2 (r - r0)^2, R19):  F_a += -k (r - r0) d/r, F_b -= same, d = minimg(x_a - x_b);
 * r == 0 gives zero force.  force (and energy if not NULL, half to each end) are ACCUMULATED.
 * ---------------------------------------------------------------------------------------------- */
void orc_forces_bonds(const double *pos, uint64_t N, const double box[3], const uint32_t *tag_a,
                      const uint32_t *tag_b, uint64_t n_bonds, double k, double r0, double *force, double *energy)
{
    (void)N;
    double d[3];
    for (uint64_t m = 0; m < n_bonds; ++m) {
        uint64_t a = tag_a[m], b = tag_b[m];
        double r2 = dist2(pos + 3 * a, pos + 3 * b, box, d);
        if (r2 > 0.0) {
            double r = sqrt(r2), f = -k * (r - r0) / r;
            for (int c = 0; c < 3; ++c) { force[3 * a + c] += f * d[c]; force[3 * b + c] -= f * d[c]; }
            if (energy) { double u = 0.5 * k * (r - r0) * (r - r0); energy[a] += 0.5 * u; energy[b] += 0.5 * u; }
        }
    }
}

/* ------------------------------------------------------------------------------------------------
 * O7 velocity-Verlet, NVE ("NVE (constant energy) ... implement the Velocity-Verlet", PAPER.md:63;
 * DESIGN.md R7).  half 1: v += (dt/2) F/m; x += dt v; wrap (x >= L/2: x -= L, image++;
 * x < -L/2: x += L, image--).  half 2: v += (dt/2) F/m.  mass NULL means m = 1.
 * ---------------------------------------------------------------------------------------------- */
void orc_vv_half1(double *pos, double *vel, int32_t *image, const double *force, const double *mass,
                  uint64_t N, const double box[3], double dt)
{
    for (uint64_t i = 0; i < N; ++i) {
        double m = mass ? mass[i] : 1.0;
        for (int a = 0; a < 3; ++a) {
            double v = vel[3 * i + a] + (0.5 * dt) * force[3 * i + a] / m;
            double x = pos[3 * i + a] + dt * v;
            double L = box[a], h = 0.5 * L;
            if (x >= h) { x -= L; if (image) image[3 * i + a] += 1; }
            else if (x < -h) { x += L; if (image) image[3 * i + a] -= 1; }
            vel[3 * i + a] = v;
            pos[3 * i + a] = x;
        }
    }
}

void orc_vv_half2(double *vel, const double *force, const double *mass, uint64_t N, double dt)
{
    for (uint64_t i = 0; i < N; ++i) {
        double m = mass ? mass[i] : 1.0;
        for (int a = 0; a < 3; ++a) vel[3 * i + a] += (0.5 * dt) * force[3 * i + a] / m;
    }
}

/* ------------------------------------------------------------------------------------------------
 * O9 probe-row mode: the same definitions restricted to pairs (probe, any of N), O(M N), still no
 * cells.  Needed because O(N^2) is infeasible beyond N ~ 1e5.
 * ---------------------------------------------------------------------------------------------- */

/* neighbour tags of each probe (ascending), at most row_stride stored per probe; counts = true count */
void orc_probe_nlist(const double *pos, uint64_t N, const double box[3], double r_list, const uint32_t *probes,
                     uint64_t M, uint32_t *counts, uint32_t *nbrs, uint64_t row_stride)
{
    double rl2 = r_list * r_list, d[3];
    for (uint64_t p = 0; p < M; ++p) {
        uint64_t a = probes[p];
        uint32_t n = 0;
        for (uint64_t b = 0; b < N; ++b) {
            if (b == a) continue;
            /* same operand order as O2: lower tag first (the square is order-independent anyway) */
            double r2 = a < b ? dist2(pos + 3 * a, pos + 3 * b, box, d) : dist2(pos + 3 * b, pos + 3 * a, box, d);
            if (r2 < rl2) {
                if (nbrs && n < row_stride) nbrs[p * row_stride + n] = (uint32_t)b;
                ++n;
            }
        }
        counts[p] = n;
    }
}

void orc_probe_forces_lj(const double *pos, uint64_t N, const double box[3], double rc, double eps, double sigma,
                         int energy_shift, const uint32_t *probes, uint64_t M, double *force, double *energy)
{
    double rc2 = rc * rc, uc = 0.0, d[3], u;
    if (energy_shift) (void)lj_pair(rc2, eps, sigma, &uc);
    for (uint64_t p = 0; p < M; ++p) {
        uint64_t a = probes[p];
        double f3[3] = {0.0, 0.0, 0.0}, e = 0.0;
        for (uint64_t b = 0; b < N; ++b) {
            if (b == a) continue;
            double r2 = dist2(pos + 3 * a, pos + 3 * b, box, d);
            if (r2 < rc2) {
                double f = lj_pair(r2, eps, sigma, &u);
                for (int k = 0; k < 3; ++k) f3[k] += f * d[k];
                e += 0.5 * (u - uc);
            }
        }
        force[3 * p] = f3[0]; force[3 * p + 1] = f3[1]; force[3 * p + 2] = f3[2];
        if (energy) energy[p] = e;
    }
}

void orc_probe_forces_dpd(const double *pos, const double *vel, uint64_t N, const double box[3], double rc,
                          double A, double gamma, double kT, double dt, uint64_t step, uint64_t seed,
                          const uint32_t *probes, uint64_t M, double *force)
{
    double rc2 = rc * rc, d[3], rhat[3];
    for (uint64_t p = 0; p < M; ++p) {
        uint64_t a = probes[p];
        double f3[3] = {0.0, 0.0, 0.0};
        for (uint64_t b = 0; b < N; ++b) {
            if (b == a) continue;
            double r2 = dist2(pos + 3 * a, pos + 3 * b, box, d);
            if (r2 < rc2 && r2 > 0.0) {
                double f = dpd_pair(d, r2, vel + 3 * a, vel + 3 * b, rc, A, gamma, kT, dt, (uint32_t)a,
                                    (uint32_t)b, step, seed, rhat);
                for (int k = 0; k < 3; ++k) f3[k] += f * rhat[k];
            }
        }
        force[3 * p] = f3[0]; force[3 * p + 1] = f3[1]; force[3 * p + 2] = f3[2];
    }
}
