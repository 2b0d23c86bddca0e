/*
 * md_oracle_ext.c -- ORACLE (test infrastructure), second file: the rows of SURVEY.md 8(f) that go beyond the five
 * configurations -- virial / pressure (row 1) and further short-range force fields (row 3).  Same rules as
 * md_oracle.c: plain C, single thread, fp64, O(N^2) over all pairs or a plain loop over the bonded terms, no cells, no
 * lists, no blocking; shares no code with the CUDA path (paper_1412_3387_b200/csrc); only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline may call it.  Built with -ffp-contract=off.
 *
 * The paper names these features and prints no formula (pair potentials "Lennard-Jones, Gaussian, Morse,
 * Yukawa", bonds "harmonic, FENE", "angle, dihedral"; NPT/NPH integrators need the pressure),
 * so each function states the textbook form it takes (R31-R38).
 *
 * Pins (tests/test_oracle_ext.py; no function here is "parity unpinned"):
 *   orc_pair_forces    Yukawa/Gaussian/Morse: closed-form values, F = -dU/dr by central differences, strict cut-off,
 *                      Newton's third law, kind 0 (LJ) equal to orc_forces_lj
 *   orc_virial_pair    two-body closed form r F(r); ideal gas (no forces) P = rho kT; tr W = -3 V dU/dV by a
 *                      finite-difference box rescale; symmetric tensor; DPD equation of state (weak, statistical)
 *   orc_forces_fene    closed form, gradient, divergence at r -> r0, Newton
 *   orc_virial_bonds   two-body closed form, -3 V dU/dV
 *   orc_forces_angles  zero force at theta0, closed form for a right angle, gradient, zero net force and torque; collinear
 *                      triplets (theta = 0, pi) skipped, 1e-6 off the line finite and on the closed form
 *   orc_dihedral_angle hand-made quadruplets (cis 0, trans pi, +-pi/2 with the sign convention), quadruplets built from
 *                      internal coordinates (the angle put in comes back), invariance under rigid motion and the
 *                      periodic wrap
 *   orc_forces_dihedrals  energy k/2 (1 + s cos(n phi)) on built quadruplets for s = +-1, n = 1, 2, 3; F = -dU/dx by
 *                      central differences on all 12 coordinates; zero net force and torque; virial against
 *                      sum x_p (x) F_p; quarter-energy bookkeeping; quadruplets with three collinear particles skipped
 *   orc_langevin_u     the words of the KAT-pinned Philox for three (tag, step, seed) triples mapped by hand; range, mean,
 *                      variance 1/3, independence of components, steps and tags; not DPD's stream
 *   orc_forces_langevin  kT = 0 (pure drag), v = 0 (pure noise), gamma = 0 (off), component variance 2 gamma kT / dt;
 *                      through Sim: exact per-step decay (1 - gamma dt / m) of free particles at kT = 0 and the
 *                      closed-form stationary variance of the discrete scheme at kT > 0
 *   orc_pair_table     table values at the nodes and the straight line between two nodes; tables linear in r reproduced
 *                      at any r; nothing outside [r_min, r_max), strict at r_max; tr W = r F(r); periodic wrap; a table
 *                      of the LJ closed forms against orc_forces_lj with second-order convergence in h
 *   orc_probe_pair_forces  equal to the probes' rows of orc_pair_forces (four kinds, shifted and not) and orc_pair_table
 *   orc_bond_table     nodes and the straight line between them, NaN outside [r_min, r_max), accumulation, bond
 *                      direction, periodic wrap, tr W = r F(r); the table of a harmonic bond against
 *                      orc_forces_bonds_kind (forces exact, energies within k h^2 / 8 per bond, from above)
 */
#include <math.h>
#include <stdint.h>
#include <string.h>

/* minimum image and squared distance: restated here (R8), the two oracle files share no helper */
static double minimg(double d, double L)
{
    double h = 0.5 * L;
    if (d >= h) d -= L;
    else if (d < -h) d += L;
    return d;
}

static double sep(const double *xa, const double *xb, const double box[3], double d[3])
{
    d[0] = minimg(xa[0] - xb[0], box[0]);
    d[1] = minimg(xa[1] - xb[1], box[1]);
    d[2] = minimg(xa[2] - xb[2], box[2]);
    return (d[0] * d[0] + d[1] * d[1]) + d[2] * d[2];
}

/* ------------------------------------------------------------------------------------------------------------------
 * R31 pair potentials, pairs with r^2 < rc^2 (strict), f = -(dU/dr)/r so that F_a = f d, d = minimg(x_a - x_b):
 *   kind 0  Lennard-Jones  U = 4 p0 ((p1/r)^12 - (p1/r)^6)                      (R1; p0 = epsilon, p1 = sigma)
 *   kind 1  Yukawa         U = p0 exp(-p1 r) / r                                (p0 = epsilon, p1 = kappa)
 *   kind 2  Gaussian       U = p0 exp(-r^2 / (2 p1^2))                          (p0 = epsilon, p1 = sigma)
 *   kind 3  Morse          U = p0 (exp(-2 p1 (r - p2)) - 2 exp(-p1 (r - p2)))   (p0 = D0, p1 = alpha, p2 = r0)
 * energy_shift: U - U(rc).  Returns f and writes U (unshifted) to *u.
 * ---------------------------------------------------------------------------------------------------------------- */
static double pair_term(int kind, double r2, const double p[4], double *u)
{
    double r = sqrt(r2);
    if (kind == 0) {
        double s2 = p[1] * p[1] / r2, s6 = s2 * s2 * s2, s12 = s6 * s6;
        *u = 4.0 * p[0] * (s12 - s6);
        return 24.0 * p[0] * (2.0 * s12 - s6) / r2;
    }
    if (kind == 1) {
        double e = p[0] * exp(-p[1] * r);
        *u = e / r;
        return e * (p[1] * r + 1.0) / (r2 * r);
    }
    if (kind == 2) {
        double e = p[0] * exp(-r2 / (2.0 * p[1] * p[1]));
        *u = e;
        return e / (p[1] * p[1]);
    }
    {
        double e1 = exp(-p[1] * (r - p[2])), e2 = e1 * e1;
        *u = p[0] * (e2 - 2.0 * e1);
        return 2.0 * p[1] * p[0] * (e2 - e1) / r;
    }
}

/* force (N*3) and energy (N, may be NULL; half of each pair energy to each particle) are OVERWRITTEN */
void orc_pair_forces(const double *pos, uint64_t N, const double box[3], double rc, int kind, const double p[4],
                     int energy_shift, double *force, double *energy)
{
    double rc2 = rc * rc, uc = 0.0, d[3], u;
    if (energy_shift) (void)pair_term(kind, rc2, p, &uc);
    memset(force, 0, sizeof(double) * 3 * N);
    if (energy) memset(energy, 0, sizeof(double) * N);
    for (uint64_t a = 0; a < N; ++a)
        for (uint64_t b = a + 1; b < N; ++b) {
            double r2 = sep(pos + 3 * a, pos + 3 * b, box, d);
            if (r2 < rc2 && r2 > 0.0) {
                double f = pair_term(kind, r2, p, &u);
                for (int k = 0; k < 3; ++k) { force[3 * a + k] += f * d[k]; force[3 * b + k] -= f * d[k]; }
                if (energy) { energy[a] += 0.5 * (u - uc); energy[b] += 0.5 * (u - uc); }
            }
        }
}

/* ------------------------------------------------------------------------------------------------------------------
 * R32 virial of the pair forces: W_ab = sum over pairs of d_a F_b (F = force on the first particle of the pair, d its
 * separation from the second), order xx, yy, zz, xy, xz, yz.  The pressure follows as
 *   P = (2 K + W_xx + W_yy + W_zz) / (3 V),  K = sum 1/2 m v^2     (virial theorem; NPT/NPH of PAPER.md:63 need it).
 * ---------------------------------------------------------------------------------------------------------------- */
static void add_virial(double W[6], const double d[3], const double F[3])
{
    W[0] += d[0] * F[0]; W[1] += d[1] * F[1]; W[2] += d[2] * F[2];
    W[3] += d[0] * F[1]; W[4] += d[0] * F[2]; W[5] += d[1] * F[2];
}

void orc_virial_pair(const double *pos, uint64_t N, const double box[3], double rc, int kind, const double p[4],
                     double W[6])
{
    double rc2 = rc * rc, d[3], u, F[3];
    memset(W, 0, sizeof(double) * 6);
    for (uint64_t a = 0; a < N; ++a)
        for (uint64_t b = a + 1; b < N; ++b) {
            double r2 = sep(pos + 3 * a, pos + 3 * b, box, d);
            if (r2 < rc2 && r2 > 0.0) {
                double f = pair_term(kind, r2, p, &u);
                F[0] = f * d[0]; F[1] = f * d[1]; F[2] = f * d[2];
                add_virial(W, d, F);
            }
        }
}

/* DPD (R9): the virial of all three terms of the pair force, as orc_forces_dpd evaluates them:
 * F = fs rhat, fs = A w - gamma w^2 (rhat . v_ab) + sqrt(2 gamma kT) w theta_ab / sqrt(dt); theta_ab is orc_dpd_theta of
 * md_oracle.c (the two files are linked into one library). */
double orc_dpd_theta(uint32_t tag_a, uint32_t tag_b, uint64_t step, uint64_t seed);
void orc_virial_dpd(const double *pos, const double *vel, uint64_t N, const double box[3], double rc, double A,
                    double gamma, double kT, double dt, uint64_t step, uint64_t seed, double W[6])
{
    double rc2 = rc * rc, d[3], F[3];
    memset(W, 0, sizeof(double) * 6);
    for (uint64_t a = 0; a < N; ++a)
        for (uint64_t b = a + 1; b < N; ++b) {
            double r2 = sep(pos + 3 * a, pos + 3 * b, box, d);
            if (r2 < rc2 && r2 > 0.0) {
                double r = sqrt(r2), w = 1.0 - r / rc;
                double rh[3] = {d[0] / r, d[1] / r, d[2] / r};
                double rv = rh[0] * (vel[3 * a] - vel[3 * b]) + rh[1] * (vel[3 * a + 1] - vel[3 * b + 1]) +
                            rh[2] * (vel[3 * a + 2] - vel[3 * b + 2]);
                double fs = A * w - gamma * w * w * rv +
                            sqrt(2.0 * gamma * kT) * w * orc_dpd_theta((uint32_t)a, (uint32_t)b, step, seed) / sqrt(dt);
                F[0] = fs * rh[0]; F[1] = fs * rh[1]; F[2] = fs * rh[2];
                add_virial(W, d, F);
            }
        }
}

/* ------------------------------------------------------------------------------------------------------------------
 * R33 bonds: kind 0 harmonic U = k/2 (r - r0)^2 (R19);  kind 1 FENE U = -1/2 k r0^2 ln(1 - (r/r0)^2), r < r0
 * (Kremer-Grest form without the WCA part, which is a pair potential here): F_a = -k d / (1 - r^2/r0^2).  r >= r0 gives
 * NaN (the bond is broken: the caller's time step was too long).  force / energy are ACCUMULATED, W (may be NULL) too.
 * ---------------------------------------------------------------------------------------------------------------- */
void orc_forces_bonds_kind(const double *pos, uint64_t N, const double box[3], const uint32_t *tag_a,
                           const uint32_t *tag_b, uint64_t n_bonds, int kind, double k, double r0, double *force,
                           double *energy, double *W)
{
    (void)N;
    double d[3], F[3];
    for (uint64_t m = 0; m < n_bonds; ++m) {
        uint64_t a = tag_a[m], b = tag_b[m];
        double r2 = sep(pos + 3 * a, pos + 3 * b, box, d);
        if (!(r2 > 0.0)) continue;
        double f, u;
        if (kind == 0) {
            double r = sqrt(r2);
            f = -k * (r - r0) / r;
            u = 0.5 * k * (r - r0) * (r - r0);
        } else {
            double x = r2 / (r0 * r0);
            f = x < 1.0 ? -k / (1.0 - x) : NAN;
            u = x < 1.0 ? -0.5 * k * r0 * r0 * log(1.0 - x) : NAN;
        }
        F[0] = f * d[0]; F[1] = f * d[1]; F[2] = f * d[2];
        if (force)
            for (int c = 0; c < 3; ++c) { force[3 * a + c] += F[c]; force[3 * b + c] -= F[c]; }
        if (energy) { energy[a] += 0.5 * u; energy[b] += 0.5 * u; }
        if (W) add_virial(W, d, F);
    }
}

/* ------------------------------------------------------------------------------------------------------------------
 * R34 harmonic angles: triplet (a, b, c) with b the vertex, r1 = minimg(x_a - x_b), r2 = minimg(x_c - x_b),
 * cos(theta) = r1.r2 / (|r1| |r2|), U = k/2 (theta - theta0)^2,
 *   F_a = (k (theta - theta0) / sin(theta)) (r2 / (|r1||r2|) - cos(theta) r1 / |r1|^2),  F_c likewise with 1 <-> 2,
 *   F_b = -F_a - F_c.  sin(theta) < 1e-12 (collinear): the term is skipped.  One third of U to each particle.
 * force / energy ACCUMULATED; W (may be NULL) += r1 (x) F_a + r2 (x) F_c.
 * ---------------------------------------------------------------------------------------------------------------- */
void orc_forces_angles(const double *pos, uint64_t N, const double box[3], const uint32_t *tag_a, const uint32_t *tag_b,
                       const uint32_t *tag_c, uint64_t n_angles, double k, double theta0, double *force,
                       double *energy, double *W)
{
    (void)N;
    double r1[3], r2[3], Fa[3], Fc[3];
    for (uint64_t m = 0; m < n_angles; ++m) {
        uint64_t a = tag_a[m], b = tag_b[m], c = tag_c[m];
        double l1s = sep(pos + 3 * a, pos + 3 * b, box, r1), l2s = sep(pos + 3 * c, pos + 3 * b, box, r2);
        if (!(l1s > 0.0) || !(l2s > 0.0)) continue;
        double l1 = sqrt(l1s), l2 = sqrt(l2s);
        double cs = (r1[0] * r2[0] + r1[1] * r2[1] + r1[2] * r2[2]) / (l1 * l2);
        if (cs > 1.0) cs = 1.0;
        if (cs < -1.0) cs = -1.0;
        double sn = sqrt(1.0 - cs * cs);
        if (sn < 1e-12) continue;
        double th = acos(cs), g = k * (th - theta0) / sn;
        for (int x = 0; x < 3; ++x) {
            Fa[x] = g * (r2[x] / (l1 * l2) - cs * r1[x] / l1s);
            Fc[x] = g * (r1[x] / (l1 * l2) - cs * r2[x] / l2s);
        }
        if (force)
            for (int x = 0; x < 3; ++x) {
                force[3 * a + x] += Fa[x];
                force[3 * c + x] += Fc[x];
                force[3 * b + x] -= Fa[x] + Fc[x];
            }
        if (energy) {
            double u = 0.5 * k * (th - theta0) * (th - theta0) / 3.0;
            energy[a] += u; energy[b] += u; energy[c] += u;
        }
        if (W) { add_virial(W, r1, Fa); add_virial(W, r2, Fc); }
    }
}

/* ------------------------------------------------------------------------------------------------------------------
 * R35 dihedrals ("dihedral" named only; the brush of PAPER.md:254 needs them): quadruplet (a, b, c, d),
 * F = minimg(x_a - x_b), G = minimg(x_b - x_c), H = minimg(x_d - x_c), A = F x G, B = H x G,
 * phi = atan2(((B x A).G)/|G|, A.B) in (-pi, pi] (0 = cis, pi = trans), U = k/2 (1 + s cos(n phi)), s = +-1, n = 1, 2, 3, ...
 * (the periodic "harmonic" dihedral of HOOMD-blue).  Gradient of phi (Blondel & Karplus 1996):
 *   dphi/dx_a = -|G|/|A|^2 A,   dphi/dx_d = +|G|/|B|^2 B,
 *   dphi/dx_b = +|G|/|A|^2 A + (F.G)/(|A|^2 |G|) A - (H.G)/(|B|^2 |G|) B,
 *   dphi/dx_c = -|G|/|B|^2 B - (F.G)/(|A|^2 |G|) A + (H.G)/(|B|^2 |G|) B,
 * force on particle p = -dU/dphi dphi/dx_p, dU/dphi = -k/2 s n sin(n phi).  Collinear triplets (|A|^2 or |B|^2 < 1e-24
 * |G|^4) are skipped.  One quarter of U to each particle.  force / energy ACCUMULATED; W (may be NULL) += sum over a, c, d
 * of (x_p - x_b) (x) F_p (minimum-image arms).
 * ---------------------------------------------------------------------------------------------------------------- */
static void cross3(const double u[3], const double v[3], double w[3])
{
    w[0] = u[1] * v[2] - u[2] * v[1];
    w[1] = u[2] * v[0] - u[0] * v[2];
    w[2] = u[0] * v[1] - u[1] * v[0];
}

static double dot3(const double u[3], const double v[3]) { return u[0] * v[0] + u[1] * v[1] + u[2] * v[2]; }

/* the angle itself (also exported for the pins): radians in (-pi, pi] */
double orc_dihedral_angle(const double *xa, const double *xb, const double *xc, const double *xd, const double box[3])
{
    double F[3], G[3], H[3], A[3], B[3], C[3];
    (void)sep(xa, xb, box, F);
    (void)sep(xb, xc, box, G);
    (void)sep(xd, xc, box, H);
    cross3(F, G, A);
    cross3(H, G, B);
    cross3(B, A, C);
    return atan2(dot3(C, G) / sqrt(dot3(G, G)), dot3(A, B));
}

void orc_forces_dihedrals(const double *pos, uint64_t N, const double box[3], const uint32_t *tag_a, const uint32_t *tag_b,
                          const uint32_t *tag_c, const uint32_t *tag_d, uint64_t n_dih, double k, int s, int n,
                          double *force, double *energy, double *W)
{
    (void)N;
    double F[3], G[3], H[3], A[3], B[3], C[3];
    for (uint64_t m = 0; m < n_dih; ++m) {
        uint64_t a = tag_a[m], b = tag_b[m], c = tag_c[m], d = tag_d[m];
        (void)sep(pos + 3 * a, pos + 3 * b, box, F);
        double g2 = sep(pos + 3 * b, pos + 3 * c, box, G);
        (void)sep(pos + 3 * d, pos + 3 * c, box, H);
        cross3(F, G, A);
        cross3(H, G, B);
        double a2 = dot3(A, A), b2 = dot3(B, B);
        if (!(g2 > 0.0) || a2 < 1e-24 * g2 * g2 || b2 < 1e-24 * g2 * g2) continue;
        double gl = sqrt(g2);
        cross3(B, A, C);
        double phi = atan2(dot3(C, G) / gl, dot3(A, B));
        double dU = -0.5 * k * (double)s * (double)n * sin((double)n * phi);
        double fg = dot3(F, G), hg = dot3(H, G);
        double Fa[3], Fb[3], Fc[3], Fd[3];
        for (int x = 0; x < 3; ++x) {
            double ga = -gl / a2 * A[x], gd = gl / b2 * B[x];
            double gb = gl / a2 * A[x] + fg / (a2 * gl) * A[x] - hg / (b2 * gl) * B[x];
            double gc = -gl / b2 * B[x] - fg / (a2 * gl) * A[x] + hg / (b2 * gl) * B[x];
            Fa[x] = -dU * ga; Fb[x] = -dU * gb; Fc[x] = -dU * gc; Fd[x] = -dU * gd;
        }
        if (force)
            for (int x = 0; x < 3; ++x) {
                force[3 * a + x] += Fa[x]; force[3 * b + x] += Fb[x];
                force[3 * c + x] += Fc[x]; force[3 * d + x] += Fd[x];
            }
        if (energy) {
            double u = 0.25 * 0.5 * k * (1.0 + (double)s * cos((double)n * phi));
            energy[a] += u; energy[b] += u; energy[c] += u; energy[d] += u;
        }
        if (W) {
            double rc_[3] = {-G[0], -G[1], -G[2]}, rd[3] = {H[0] - G[0], H[1] - G[1], H[2] - G[2]};
            add_virial(W, F, Fa);
            add_virial(W, rc_, Fc);
            add_virial(W, rd, Fd);
        }
    }
}

/* ------------------------------------------------------------------------------------------------------------------
 * R36 Langevin thermostat ("Brownian (or Langevin) dynamics"; "from the same
 * counter-based hash").  A one-body force evaluated with the other forces of the step, i.e. at the velocities after
 * half 1 like the DPD drag (R15), and integrated by the velocity-Verlet halves:
 *   F_a += -gamma v_a + sqrt(6 gamma kT / dt) (u_x, u_y, u_z),
 *   u uniform on (-1, 1) (variance 1/3, so each component of the random force has variance 2 gamma kT / dt),
 *   (X0, X1, X2, .) = Philox4x32-10(counter = (tag, 0xffffffff, step lo, step hi), key = (seed lo, seed hi)),
 *   u_k = 2 (X_k + 0.5) 2^-32 - 1.
 * The second counter word 0xffffffff keeps the stream apart from the DPD pair stream (min tag, max tag, ...), whose
 * second word is a tag < N <= 2^32 - 1.  No energy, no virial (a one-body force).  force ACCUMULATED.
 * ---------------------------------------------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

void orc_langevin_u(uint32_t tag, uint64_t step, uint64_t seed, double u[3])
{
    uint32_t ctr[4], key[2], out[4];
    ctr[0] = tag;
    ctr[1] = 0xffffffffu;
    ctr[2] = (uint32_t)(step & 0xffffffffu);
    ctr[3] = (uint32_t)(step >> 32);
    key[0] = (uint32_t)(seed & 0xffffffffu);
    key[1] = (uint32_t)(seed >> 32);
    orc_philox4x32_10(ctr, key, out);
    for (int k = 0; k < 3; ++k) u[k] = 2.0 * (((double)out[k] + 0.5) * (1.0 / 4294967296.0)) - 1.0;
}

void orc_forces_langevin(const double *vel, uint64_t N, double gamma, double kT, double dt, uint64_t step, uint64_t seed,
                         double *force)
{
    double amp = sqrt(6.0 * gamma * kT / dt), u[3];
    for (uint64_t a = 0; a < N; ++a) {
        orc_langevin_u((uint32_t)a, step, seed, u);
        for (int k = 0; k < 3; ++k) force[3 * a + k] += -gamma * vel[3 * a + k] + amp * u[k];
    }
}

/* ------------------------------------------------------------------------------------------------------------------
 * R37 tabulated pair potential ("tabulated potentials"; no formula).  The caller gives U_k and F_k = -dU/dr
 * at r_k = r_min + k h, k = 0 .. M-1, h = (r_max - r_min) / (M - 1); both are interpolated LINEARLY:
 *   s = (r - r_min) / h,  k = floor(s) (clamped to M-2),  t = s - k,
 *   U(r) = U_k + t (U_{k+1} - U_k),   F(r) = F_k + t (F_{k+1} - F_k),   force on a = F(r) d / r, d = minimg(x_a - x_b).
 * Pairs with r_min <= r < r_max contribute (r^2 < r_max^2 strict, like every cut-off here; a pair closer than r_min is
 * outside the table and contributes nothing).  No energy shift: the table is what the caller wants.
 * force / energy (may be NULL) OVERWRITTEN; W (may be NULL) = sum over pairs of d (x) F, overwritten.
 * ---------------------------------------------------------------------------------------------------------------- */
void orc_pair_table(const double *pos, uint64_t N, const double box[3], double r_min, double r_max, uint64_t M,
                    const double *U, const double *F, double *force, double *energy, double *W)
{
    double h = (r_max - r_min) / (double)(M - 1), d[3], Fv[3];
    if (force) memset(force, 0, sizeof(double) * 3 * N);
    if (energy) memset(energy, 0, sizeof(double) * N);
    if (W) memset(W, 0, sizeof(double) * 6);
    for (uint64_t a = 0; a < N; ++a)
        for (uint64_t b = a + 1; b < N; ++b) {
            double r2 = sep(pos + 3 * a, pos + 3 * b, box, d);
            if (!(r2 < r_max * r_max)) continue;
            double r = sqrt(r2);
            if (r < r_min) continue;
            double s = (r - r_min) / h;
            uint64_t k = (uint64_t)floor(s);
            if (k > M - 2) k = M - 2;
            double t = s - (double)k;
            double u = U[k] + t * (U[k + 1] - U[k]);
            double f = (F[k] + t * (F[k + 1] - F[k])) / r;
            for (int x = 0; x < 3; ++x) Fv[x] = f * d[x];
            if (force)
                for (int x = 0; x < 3; ++x) { force[3 * a + x] += Fv[x]; force[3 * b + x] -= Fv[x]; }
            if (energy) { energy[a] += 0.5 * u; energy[b] += 0.5 * u; }
            if (W) add_virial(W, d, Fv);
        }
}

/* ------------------------------------------------------------------------------------------------------------------
 * R38 tabulated bonds ("harmonic, FENE and tabulated bonds"; no formula).  Same table and the same linear
 * interpolation as the tabulated pair potential (R37), evaluated on the bond list:
 *   U_k, F_k = -dU/dr at r_k = r_min + k h, h = (r_max - r_min) / (M - 1);  s = (r - r_min) / h, k = floor(s) clamped to
 *   M - 2, t = s - k;  U(r) = U_k + t (U_{k+1} - U_k), F(r) = F_k + t (F_{k+1} - F_k);  F_a += F(r) d / r, F_b -= same,
 *   d = minimg(x_a - x_b); half of U(r) to each particle.
 * A bond with r < r_min or r >= r_max has left its table: NaN (like the FENE bond beyond r0, R33).
 * force / energy / W (each may be NULL) are ACCUMULATED.
 * ---------------------------------------------------------------------------------------------------------------- */
void orc_bond_table(const double *pos, uint64_t N, const double box[3], const uint32_t *tag_a, const uint32_t *tag_b,
                    uint64_t n_bonds, double r_min, double r_max, uint64_t M, const double *U, const double *F,
                    double *force, double *energy, double *W)
{
    (void)N;
    double h = (r_max - r_min) / (double)(M - 1), d[3], Fv[3];
    for (uint64_t m = 0; m < n_bonds; ++m) {
        uint64_t a = tag_a[m], b = tag_b[m];
        double r2 = sep(pos + 3 * a, pos + 3 * b, box, d);
        if (!(r2 > 0.0)) continue;
        double r = sqrt(r2), f, u;
        if (r < r_min || !(r < r_max)) {
            f = NAN; u = NAN;
        } else {
            double s = (r - r_min) / h;
            uint64_t k = (uint64_t)floor(s);
            if (k > M - 2) k = M - 2;
            double t = s - (double)k;
            u = U[k] + t * (U[k + 1] - U[k]);
            f = (F[k] + t * (F[k + 1] - F[k])) / r;
        }
        for (int x = 0; x < 3; ++x) Fv[x] = f * d[x];
        if (force)
            for (int x = 0; x < 3; ++x) { force[3 * a + x] += Fv[x]; force[3 * b + x] -= Fv[x]; }
        if (energy) { energy[a] += 0.5 * u; energy[b] += 0.5 * u; }
        if (W) add_virial(W, d, Fv);
    }
}

/* ------------------------------------------------------------------------------------------------------------------
 * Probe rows of the pair potentials (the O9 idea of md_oracle.c for R31 and R37): force and energy of M probe particles,
 * each against ALL N particles by brute force -- O(M N), usable at the full sizes where the O(N^2) routines are not.
 * Pinned as the rows of orc_pair_forces / orc_pair_table on a small system (tests/test_oracle_ext.py).
 * kind 0..3: R31 with parameters p; kind 4: the table (r_min, r_max, M_tab, U, F) of R37, rc ignored.
 * ---------------------------------------------------------------------------------------------------------------- */
void orc_probe_pair_forces(const double *pos, uint64_t N, const double box[3], double rc, int kind, const double p[4],
                           int energy_shift, double r_min, double r_max, uint64_t M_tab, const double *U, const double *F,
                           const uint32_t *probes, uint64_t M, double *force, double *energy)
{
    double rc2 = kind == 4 ? r_max * r_max : rc * rc, uc = 0.0, d[3], u;
    double h = kind == 4 ? (r_max - r_min) / (double)(M_tab - 1) : 0.0;
    if (energy_shift && kind != 4) (void)pair_term(kind, rc2, p, &uc);
    for (uint64_t q = 0; q < M; ++q) {
        uint64_t a = probes[q];
        double f3[3] = {0.0, 0.0, 0.0}, e = 0.0;
        for (uint64_t b = 0; b < N; ++b) {
            if (b == a) continue;
            double r2 = sep(pos + 3 * a, pos + 3 * b, box, d);
            if (!(r2 < rc2) || !(r2 > 0.0)) continue;
            double f;
            if (kind == 4) {
                double r = sqrt(r2);
                if (r < r_min) continue;
                double s = (r - r_min) / h;
                uint64_t k = (uint64_t)floor(s);
                if (k > M_tab - 2) k = M_tab - 2;
                double t = s - (double)k;
                u = U[k] + t * (U[k + 1] - U[k]);
                f = (F[k] + t * (F[k + 1] - F[k])) / r;
            } else {
                f = pair_term(kind, r2, p, &u);
            }
            for (int x = 0; x < 3; ++x) f3[x] += f * d[x];
            e += 0.5 * (u - uc);
        }
        force[3 * q] = f3[0]; force[3 * q + 1] = f3[1]; force[3 * q + 2] = f3[2];
        if (energy) energy[q] = e;
    }
}
