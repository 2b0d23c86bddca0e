// integrate.cu -- S6 velocity-Verlet NVE (R7) and S3 displacement check.
#include <algorithm>

#include "md_device.cuh"

// half 1: v += (dt/2) F/m ; x += dt v ; wrap ; displacement since the last binning vs (r_buff/2)^2.
// FUSED: the second half-kick of the previous step is applied first (same force, same operations in the same order
// as k_half2 followed by k_half1, so the result is bit-identical to the two separate launches).
// The largest squared displacement of the step goes to flags->max_d2[slot] (float bits; the host uses it to
// predict the step at which the criterion will fire, see md_step); the other slot is cleared for the next step.
// NVT (R30): v <- (v + kick) / (1 + (dt/2) xi) in half 1, v <- v + (dt/2)(F/m - xi v) in half 2, xi read from
// nvt[0]; the fused launch applies half 2 and the next half 1 with the same xi (the one the thermostat update left).
template <bool FUSED, bool NVT>
__global__ void __launch_bounds__(MD_HALF1_MAX_BLOCK, 6) k_half1(double4 *__restrict__ pos, double4 *__restrict__ vel, const double4 *__restrict__ force,
                        int *__restrict__ image, const double *__restrict__ pos_ref,
                        const uint32_t *__restrict__ cell_lin, float4 *__restrict__ rel, Geom g, double dt,
                        double half_dt, double thr2, double danger2, DevFlags *flags, int slot,
                        const double *__restrict__ nvt, Gate gate, unsigned int at_val)
{
    if (md_gate_closed(gate)) return;
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    float d2f = 0.f;
    unsigned fire = 0u;  // bit 0: moved more than r_buff / 2 since the binning; bit 1: more than r_buff (a pair may have been missed)
    const double xi = NVT ? nvt[0] : 0.0;
    const double denom = __dadd_rn(1.0, __dmul_rn(half_dt, xi));
    if (i < g.N) {
        double4 p = pos[i];
        double4 v = vel[i];
        const double4 f = force[i];
        const double m = v.w;
        double x[3] = {p.x, p.y, p.z};
        double u[3] = {v.x, v.y, v.z};
        const double ff[3] = {f.x, f.y, f.z};
        double d2 = 0.0;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            // same operation order as the definition: v + ((dt/2) F)/m ; x + dt v   (no FMA: positions parity 1e-12
            // does not need it, but it keeps single steps bit-comparable with a plain CPU evaluation)
            const double kick = __ddiv_rn(__dmul_rn(half_dt, ff[a]), m);
            if (NVT) {
                if (FUSED) u[a] = __dadd_rn(u[a], __dmul_rn(half_dt, __dsub_rn(__ddiv_rn(ff[a], m), __dmul_rn(xi, u[a]))));
                u[a] = __ddiv_rn(__dadd_rn(u[a], kick), denom);
            } else {
                if (FUSED) u[a] = __dadd_rn(u[a], kick);
                u[a] = __dadd_rn(u[a], kick);
            }
            double xn = __dadd_rn(x[a], __dmul_rn(dt, u[a]));
            if (xn >= g.h[a]) { xn = __dsub_rn(xn, g.L[a]); image[3ull * i + a] += 1; }
            else if (xn < -g.h[a]) { xn = __dadd_rn(xn, g.L[a]); image[3ull * i + a] -= 1; }
            x[a] = xn;
            const double d = md_min_image(__dsub_rn(xn, pos_ref[3ull * i + a]), g.L[a], g.h[a]);
            d2 = a == 0 ? __dmul_rn(d, d) : __dadd_rn(d2, __dmul_rn(d, d));
        }
        pos[i] = make_double4(x[0], x[1], x[2], p.w);
        if (MD_STAGE_FROM_REL) rel[i] = md_rel_record(x[0], x[1], x[2], cell_lin[i], g);  // meaningful once binned
        vel[i] = make_double4(u[0], u[1], u[2], m);
        fire = d2 > thr2 ? (d2 > danger2 ? 3u : 1u) : 0u;
        d2f = __double2float_ru(d2);
    }
    // the criterion of PAPER.md:79 into the device flags.  In a DPD fluid thousands of particles cross the threshold in the
    // same step; one store per crossing particle to the same address serialises in L2 (measured: 38 -> 120 us for this
    // kernel at 10^6 particles), so a warp stores once, and only while the flag is not yet up (benign race: every writer
    // stores the same value, and nobody reads the flags before the kernel has finished)
    const unsigned wfire = __reduce_or_sync(0xffffffffu, fire);
    if ((threadIdx.x & 31u) == 0 && wfire) {
        if (*(volatile int *)&flags->rebuild == 0) flags->rebuild = 1;
        if (at_val && *(volatile unsigned int *)&flags->rebuild_at == 0u) flags->rebuild_at = at_val;
        if ((wfire & 2u) && *(volatile int *)&flags->dangerous == 0) flags->dangerous = 1;
    }
    const unsigned wmax = __reduce_max_sync(0xffffffffu, __float_as_uint(d2f));  // non-negative floats order as uints
    if ((threadIdx.x & 31u) == 0 && wmax > flags->max_d2[slot]) atomicMax(&flags->max_d2[slot], wmax);
    if (i == 0) flags->max_d2[slot ^ 1] = 0u;
}

__global__ void k_half2_nvt(double4 *__restrict__ vel, const double4 *__restrict__ force, uint32_t N, double half_dt,
                            const double *__restrict__ nvt, Gate gate)
{
    if (md_gate_closed(gate)) return;
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double xi = nvt[0];
    double4 v = vel[i];
    const double4 f = force[i];
    v.x = __dadd_rn(v.x, __dmul_rn(half_dt, __dsub_rn(__ddiv_rn(f.x, v.w), __dmul_rn(xi, v.x))));
    v.y = __dadd_rn(v.y, __dmul_rn(half_dt, __dsub_rn(__ddiv_rn(f.y, v.w), __dmul_rn(xi, v.y))));
    v.z = __dadd_rn(v.z, __dmul_rn(half_dt, __dsub_rn(__ddiv_rn(f.z, v.w), __dmul_rn(xi, v.z))));
    vel[i] = v;
}

__global__ void k_half2(double4 *__restrict__ vel, const double4 *__restrict__ force, uint32_t N, double half_dt, Gate gate)
{
    if (md_gate_closed(gate)) return;
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    double4 v = vel[i];
    const double4 f = force[i];
    v.x = __dadd_rn(v.x, __ddiv_rn(__dmul_rn(half_dt, f.x), v.w));
    v.y = __dadd_rn(v.y, __ddiv_rn(__dmul_rn(half_dt, f.y), v.w));
    v.z = __dadd_rn(v.z, __ddiv_rn(__dmul_rn(half_dt, f.z), v.w));
    vel[i] = v;
}

int launch_half1(md_ctx *c, double dt, bool fused, bool nvt)
{
    LaunchCfg cf = c->cfg[MD_K_INTEGRATE];
    cf.block = std::min(cf.block, MD_HALF1_MAX_BLOCK);  // k_half1 is compiled for 6 blocks of 256 threads per SM (latency bound: occupancy)
    const double t = 0.5 * c->r_buff;
    c->d2_slot ^= 1;
    const unsigned grid = md_grid(c->N, cf.block);
    // gate of a plain half 1 of index s: closed by an EARLIER firing only (index < s); of the fused launch (half 2 of s +
    // half 1 of s + 1): closed by a firing at <= s
    const Gate hg = fused ? md_gate(c) : Gate{c->gate_s > 1 ? &c->d_flags->rebuild_at : nullptr, c->gate_s - 1};
#define HALF1_ARGS c->pos, c->vel, c->force, c->image, c->pos_ref, c->cell_lin, c->rel, c->g, dt, 0.5 * dt, t * t, \
                   c->r_buff * c->r_buff, c->d_flags, c->d2_slot, c->nvt_state, hg, c->gate_set
    if (nvt) {
        if (fused) k_half1<true, true><<<grid, cf.block, 0, c->stream>>>(HALF1_ARGS);
        else k_half1<false, true><<<grid, cf.block, 0, c->stream>>>(HALF1_ARGS);
    } else {
        if (fused) k_half1<true, false><<<grid, cf.block, 0, c->stream>>>(HALF1_ARGS);
        else k_half1<false, false><<<grid, cf.block, 0, c->stream>>>(HALF1_ARGS);
    }
#undef HALF1_ARGS
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

int launch_half2(md_ctx *c, double dt, bool nvt)
{
    const LaunchCfg &cf = c->cfg[MD_K_INTEGRATE];
    if (nvt)
        k_half2_nvt<<<md_grid(c->N, cf.block), cf.block, 0, c->stream>>>(c->vel, c->force, (uint32_t)c->N, 0.5 * dt, c->nvt_state, md_gate(c));
    else
        k_half2<<<md_grid(c->N, cf.block), cf.block, 0, c->stream>>>(c->vel, c->force, (uint32_t)c->N, 0.5 * dt, md_gate(c));
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

// ------------------------------------------------------------------------------------------------------------
// md_thermo: kinetic energy, potential energy and momentum.  Fixed summation order: block b
// sums a contiguous range of slots (thread-strided, then a shared-memory tree), one block then sums the partials.
// ------------------------------------------------------------------------------------------------------------
constexpr int THERMO_BLOCK = 256;
constexpr uint32_t THERMO_PER_BLOCK = 4096;  // slots per block of the first pass

__device__ __forceinline__ void thermo_block_sum(double v[5], double *sm /* [5][THERMO_BLOCK] */)
{
#pragma unroll
    for (int k = 0; k < 5; ++k) sm[k * THERMO_BLOCK + threadIdx.x] = v[k];
    __syncthreads();
    for (int o = THERMO_BLOCK / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) {
#pragma unroll
            for (int k = 0; k < 5; ++k) sm[k * THERMO_BLOCK + threadIdx.x] += sm[k * THERMO_BLOCK + threadIdx.x + o];
        }
        __syncthreads();
    }
}

__global__ void __launch_bounds__(THERMO_BLOCK) k_thermo_partial(const double4 *__restrict__ vel,
                                                                 const double4 *__restrict__ force, uint32_t N,
                                                                 double *__restrict__ partial /* [gridDim.x][5] */, Gate gate)
{
    if (md_gate_closed(gate)) return;
    __shared__ double sm[5 * THERMO_BLOCK];
    const uint32_t b0 = blockIdx.x * THERMO_PER_BLOCK, b1 = min(N, b0 + THERMO_PER_BLOCK);
    double v[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    for (uint32_t i = b0 + threadIdx.x; i < b1; i += THERMO_BLOCK) {
        const double4 u = vel[i];
        v[0] += 0.5 * u.w * (u.x * u.x + u.y * u.y + u.z * u.z);
        v[1] += force[i].w;
        v[2] += u.w * u.x; v[3] += u.w * u.y; v[4] += u.w * u.z;
    }
    thermo_block_sum(v, sm);
    if (threadIdx.x < 5) partial[5ull * blockIdx.x + threadIdx.x] = sm[threadIdx.x * THERMO_BLOCK];
}

__global__ void __launch_bounds__(THERMO_BLOCK) k_thermo_final(const double *__restrict__ partial, uint32_t n_partial,
                                                               double *__restrict__ out /* [5] */, Gate gate)
{
    if (md_gate_closed(gate)) return;
    __shared__ double sm[5 * THERMO_BLOCK];
    double v[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    for (uint32_t b = threadIdx.x; b < n_partial; b += THERMO_BLOCK) {
#pragma unroll
        for (int k = 0; k < 5; ++k) v[k] += partial[5ull * b + k];
    }
    thermo_block_sum(v, sm);
    if (threadIdx.x < 5) out[threadIdx.x] = sm[threadIdx.x * THERMO_BLOCK];
}

static int thermo_reduce(md_ctx *c, double **res_out, Gate gate = Gate{nullptr, 0});

int launch_thermo(md_ctx *c, double *out5_host)
{
    double *res = nullptr;
    MD_TRY(thermo_reduce(c, &res));
    MD_CUDA_CHECK(c, cudaMemcpyAsync(out5_host, res, 5 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    return md_sync(c);
}

// Nose-Hoover thermostat update (R30), on the device: K' from the two reduction kernels above, then one thread
__global__ void k_nvt_update(const double *__restrict__ sums, double *__restrict__ nvt, double dt, double kT, double tau,
                             double dof, Gate gate)
{
    if (md_gate_closed(gate)) return;
    const double K = sums[0];
    const double xi_old = nvt[0];
    const double xi = xi_old + (dt / (tau * tau)) * (2.0 * K / (dof * kT) - 1.0);
    nvt[0] = xi;
    nvt[1] = nvt[1] + 0.5 * dt * (xi + xi_old);
}

static int thermo_reduce(md_ctx *c, double **res_out, Gate gate)
{
    const uint32_t N = (uint32_t)c->N;
    const uint32_t nb = (N + THERMO_PER_BLOCK - 1) / THERMO_PER_BLOCK;
    const uint64_t need = 5ull * nb + 8;
    if (need > c->thermo_len) {
        if (c->thermo_buf) { md_free(c, c->thermo_buf); c->thermo_buf = nullptr; }
        c->thermo_len = 0;
        MD_TRY(md_alloc(c, (void **)&c->thermo_buf, need * sizeof(double)));
        c->thermo_len = need;
    }
    double *res = c->thermo_buf + 5ull * nb;
    k_thermo_partial<<<nb, THERMO_BLOCK, 0, c->stream>>>(c->vel, c->force, N, c->thermo_buf, gate);
    MD_LAUNCH_CHECK(c);
    k_thermo_final<<<1, THERMO_BLOCK, 0, c->stream>>>(c->thermo_buf, nb, res, gate);
    MD_LAUNCH_CHECK(c);
    *res_out = res;
    return MD_OK;
}

// Martyna-Tobias-Klein thermostat factor T(dt/2) (R39), `halves` of them in a row (2: the trailing factor of one step and
// the leading factor of the next): xi += (dt/4) G; s = exp(-xi dt/2); K <- s^2 K; eta += xi dt/2; xi += (dt/4) G', with
// G = (2K - g kT)/Q, Q = g kT tau^2.  K comes from the reduction kernels above; the product of the scale factors goes to
// nvt[2] and k_mtk_scale applies it to every velocity.
__global__ void k_mtk_update(const double *__restrict__ sums, double *__restrict__ nvt, double dt, double kT, double tau,
                             double dof, int halves, Gate gate)
{
    if (md_gate_closed(gate)) return;
    double K = sums[0], xi = nvt[0], eta = nvt[1], s_tot = 1.0;
    const double Q = dof * kT * tau * tau;
    for (int h = 0; h < halves; ++h) {
        xi = xi + 0.25 * dt * (2.0 * K - dof * kT) / Q;
        const double s = exp(-0.5 * dt * xi);
        K = K * s * s;
        eta = eta + 0.5 * dt * xi;
        xi = xi + 0.25 * dt * (2.0 * K - dof * kT) / Q;
        s_tot *= s;
    }
    nvt[0] = xi;
    nvt[1] = eta;
    nvt[2] = s_tot;
}

__global__ void k_mtk_scale(double4 *__restrict__ vel, uint32_t N, const double *__restrict__ nvt, Gate gate)
{
    if (md_gate_closed(gate)) return;
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double s = nvt[2];
    double4 v = vel[i];
    v.x *= s; v.y *= s; v.z *= s;
    vel[i] = v;
}

int launch_mtk_thermostat(md_ctx *c, double dt, double kT, double tau, int halves)
{
    const Gate tg = md_gate(c);  // part of the step whose index is c->gate_s (MD_SCHED_BATCH), open otherwise
    double *res = nullptr;
    MD_TRY(thermo_reduce(c, &res, tg));
    k_mtk_update<<<1, 1, 0, c->stream>>>(res, c->nvt_state, dt, kT, tau, 3.0 * (double)c->N - 3.0, halves, tg);
    MD_LAUNCH_CHECK(c);
    const LaunchCfg &cf = c->cfg[MD_K_INTEGRATE];
    k_mtk_scale<<<md_grid(c->N, cf.block), cf.block, 0, c->stream>>>(c->vel, (uint32_t)c->N, c->nvt_state, tg);
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}

int launch_nvt_thermostat(md_ctx *c, double dt, double kT, double tau)
{
    // part of the half 1 it follows: same gate as that launch (c->gate_nvt is set by the caller)
    const Gate tg = Gate{c->gate_nvt ? &c->d_flags->rebuild_at : nullptr, c->gate_nvt};
    double *res = nullptr;
    MD_TRY(thermo_reduce(c, &res, tg));
    k_nvt_update<<<1, 1, 0, c->stream>>>(res, c->nvt_state, dt, kT, tau, 3.0 * (double)c->N - 3.0, tg);
    MD_LAUNCH_CHECK(c);
    return MD_OK;
}
