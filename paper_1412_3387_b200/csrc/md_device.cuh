// md_device.cuh -- device helpers of the CUDA path (decision arithmetic, minimum image, hash, warp segments).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "md_internal.h"

// ---- decision arithmetic: plain IEEE double, explicitly rounded, never contracted into FMA (R2) ----
__device__ __forceinline__ double md_min_image(double d, double L, double h)
{
    if (d >= h) d = __dsub_rn(d, L);
    else if (d < -h) d = __dadd_rn(d, L);
    return d;
}

__device__ __forceinline__ double md_r2_exact(double dx, double dy, double dz)
{
    return __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
}

// cell coordinate along one axis (R5): f = (x - lo)/L, c = (int)(f n), clamp to [0, n-1]
__device__ __forceinline__ uint32_t md_cell_coord(double x, double lo, double L, double dn, uint32_t n)
{
    double f = __ddiv_rn(__dsub_rn(x, lo), L);
    long long k = (long long)__dmul_rn(f, dn);
    if (k >= (long long)n) k = (long long)n - 1;
    if (k < 0) k = 0;
    return (uint32_t)k;
}

// Staging of the fp32 tile kernels: true = from the fp32 cell-relative records `rel` (three fp32 roundings per
// coordinate, 16 bytes per particle, half 1 keeps them current); false = from the fp64 positions with one rounding.
// Measured at config 2: true is 3 % faster per step (0.406 vs 0.417 ms); false lowers the largest
// mixed-precision force error over all 2^20 particles from 4.4e-4 to 3.2e-4 (R11 norm) -- neither reaches 1e-4 there.
constexpr bool MD_STAGE_FROM_REL = true;

// Three signed 10-bit integers in one word: residuals of fp32 coordinates in units of a quantum, clamped to +-511 and
// stored biased by 512.  Conversions between integers and doubles go through the 2^52 trick (an integer n in the low
// word of a double with exponent 2^52 IS the double 2^52 + n): the conversion unit runs at 1/8 of the FP32 rate on B200
// (md_debug_peak) and was the bottleneck of the mixed-precision force kernel when these used cvt instructions.
#define MD_TWO52 4503599627370496.0
__device__ __forceinline__ double md_small_int_to_double(int n)  // |n| < 2^31
{
    return __hiloint2double(0x43300000, (int)((unsigned)n ^ 0x80000000u)) - (MD_TWO52 + 2147483648.0);
}
__device__ __forceinline__ int md_round_to_int(double x)  // |x| < 2^31, round to nearest even
{
    return __double2loint(x + (MD_TWO52 + 2147483648.0)) ^ (int)0x80000000;
}
// fields of a packed residual word: 10 bits each, value + 255 (value in [-255, 255]); the sum of two such words is a
// word of fields value_a + value_b + 510 in [0, 1020] (no carry between fields), and differences of equally biased
// fields need no un-biasing
__device__ __forceinline__ int md_res_x(uint32_t w) { return (int)(w & 0x3ffu); }
__device__ __forceinline__ int md_res_y(uint32_t w) { return (int)((w >> 10) & 0x3ffu); }
__device__ __forceinline__ int md_res_z(uint32_t w) { return (int)((w >> 20) & 0x3ffu); }

// one coordinate on the grid: n q0 as a float (exact: |n| < 2^24) and the residual (v - n q0) / qr in [-255, 255] + 255
__device__ __forceinline__ float md_grid_coord(double v, double q0, double q0i, double qri, uint32_t &field)
{
    const double n = (double)md_round_to_int(v * q0i);
    const double vq = n * q0;
    field = (uint32_t)(max(-255, min(255, md_round_to_int((v - vq) * qri))) + 255);
    return (float)vq;
}

// Centre of cell c along axis a, SNAPPED to the grid q0 (explicitly rounded operations: the binning, half 1 and the tile
// kernels must all get the same value).  The fp32 records are relative to these snapped centres, so the offset between
// two cells is an exact multiple of q0 -- the same in every tile: x_i - x_j is the same real number in the tile of i and
// in the tile of j, pair forces are exactly antisymmetric and the total momentum is conserved to fp64 rounding.
__device__ __forceinline__ double md_cell_centre_q(uint32_t c, int a, const Geom &g)
{
    const double cc = __dadd_rn(g.lo[a], __dmul_rn(__dadd_rn((double)c, 0.5), g.cw[a]));
    return __dmul_rn(rint(__dmul_rn(cc, g.q0i)), g.q0);
}

// fp32 record of a position relative to the (snapped) centre of cell `lin` (linear id), minimum image applied: what the fp32
// tile kernels stage.  x, y, z are rounded to the grid q0 (a multiple of q0 below 2^24 q0 is an exact float, and so is
// its sum with a cell offset on the same grid: the tile kernels stage WITHOUT a rounding); what the grid drops is kept in
// .w as three 10-bit residuals in units of qr = q0 / 512 (clamped to +-255), so that the mixed-precision force kernel can rebuild
// separations to ~1e-9 for the pairs of the first shell (R25).
__device__ __forceinline__ float4 md_rel_record(double x, double y, double z, uint32_t lin, const Geom &g)
{
    const uint32_t nxy = g.n[0] * g.n[1];
    const uint32_t cz = lin / nxy, rem = lin - cz * nxy;
    const uint32_t cy = rem / g.n[0], cx = rem - cy * g.n[0];
    const double rx = md_min_image(x - md_cell_centre_q(cx, 0, g), g.L[0], g.h[0]);
    const double ry = md_min_image(y - md_cell_centre_q(cy, 1, g), g.L[1], g.h[1]);
    const double rz = md_min_image(z - md_cell_centre_q(cz, 2, g), g.L[2], g.h[2]);
    uint32_t fx, fy, fz;
    const float vx = md_grid_coord(rx, g.q0, g.q0i, g.qri, fx);
    const float vy = md_grid_coord(ry, g.q0, g.q0i, g.qri, fy);
    const float vz = md_grid_coord(rz, g.q0, g.q0i, g.qri, fz);
    return make_float4(vx, vy, vz, __uint_as_float(fx | (fy << 10) | (fz << 20)));
}

// fast reciprocal: fp32 = MUFU.RCP (about 1 ulp), fp64 = IEEE division
__device__ __forceinline__ float md_rcp(float x)
{
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ double md_rcp(double x) { return 1.0 / x; }

// closed <=> a half 1 of enqueue index <= g.s has fired the criterion (uniform over the grid: read once per thread)
__device__ __forceinline__ bool md_gate_closed(const Gate g)
{
    if (!g.at) return false;
    const unsigned int at = *(const volatile unsigned int *)g.at;
    return at != 0u && at <= g.s;
}
static inline Gate md_gate(md_ctx *c) { return Gate{c->gate_s ? &c->d_flags->rebuild_at : nullptr, c->gate_s}; }

// ---- tag lane: pos.w carries the particle tag as raw bits --------------------------------------------------
__device__ __forceinline__ double md_tag_to_lane(uint32_t tag) { return __longlong_as_double((long long)tag); }
__device__ __forceinline__ uint32_t md_lane_to_tag(double w) { return (uint32_t)__double_as_longlong(w); }

// ---- Philox4x32-10 (Salmon et al., SC'11), word 0 only is used by DPD (R14) -------------------------
__device__ __forceinline__ uint4 md_philox4x32_10(uint4 c, uint2 k)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
        c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
        k.x += 0x9E3779B9u;
        k.y += 0xBB67AE85u;
    }
    return c;
}

// theta_ij: uniform, zero mean, unit variance, symmetric in (i, j)
__device__ __forceinline__ double md_dpd_theta(uint32_t ti, uint32_t tj, uint64_t step, uint64_t seed)
{
    const uint32_t lo = min(ti, tj), hi = max(ti, tj);
    uint4 x = md_philox4x32_10(make_uint4(lo, hi, (uint32_t)step, (uint32_t)(step >> 32)),
                               make_uint2((uint32_t)seed, (uint32_t)(seed >> 32)));
    const double u = ((double)x.x + 0.5) * (1.0 / 4294967296.0);
    return 1.7320508075688772 * (2.0 * u - 1.0);
}

// ---- warp segments of W cooperating threads ("w threads per particle") -----------------------
template <int W>
__device__ __forceinline__ unsigned md_seg_mask()
{
    if constexpr (W == 32) {
        return 0xffffffffu;
    } else {
        const unsigned lane = threadIdx.x & 31u;
        return ((1u << W) - 1u) << (lane & ~(unsigned)(W - 1));
    }
}

template <int W>
__device__ __forceinline__ double md_seg_sum(double v, unsigned mask)
{
#pragma unroll
    for (int o = W / 2; o > 0; o >>= 1) v += __shfl_xor_sync(mask, v, o, W);
    return v;
}

// dispatch a launch templated on W
#define MD_DISPATCH_W(w, ...)            \
    switch (w) {                          \
    case 1: { constexpr int W_ = 1; __VA_ARGS__; } break;   \
    case 2: { constexpr int W_ = 2; __VA_ARGS__; } break;   \
    case 4: { constexpr int W_ = 4; __VA_ARGS__; } break;   \
    case 8: { constexpr int W_ = 8; __VA_ARGS__; } break;   \
    case 16: { constexpr int W_ = 16; __VA_ARGS__; } break; \
    default: { constexpr int W_ = 32; __VA_ARGS__; } break; \
    }

#define MD_LAUNCH_CHECK(c)                                                                   \
    do {                                                                                     \
        cudaError_t _e = cudaGetLastError();                                                 \
        (c)->stats.launches++;                                                               \
        if (_e != cudaSuccess) {                                                             \
            (c)->err = std::string("kernel launch: ") + cudaGetErrorString(_e) + " (" +      \
                       __FILE__ + ":" + std::to_string(__LINE__) + ")";                      \
            return MD_ECUDA;                                                                 \
        }                                                                                    \
    } while (0)

static inline unsigned md_grid(uint64_t work_items, int block) { return (unsigned)((work_items + block - 1) / block); }
