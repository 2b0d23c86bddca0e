// noalloc.cu -- md_kinetic_noalloc: the kinetic-energy / momentum reduction of md_thermo (integrate.cu: k_thermo_partial,
// k_thermo_final: one kinetic-energy reduction per NVT step) for callers that
// cannot allocate device memory: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
// The per-block partial sums, which md_thermo keeps in a buffer of the context (md_alloc), live here in a file-scope
// __device__ array of fixed size; the entry point calls no cudaMalloc / cudaFree and no allocating library routine, takes
// no context, and only enqueues two kernels on the caller's stream.
//
// The array: NOALLOC_MAX_BLOCKS x 4 doubles = 256 KiB, held by every GPU that loads this library until the process
// exits.  It bounds the problem size: N <= MD_NOALLOC_MAX_N = NOALLOC_MAX_BLOCKS * NOALLOC_PER_BLOCK.
// In HOST code the array's name is a host-side stand-in, not a device address, so the address the kernels get is taken
// once per device with cudaGetSymbolAddress (device current) and cached.
// All calls share the array and it keeps the last call's contents.  Nothing in it has to start at zero: the first kernel
// of a call writes every slot the second kernel of that call reads (slots [0, ceil(N / NOALLOC_PER_BLOCK)) x 4), and
// stale slots beyond that are never read.  Calls that overlap on the GPU (different streams, or graph branches without
// a dependency) RACE on it: serialise them.
#include <cuda_runtime.h>

#include <mutex>
#include <string>

#include "../../include/b200md.h"

namespace {

constexpr int NOALLOC_BLOCK = 256;
constexpr uint32_t NOALLOC_PER_BLOCK = 4096;   // particles per block of the first pass (as md_thermo's)
constexpr uint32_t NOALLOC_MAX_BLOCKS = 8192;  // 8192 * 4 doubles = 256 KiB of scratch
static_assert((uint64_t)NOALLOC_MAX_BLOCKS * NOALLOC_PER_BLOCK == MD_NOALLOC_MAX_N, "header and scratch size disagree");
constexpr int NOALLOC_MAX_DEVICES = 64;

static __device__ __align__(256) double g_noalloc_scratch[4ull * NOALLOC_MAX_BLOCKS];

std::mutex g_noalloc_mu;
double *g_noalloc_ptr[NOALLOC_MAX_DEVICES];  // device address of g_noalloc_scratch on each device, once taken
thread_local std::string g_noalloc_err;

__device__ __forceinline__ void noalloc_block_sum(double v[4], double *sm /* [4][NOALLOC_BLOCK] */)
{
#pragma unroll
    for (int k = 0; k < 4; ++k) sm[k * NOALLOC_BLOCK + threadIdx.x] = v[k];
    __syncthreads();
    for (int o = NOALLOC_BLOCK / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) {
#pragma unroll
            for (int k = 0; k < 4; ++k) sm[k * NOALLOC_BLOCK + threadIdx.x] += sm[k * NOALLOC_BLOCK + threadIdx.x + o];
        }
        __syncthreads();
    }
}

// block b sums particles [b * PER_BLOCK, (b + 1) * PER_BLOCK): thread-strided, then a shared-memory tree (fixed order)
__global__ void __launch_bounds__(NOALLOC_BLOCK) k_kinetic_partial_na(const double *__restrict__ vel /* [N][3] */,
                                                                     const double *__restrict__ mass /* [N] or null */,
                                                                     uint64_t N, double *__restrict__ partial /* [grid][4] */)
{
    __shared__ double sm[4 * NOALLOC_BLOCK];
    const uint64_t b0 = (uint64_t)blockIdx.x * NOALLOC_PER_BLOCK;
    const uint64_t b1 = b0 + NOALLOC_PER_BLOCK < N ? b0 + NOALLOC_PER_BLOCK : N;
    double v[4] = {0.0, 0.0, 0.0, 0.0};
    for (uint64_t i = b0 + threadIdx.x; i < b1; i += NOALLOC_BLOCK) {
        const double x = vel[3 * i], y = vel[3 * i + 1], z = vel[3 * i + 2];
        const double m = mass ? mass[i] : 1.0;
        v[0] += 0.5 * m * (x * x + y * y + z * z);
        v[1] += m * x; v[2] += m * y; v[3] += m * z;
    }
    noalloc_block_sum(v, sm);
    if (threadIdx.x < 4) partial[4ull * blockIdx.x + threadIdx.x] = sm[threadIdx.x * NOALLOC_BLOCK];
}

__global__ void __launch_bounds__(NOALLOC_BLOCK) k_kinetic_final_na(const double *__restrict__ partial, uint32_t n_partial,
                                                                   double *__restrict__ out /* [4] */)
{
    __shared__ double sm[4 * NOALLOC_BLOCK];
    double v[4] = {0.0, 0.0, 0.0, 0.0};
    for (uint32_t b = threadIdx.x; b < n_partial; b += NOALLOC_BLOCK) {
#pragma unroll
        for (int k = 0; k < 4; ++k) v[k] += partial[4ull * b + k];
    }
    noalloc_block_sum(v, sm);
    if (threadIdx.x < 4) out[threadIdx.x] = sm[threadIdx.x * NOALLOC_BLOCK];
}

int noalloc_fail(int code, const std::string &msg)
{
    g_noalloc_err = msg;
    return code;
}

// device address of the scratch array on the CURRENT device (taken once per device)
int noalloc_scratch(double **p)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return noalloc_fail(MD_ECUDA, std::string("md_kinetic_noalloc: cudaGetDevice: ") + cudaGetErrorString(e) +
                                          " (this library has no CPU fallback)");
    }
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return noalloc_fail(MD_EINVAL, "md_kinetic_noalloc: device ordinal out of range");
    std::lock_guard<std::mutex> lock(g_noalloc_mu);
    if (!g_noalloc_ptr[dev]) {
        double *ptr = nullptr;
        e = cudaGetSymbolAddress((void **)&ptr, g_noalloc_scratch);
        if (e != cudaSuccess || !ptr) {
            cudaGetLastError();
            return noalloc_fail(MD_ECUDA, std::string("md_kinetic_noalloc: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
        }
        g_noalloc_ptr[dev] = ptr;
    }
    *p = g_noalloc_ptr[dev];
    return MD_OK;
}

bool noalloc_on_device(const void *p)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

}  // namespace

extern "C" const char *md_noalloc_last_error(void) { return g_noalloc_err.c_str(); }

extern "C" int md_kinetic_noalloc(const double *vel, const double *mass, uint64_t N, double *out4, void *stream)
{
    if (!out4 || (N > 0 && !vel)) return noalloc_fail(MD_EINVAL, "md_kinetic_noalloc: vel and out4 are required");
    if (N > MD_NOALLOC_MAX_N)
        return noalloc_fail(MD_EINVAL, "md_kinetic_noalloc: N = " + std::to_string(N) + " exceeds MD_NOALLOC_MAX_N = " +
                                           std::to_string((uint64_t)MD_NOALLOC_MAX_N) +
                                           " (the static scratch array holds 8192 block partials of 4096 particles each); "
                                           "use md_thermo on a context for larger systems");
    double *scratch = nullptr;
    const int s = noalloc_scratch(&scratch);
    if (s != MD_OK) return s;
    if ((N > 0 && !noalloc_on_device(vel)) || (mass && !noalloc_on_device(mass)) || !noalloc_on_device(out4))
        return noalloc_fail(MD_EINVAL, "md_kinetic_noalloc: vel, mass and out4 must be DEVICE pointers (no staging buffer is allocated here)");
    cudaStream_t st = (cudaStream_t)stream;
    const uint32_t nb = (uint32_t)((N + NOALLOC_PER_BLOCK - 1) / NOALLOC_PER_BLOCK);
    if (nb) k_kinetic_partial_na<<<nb, NOALLOC_BLOCK, 0, st>>>(vel, mass, N, scratch);
    k_kinetic_final_na<<<1, NOALLOC_BLOCK, 0, st>>>(scratch, nb, out4);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return noalloc_fail(MD_ECUDA, std::string("md_kinetic_noalloc: kernel launch: ") + cudaGetErrorString(e));
    return MD_OK;
}
