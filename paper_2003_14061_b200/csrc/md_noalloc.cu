// md_velocity_sums_noalloc: the velocity part of the reductions S7 / F2 (kinetic energy, total momentum,
// largest speed -- the input of the rebuild rule) for callers that cannot allocate: code under CUDA-graph capture,
// tight serving loops, harnesses that forbid cudaMalloc.  It is the two-stage reduction of md_device.cuh:reduce_finish (warp
// shuffles -> shared memory -> one partial per block -> the last block, found with an atomic ticket + memory fence as in
// PAPER.md:66, sums the partials in a fixed order) with the block partials and the ticket held in a file-scope
// `static __device__` array instead of md_system's device buffers.  No md_system is needed; nothing is allocated or freed.
//
// The array has a fixed size, so the call has a maximum problem size (MD_NOALLOC_MAX_ATOMS); every GPU that loads the
// library holds the array (~0.64 MB) until the process exits.  ALL calls share it: two calls that overlap on the GPU (different
// streams, or different host threads) race on the partials and the ticket -- callers serialise them.  The array keeps the
// last call's contents; the ticket must start at zero and is cleared before every launch, the partials are overwritten before
// they are read.
//
// In host code the array's name `g_scratch` is a host-side stand-in, not a device address: its device address is taken once
// per device with cudaGetSymbolAddress (with that device current) and that pointer is what the kernel gets.
#include <mutex>

#include "md_types.h"

namespace {

constexpr int NA_THREADS = 256;
constexpr int NA_PER_THREAD = 4;                                  // atoms per thread
constexpr int NA_PER_BLOCK = NA_THREADS * NA_PER_THREAD;          // 1024 atoms per block
constexpr int NA_MAX_BLOCKS = MD_NOALLOC_MAX_ATOMS / NA_PER_BLOCK;
constexpr int NA_Q = 5;                                           // ke, px, py, pz, max v^2
constexpr int NA_TICKET_AT = NA_Q * NA_MAX_BLOCKS;                // the ticket: first word of the last 256 bytes
static_assert(MD_NOALLOC_MAX_ATOMS % NA_PER_BLOCK == 0, "the maximum is a whole number of blocks");

// [q * NA_MAX_BLOCKS + block] block partials of quantity q, then 32 doubles (256 bytes) whose first word is the ticket
static __device__ __align__(256) double g_scratch[NA_Q * NA_MAX_BLOCKS + 32];

__device__ __forceinline__ double na_warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double na_warp_max(double v)
{
#pragma unroll
    for (int o = 16; o; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// v: 3 n doubles, v[3 i + k] (the boundary layout of md_get_velocities_device).  out: ke, px, py, pz, vmax.
// scratch: the device address of g_scratch; its ticket word is zero on entry and zero again on exit.
__global__ void __launch_bounds__(NA_THREADS) k_velocity_sums(const double *__restrict__ v, long long n, double *scratch, double *out)
{
    __shared__ double sm[NA_Q][NA_THREADS / 32];
    __shared__ bool last;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nblk = gridDim.x;
    double q[NA_Q] = {0.0, 0.0, 0.0, 0.0, 0.0};
    const long long base = (long long)blockIdx.x * NA_PER_BLOCK;
#pragma unroll
    for (int k = 0; k < NA_PER_THREAD; k++) {
        const long long i = base + k * NA_THREADS + threadIdx.x;
        if (i < n) {
            const double vx = __ldg(v + 3 * i), vy = __ldg(v + 3 * i + 1), vz = __ldg(v + 3 * i + 2);
            const double v2 = vx * vx + vy * vy + vz * vz;
            q[0] += 0.5 * v2; q[1] += vx; q[2] += vy; q[3] += vz;
            q[4] = fmax(q[4], v2);
        }
    }
#pragma unroll
    for (int k = 0; k < NA_Q; k++) {
        const double r = k == 4 ? na_warp_max(q[k]) : na_warp_sum(q[k]);
        if (lane == 0) sm[k][wid] = r;
    }
    __syncthreads();
    if (threadIdx.x < NA_Q) {
        const int k = threadIdx.x;
        double r = sm[k][0];
        for (int w = 1; w < NA_THREADS / 32; w++) r = k == 4 ? fmax(r, sm[k][w]) : r + sm[k][w];
        scratch[(size_t)k * NA_MAX_BLOCKS + blockIdx.x] = r;
    }
    __threadfence();
    __syncthreads();
    unsigned *ticket = reinterpret_cast<unsigned *>(scratch + NA_TICKET_AT);
    if (threadIdx.x == 0) last = atomicInc(ticket, nblk - 1) == (unsigned)(nblk - 1);      // wraps to zero with the last block
    __syncthreads();
    if (!last) return;
    __threadfence();
    // the last block sums the partials of all blocks (itself included) in a fixed order: reproducible results
    for (int k = 0; k < NA_Q; k++) {
        double r = 0.0;
        const volatile double *p = scratch + (size_t)k * NA_MAX_BLOCKS;
        for (int b = threadIdx.x; b < nblk; b += NA_THREADS) r = k == 4 ? fmax(r, p[b]) : r + p[b];
        r = k == 4 ? na_warp_max(r) : na_warp_sum(r);
        __syncthreads();
        if (lane == 0) sm[0][wid] = r;
        __syncthreads();
        if (threadIdx.x == 0) {
            double t = sm[0][0];
            for (int w = 1; w < NA_THREADS / 32; w++) t = k == 4 ? fmax(t, sm[0][w]) : t + sm[0][w];
            out[k] = k == 4 ? sqrt(t) : t;
        }
    }
}

// device address of g_scratch, per device: taken once, with that device current (set-up, not the per-call path)
constexpr int NA_MAX_DEVICES = 64;
double *g_scratch_ptr[NA_MAX_DEVICES] = {};
std::mutex g_scratch_mutex;

int fail(int code, const char *msg)
{
    mdk_set_error(msg);
    return code;
}

bool on_device(const void *p, int dev)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return (a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged) && (a.type == cudaMemoryTypeManaged || a.device == dev);
}

}  // namespace

int md_velocity_sums_noalloc(const double *vxyz_device, int64_t n_atoms, double *out5_device, void *stream)
{
    if (!vxyz_device || !out5_device) return fail(MD_ERR_INVALID, "md_velocity_sums_noalloc: null argument");
    if (n_atoms < 1) return fail(MD_ERR_INVALID, "md_velocity_sums_noalloc: n_atoms must be >= 1");
    if (n_atoms > (int64_t)MD_NOALLOC_MAX_ATOMS)
        return fail(MD_ERR_INVALID, "md_velocity_sums_noalloc: n_atoms exceeds MD_NOALLOC_MAX_ATOMS (16,777,216): the scratch array is static; "
                                    "use md_energies of an md_system for larger systems");
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return fail(MD_ERR_CUDA, "md_velocity_sums_noalloc: no CUDA device"); }
    if (dev < 0 || dev >= NA_MAX_DEVICES) return fail(MD_ERR_INVALID, "md_velocity_sums_noalloc: device ordinal out of range");
    if (!on_device(vxyz_device, dev) || !on_device(out5_device, dev))
        return fail(MD_ERR_INVALID, "md_velocity_sums_noalloc: vxyz_device and out5_device must be device memory of the CURRENT device");
    double *scratch = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_scratch_mutex);
        if (!g_scratch_ptr[dev]) {
            // once per device, that device current: `g_scratch` itself is not a device address in host code
            double *p = nullptr;
            const cudaError_t e = cudaGetSymbolAddress((void **)&p, g_scratch);
            if (e != cudaSuccess || !p) {
                cudaGetLastError();
                return fail(MD_ERR_CUDA, "md_velocity_sums_noalloc: cudaGetSymbolAddress of the scratch array failed");
            }
            g_scratch_ptr[dev] = p;
        }
        scratch = g_scratch_ptr[dev];
    }
    cudaStream_t st = (cudaStream_t)stream;
    // the ticket must start at zero whatever an earlier (possibly aborted) call left behind; the partials need no clearing
    if (cudaMemsetAsync(scratch + NA_TICKET_AT, 0, 256, st) != cudaSuccess) { cudaGetLastError(); return fail(MD_ERR_CUDA, "md_velocity_sums_noalloc: clearing the ticket failed"); }
    const int blocks = (int)((n_atoms + NA_PER_BLOCK - 1) / NA_PER_BLOCK);
    k_velocity_sums<<<blocks, NA_THREADS, 0, st>>>(vxyz_device, (long long)n_atoms, scratch, out5_device);
    if (cudaGetLastError() != cudaSuccess) return fail(MD_ERR_CUDA, "md_velocity_sums_noalloc: kernel launch failed");
    return MD_OK;
}
