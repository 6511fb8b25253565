// gn_static.cu -- gn_check_headroom_static: the one entry point of the library that needs no device memory from anybody.
//
// Everything else in libgn.so lives in a workspace the caller allocates and hands to gn_create.  Some callers have no way
// to produce such a buffer at the moment they need an answer: a plug-in inside a host program that gave the whole GPU to
// its own pool (a training framework's caching allocator, an inference server's arena) and forbids driver allocations; a
// control loop that must not call cudaMalloc / cudaFree because both stall every stream of the device; a process that is
// already at its memory limit because the network's workspace took what was left.  For them the per-target accumulator
// that the overflow check of gn_create keeps in the workspace (gn_validate_kernel's abs_in, gn_kernels.cu) is kept here
// in a fixed array that is part of the loaded library image: GN_STATIC_MAX_VERTICES x 8 bytes = 8 MB on every GPU that
// loads libgn.so, from the first CUDA call of the process to its exit, whether this entry point is ever called or not.
//
// The array, the kernel that uses it and the host code that looks its address up sit in this one file on purpose: in host
// code the array's name is only a handle for the runtime, not a device address, so the address is asked for once per
// device with cudaGetSymbolAddress (below) and that pointer is what the kernel and cudaMemsetAsync are given.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include <mutex>

#include "gn_internal.h"

namespace {

// sum of |w_fx| over the in-edges of every target, in units of 2^-16: shared by every call on this device
static __device__ __align__(256) unsigned long long gn_static_abs_in[GN_STATIC_MAX_VERTICES];

constexpr int kMaxDevices = 64;
std::mutex g_lookup_mutex;
unsigned long long *g_abs_in_of_device[kMaxDevices];   // device address of gn_static_abs_in on each device, once known

// One thread per edge (grid-stride).  The quantisation is gn_quantise_kernel's, the accumulation gn_validate_kernel's;
// because every addend is >= 0 a target's sum only grows, so "the final sum exceeds the limit" is the same as "one add
// carried the sum across the limit", and exactly one add does: that one counts the target.  No second pass is needed.
__global__ void __launch_bounds__(256)
gn_headroom_static_kernel(unsigned long long *__restrict__ abs_in, const uint32_t n_vertices, const uint64_t n_edges,
                          const uint32_t *__restrict__ targets, const float *__restrict__ weights,
                          const unsigned long long limit, uint32_t *__restrict__ out)
{
    uint32_t at_risk = 0u, skipped = 0u;
    for (uint64_t e = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; e < n_edges; e += (uint64_t)gridDim.x * blockDim.x) {
        const uint32_t m = targets[e];
        const float s = __fmul_rn(weights[e], 65536.0f);
        if (m >= n_vertices || !(fabsf(s) < 2147483648.0f)) { ++skipped; continue; }   // gn_create: BAD_GRAPH
        const long long w = __float2int_rn(s);
        const unsigned long long a = (unsigned long long)(w < 0 ? -w : w);
        if (a == 0ull) continue;
        const unsigned long long before = atomicAdd(&abs_in[m], a);
        if (before <= limit && before + a > limit) ++at_risk;
    }
    if (at_risk) atomicAdd(&out[0], at_risk);
    if (skipped) atomicAdd(&out[1], skipped);
}

}  // namespace

extern "C" int gn_check_headroom_static(void *cuda_stream, uint32_t n_vertices, uint64_t n_edges, const uint32_t *targets,
                                        const float *weights, float largest_kick, uint32_t *out)
{
    if (!out) return gn_fail(GN_E_INVALID_ARG, "out is NULL");
    if (n_edges && (!targets || !weights)) return gn_fail(GN_E_INVALID_ARG, "targets/weights are NULL with n_edges > 0");
    if (n_vertices == 0 || n_vertices > GN_STATIC_MAX_VERTICES)
        return gn_fail(GN_E_INVALID_ARG, "gn_check_headroom_static holds its per-target sums in a fixed %u-entry array: "
                       "n_vertices = %u is outside 1 .. GN_STATIC_MAX_VERTICES (larger networks are checked by gn_create, in "
                       "the caller's workspace)", (unsigned)GN_STATIC_MAX_VERTICES, (unsigned)n_vertices);
    if (n_edges >= 0xFFFFFFFFull) return gn_fail(GN_E_INVALID_ARG, "n_edges must be < 2^32 - 1");
    const double kick = nearbyint(fabs((double)largest_kick) * 65536.0);              // |kick_fx| as gn_create forms it
    if (!(kick < 2147483648.0)) return gn_fail(GN_E_INVALID_ARG, "largest_kick out of the fixed-point range");
    const unsigned long long limit = 2147483647ull - (unsigned long long)kick;       // sum |w_fx| may reach this, not pass it

    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return gn_fail(GN_E_CUDA, "cudaGetDevice failed: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices) return gn_fail(GN_E_CUDA, "device ordinal %d is beyond the %d this entry point keeps addresses for", dev, kMaxDevices);
    unsigned long long *abs_in = nullptr;
    {
        // Set-up, on the first call with this device current: ask the runtime where the array lives on THIS device.
        std::lock_guard<std::mutex> lock(g_lookup_mutex);
        if (!g_abs_in_of_device[dev]) {
            void *p = nullptr;
            e = cudaGetSymbolAddress(&p, gn_static_abs_in);
            if (e != cudaSuccess || !p)
                return gn_fail(GN_E_CUDA, "cudaGetSymbolAddress(gn_static_abs_in) failed on device %d: %s", dev, cudaGetErrorString(e));
            g_abs_in_of_device[dev] = (unsigned long long *)p;
        }
        abs_in = g_abs_in_of_device[dev];
    }
    // The array still holds the previous call's sums, the output whatever the caller left there: both start at zero.
    e = cudaMemsetAsync(abs_in, 0, (size_t)n_vertices * sizeof(unsigned long long), st);
    if (e == cudaSuccess) e = cudaMemsetAsync(out, 0, 2 * sizeof(uint32_t), st);
    if (e != cudaSuccess) return gn_fail(GN_E_CUDA, "cudaMemsetAsync failed: %s", cudaGetErrorString(e));
    if (n_edges) {
        const uint64_t want = (n_edges + 255u) / 256u;
        const uint32_t grid = (uint32_t)(want < 148u * 8u ? want : 148u * 8u);       // 8 CTAs of 256 threads on each of the 148 SMs
        gn_headroom_static_kernel<<<grid, 256, 0, st>>>(abs_in, n_vertices, n_edges, targets, weights, limit, out);
        e = cudaGetLastError();
        if (e != cudaSuccess) return gn_fail(GN_E_CUDA, "gn_headroom_static_kernel launch failed: %s", cudaGetErrorString(e));
    }
    return GN_OK;
}
