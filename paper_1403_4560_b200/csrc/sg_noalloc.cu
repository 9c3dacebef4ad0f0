// sg_noalloc.cu — the state hash for callers that must not allocate device memory (sg_get_state_hash_noalloc).
//
// Who this is for.  Some programs that embed this library cannot call cudaMalloc at the moment they want a state hash:
//   - a host application that has handed the whole device to its own pool (a framework's caching allocator, a job
//     runner with a fixed arena): a raw cudaMalloc from a library either fails for lack of memory or takes pages the
//     pool believes it owns;
//   - a monitoring / checkpoint-verification hook called from inside a running simulation loop: cudaMalloc and
//     cudaFree synchronise the whole device, which would stall every stream of the run each time the hook fires;
//   - a caller that was given an sg_ctx built on somebody else's workspace and has no allocator of its own at all.
// The ordinary sg_get_state_hash stages the per-system hashes in a workspace buffer whose size grows with the pool.
// The variant here stages them in ONE fixed array that is part of the library image instead, so the call needs no
// allocation of any kind: no cudaMalloc / cudaFree / cudaMallocAsync / stream or event creation, neither here nor in
// anything it calls.
//
// The price.  The array below occupies SG_NOALLOC_MAX_SYSTEMS * 8 bytes = 512 KiB of device memory on EVERY GPU on
// which this library's device code gets loaded, from that load until the process exits, whether or not the entry point
// is ever used.  Pools larger than SG_NOALLOC_MAX_SYSTEMS systems are refused (use sg_get_state_hash for those).
//
// Sharing.  There is one array per GPU and every call on that GPU uses it.  It is not cleared between calls: a call
// writes entries [0, n_sys) and reads back exactly those, so nothing has to start at zero and whatever an earlier,
// larger call left behind in [n_sys, max) is never looked at.  Two calls whose GPU work can overlap (different contexts
// on different streams, driven from different host threads) would write the same entries: that is a data race and the
// hashes of both are undefined.  Calls from one thread are safe: each call waits for its copy before it returns.
//
// A trap for whoever edits this file: in HOST code the name `g_hash_scratch` is only a handle that the runtime uses to
// look the array up; it is not the array's device address.  Handing `g_hash_scratch` itself to a kernel or to
// cudaMemcpy gives the kernel a host address: an illegal-address fault, or, on a system where the GPU can reach host
// memory, a silent read / write of the wrong bytes.  The device address comes from cudaGetSymbolAddress, asked once per
// device with that device current (scratch_address below), and that pointer is what the kernel and the copy get.
// (Device code in this file could name the array directly; the kernel takes the pointer so that it stays the same
// code as the workspace version.)
#include <mutex>

#include "sg_internal.h"

namespace sg {

namespace {

constexpr int MAX_DEVICES = 64;

static __device__ __align__(256) unsigned long long g_hash_scratch[SG_NOALLOC_MAX_SYSTEMS];

std::mutex g_setup_mutex;
unsigned long long *g_scratch_addr[MAX_DEVICES];        // device address of g_hash_scratch per device ordinal (nullptr: not asked yet)

// Device address of the scratch array on the CURRENT device; looked up on the first call per device and remembered.
// That first call makes the runtime load this library's device code onto the device if it is not there yet.
cudaError_t scratch_address(unsigned long long **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_addr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_hash_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_scratch_addr[dev] = static_cast<unsigned long long *>(p);
    }
    *out = g_scratch_addr[dev];
    return cudaSuccess;
}

// Same hash as k_hash_words (sg_pmj.cu; definition in include/sg.h at sg_get_state_hash): one warp per system, the sum
// over the system's 32-bit words of mix64(index << 32 | word).  Written out again here so that nothing in the existing
// kernels changes; tests/test_zz_no_alloc.py holds the two to the same values.
__device__ __forceinline__ uint64_t mix64_noalloc(uint64_t x)
{
    x ^= x >> 30; x *= 0xbf58476d1ce4e5b9ULL;
    x ^= x >> 27; x *= 0x94d049bb133111ebULL;
    x ^= x >> 31;
    return x;
}

__global__ void __launch_bounds__(128)
k_hash_words_noalloc(const uint32_t *__restrict__ words, long long n_sys, int words_per_sys,
                     unsigned long long *__restrict__ scratch)
{
    const int lane = threadIdx.x & 31;
    const long long sys = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (sys >= n_sys) return;
    const uint32_t *p = words + (size_t)sys * words_per_sys;
    uint64_t h = 0;
    for (int i = lane; i < words_per_sys; i += 32) h += mix64_noalloc(((uint64_t)(uint32_t)i << 32) | p[i]);
    for (int o = 16; o; o >>= 1) h += __shfl_xor_sync(0xffffffffu, h, o);
    if (lane == 0) scratch[sys] = h;
}

}  // namespace

// Hash of every system of the context's current state into the HOST buffer `out_host`, staged through the static array.
// Returns cudaSuccess or the first CUDA error; *too_large is set (and nothing is launched) if the pool has more than
// SG_NOALLOC_MAX_SYSTEMS systems.  One kernel launch, one device-to-host copy, one stream synchronisation.
cudaError_t hash_noalloc(sg_ctx *c, uint64_t *out_host, bool *too_large, int *launches)
{
    const Dims &d = c->d;
    const long long n_sys = (long long)d.W * d.R * d.NT;
    *too_large = n_sys > (long long)SG_NOALLOC_MAX_SYSTEMS;
    *launches = 0;
    if (*too_large) return cudaSuccess;
    unsigned long long *scratch = nullptr;
    cudaError_t e = scratch_address(&scratch);
    if (e != cudaSuccess) return e;
    const int wps = is_packed(c) ? d.N : d.N / 4;
    const uint32_t *words = is_packed(c) ? c->spins : reinterpret_cast<const uint32_t *>(c->spins8);
    k_hash_words_noalloc<<<(unsigned)((n_sys + 3) / 4), 128, 0, c->stream>>>(words, n_sys, wps, scratch);
    *launches = 1;
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    if ((e = cudaMemcpyAsync(out_host, scratch, sizeof(uint64_t) * (size_t)n_sys, cudaMemcpyDeviceToHost, c->stream)) != cudaSuccess)
        return e;
    return cudaStreamSynchronize(c->stream);
}

}  // namespace sg
