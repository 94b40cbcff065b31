// rfa_noalloc.cu -- device scratch that nobody has to allocate, for rfa_step_record_static (include/rfa.h).
//
// rfa_step_record with a host result buffer keeps the probe rows of a run in device memory that the library obtains
// with cudaMalloc on the first call and again whenever a longer series is asked for (rfa_set_probes allocates the probe list the
// same way).  That is fine for a script, and wrong for two kinds of caller:
//   * a frame loop that must not stall -- cudaMalloc / cudaFree wait for the whole device, so an allocation in the
//     middle of a session stops the stepping stream of every simulation on that GPU, not only the caller's;
//   * a host application that gave all device memory away at start-up (its own pool, a caching allocator that has
//     reserved the card, a fixed budget negotiated with other processes): there cudaMalloc simply fails.
// For them the probe list and the probe rows live in the array below, which is part of the library image: every GPU
// that loads librfa.so holds RFA_STATIC_SCRATCH_BYTES (1 MiB + 8 KiB) from then until the process ends, used or not.
//
// Rules that follow from "one array per GPU":
//   * every call on a GPU shares it, so two calls that are in flight on the same GPU at the same time (two host
//     threads, two simulations) overwrite each other's rows: callers serialise, the library takes no lock;
//   * it keeps whatever the last call left.  Nothing in it has to start at zero: a call first writes its probe list,
//     then one row per record, and reads back exactly the elements it wrote, so stale contents are never seen;
//   * `rfa_static_scratch` in HOST code is only the host-side shadow of the symbol, not a device address -- a kernel
//     handed that name would fault (or scribble over host memory on a machine where the GPU can reach it).  The
//     device address is asked of the runtime once per device, with that device current (static_scratch_base
//     below), and only that pointer is ever given to a kernel or a copy.
#include <cstdio>
#include <mutex>

#include "../../include/rfa.h"
#include "rfa_internal.h"

#define RFA_STATIC_MAX_DEVICES 64

constexpr size_t RFA_STATIC_INDEX_BYTES = (size_t)RFA_STATIC_RECORD_MAX_PROBES * sizeof(long long);     // probe list first,
constexpr size_t RFA_STATIC_SCRATCH_BYTES = RFA_STATIC_INDEX_BYTES + (size_t)RFA_STATIC_RECORD_MAX_FLOATS * sizeof(float);   // rows behind it
static_assert(RFA_STATIC_INDEX_BYTES % 256 == 0, "the rows start 256-byte aligned");

static __device__ __align__(256) unsigned char rfa_static_scratch[RFA_STATIC_SCRATCH_BYTES];

// Device address of the array on the CURRENT device.  The first call on a device asks the runtime
// (cudaGetSymbolAddress also makes the runtime load this module on that device); later calls return the cached
// pointer.  A device ordinal beyond the cache is served without caching.
static cudaError_t static_scratch_base(unsigned char **base)
{
    static std::mutex mu;
    static unsigned char *cached[RFA_STATIC_MAX_DEVICES];   // zero-initialised: "not asked yet"
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const bool slot = dev >= 0 && dev < RFA_STATIC_MAX_DEVICES;
    std::lock_guard<std::mutex> lock(mu);
    if (slot && cached[dev]) {
        *base = cached[dev];
        return cudaSuccess;
    }
    void *p = nullptr;
    e = cudaGetSymbolAddress(&p, rfa_static_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    if (slot) cached[dev] = (unsigned char *)p;
    *base = (unsigned char *)p;
    return cudaSuccess;
}

// Step 1 of a recorded run: put the caller's probe list at the head of the scratch (asynchronous on `st`; a pageable host
// list has been read by the time the call returns).
cudaError_t rfa_static_record_begin(int n_probes, const long long *index_host, cudaStream_t st)
{
    unsigned char *base = nullptr;
    cudaError_t e = static_scratch_base(&base);
    if (e != cudaSuccess) return e;
    return cudaMemcpyAsync(base, index_host, (size_t)n_probes * sizeof(long long), cudaMemcpyHostToDevice, st);
}

// Step 2, once per record: the probe kernel of rfa_step_record, reading the list from and writing row `row` to the scratch.
cudaError_t rfa_static_record_probe(const RfaGrid &g, int n_probes, const float *theta, size_t row, cudaStream_t st)
{
    unsigned char *base = nullptr;
    cudaError_t e = static_scratch_base(&base);
    if (e != cudaSuccess) return e;
    const long long *index_dev = (const long long *)base;
    float *rows = (float *)(base + RFA_STATIC_INDEX_BYTES);
    return rfa_launch_probe(g, n_probes, index_dev, theta, rows + row * (size_t)n_probes, st);
}

// Step 3: the first `floats` recorded values to the caller's buffer (host or device; asynchronous on `st`).
cudaError_t rfa_static_record_fetch(float *out, size_t floats, cudaStream_t st)
{
    unsigned char *base = nullptr;
    cudaError_t e = static_scratch_base(&base);
    if (e != cudaSuccess) return e;
    return cudaMemcpyAsync(out, base + RFA_STATIC_INDEX_BYTES, floats * sizeof(float), cudaMemcpyDefault, st);
}
