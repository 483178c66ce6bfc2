// no_alloc.cu -- cute_count_pairs_static: the pair count for callers that have no device memory to spare for
// its scratch and no way of getting any.
//
// Who that is.  Everywhere else in this library the caller hands over every byte of device memory, including the
// few hundred bytes of scratch (work counter, status word, statistics, bin edges) the pair kernel needs next to
// its inputs and its histogram.  Some callers cannot produce even that: an in-situ analysis hook inside an N-body
// code whose own memory manager took the whole device at start-up and hands the hook nothing but the particle
// arrays and a histogram to fill; a plug-in that runs under a host application's fixed memory budget; a thread
// that must not call cudaMalloc because the allocation would synchronise the device under a latency-critical
// loop, or because another thread of the process is recording a stream and an allocation there is an error.
// For them the scratch lives in the library image itself: a file-scope __device__ array that every GPU which
// loads the library carries until the process exits (kStaticBytes per device, nothing else).
//
// What the array is and is not.  In host code the name g_static_scratch is only a handle for the runtime, NOT a
// device address: handing it to a kernel would fault, or, on a system where the GPU can reach host memory,
// quietly use the wrong bytes.  The device address is asked for with cudaGetSymbolAddress, once per device and
// with that device current, and that pointer is what the kernel receives (it goes in exactly where the caller's
// d_scratch goes in cute_count_pairs; nothing else about the count differs).
#include "cute_internal.h"

#include <mutex>

namespace {

constexpr size_t kStaticBytes = CUTE_STATIC_SCRATCH_BYTES;
static_assert(kStaticBytes % 256 == 0, "the scratch layout is 256-byte granular");

static __device__ __align__(256) unsigned char g_static_scratch[kStaticBytes];

constexpr int kMaxDevices = 64;
std::mutex g_lock[kMaxDevices];      // one per device: set-up, and the array's single user at a time
void *g_addr[kMaxDevices];           // device address of g_static_scratch on device d (nullptr: not asked yet)

} // namespace

extern "C" int cute_count_pairs_static(int kind, const cute_grid *g1, const cute_grid *g2, const cute_bin_spec *bins,
                                       uint64_t *d_hist, const cute_count_opts *opts, void *stream, uint64_t stats[4])
{
    // the size test comes first and touches no CUDA state: binning too fine for the fixed array is refused outright
    size_t need = 0;
    int rc = cute_count_scratch_bytes(bins, opts, &need);
    if (rc) return rc;
    if (need > kStaticBytes) return CUTE_ERR_STATIC_SCRATCH_LIMIT;

    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return CUTE_ERR_CUDA;
    if (dev < 0 || dev >= kMaxDevices) return CUTE_ERR_UNSUPPORTED;

    // Every call on this device uses the same bytes.  Two counts in flight at once would share one work counter and
    // overwrite each other's bin edges, so the lock is held until this call's work has left the GPU (the status
    // read below synchronises the stream).  That orders the calls of one process; it cannot order anything else.
    std::lock_guard<std::mutex> hold(g_lock[dev]);
    if (!g_addr[dev]) {
        void *p = nullptr;
        if (cudaGetSymbolAddress(&p, g_static_scratch) != cudaSuccess || !p) return CUTE_ERR_CUDA;
        g_addr[dev] = p;
    }
    // The array still holds whatever the previous count left there.  cute_count_pairs starts by zeroing the work
    // counter, status word and statistics on the stream and copies in this call's bin edges; it reads nothing else.
    rc = cute_count_pairs(kind, g1, g2, bins, d_hist, g_addr[dev], kStaticBytes, opts, stream);
    if (rc < 0) return rc;
    return cute_count_status(g_addr[dev], stream, stats);
}
