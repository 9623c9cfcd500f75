// merge_static.cu -- ising_merge_lists_static: the list merge of ising_merge_lists (the
// low_en / low_st merge) for callers that must not allocate device memory.
//
// Who that is. ising_merge_lists takes its sort scratch from the per-thread workspace, and the first call of a host
// thread creates that workspace with about a dozen cudaMalloc calls (two 64 MiB candidate pools among them). That is
// wrong for a caller that only ever merges -- the rank-local collector thread of a sharded run, say -- and it is
// impossible for a caller that runs where cudaMalloc cannot succeed or cannot be afforded: a process whose HBM has
// been handed over in full to another component's memory pool (a training or serving framework that reserves the
// device up front leaves the driver nothing to give), or a latency-critical section in which the device-wide
// synchronisation that cudaMalloc / cudaFree imply would stall every other stream of the process.
//
// What this file does instead. The scratch is the file-scope device array below: ISING_MERGE_STATIC_MAX entries of
// 16 bytes = 2 MiB, part of the library image, so every GPU that loads the library carries it until the process
// exits whether or not this entry point is ever called. In HOST code the array's name is only a handle for the
// runtime, not a device address (a kernel handed `s_merge_scratch` itself would fault, or scribble over host memory
// where the GPU can reach it); the device address is looked up once per device with cudaGetSymbolAddress -- in this
// file, because the symbol is only visible here -- and that pointer is what the kernels get.
//
// Contract (also in include/ising.h):
//  * no cudaMalloc, cudaFree, cudaMallocHost or allocating library routine, on the first call or any later one;
//  * the FIRST call on each device does the address lookup and sets the sort kernels' shared-memory attribute; make
//    that call before starting any stream capture;
//  * n > ISING_MERGE_STATIC_MAX is refused with ISING_ERR_BAD_S and a message naming the limit, before any CUDA work;
//  * every call on a device uses the same array. Nothing in it has to start at zero: each call first writes its n
//    packed entries and the sort pads the rest of its power-of-two extent with sentinels, so what the previous call
//    left behind is never read. Two calls that overlap on the GPU (different streams, different host threads) race
//    on the array and both results are garbage: serialise them.
#include <mutex>

#include "common.cuh"
#include "../../include/ising.h"

namespace ising {
namespace {

static_assert((ISING_MERGE_STATIC_MAX & (ISING_MERGE_STATIC_MAX - 1)) == 0,
              "the sort pads to the next power of two: the limit must be one, or the padding would run past the array");
static_assert(sizeof(Entry) == 16, "size of the scratch array as documented (2 MiB)");

// The scratch. Raw bytes, viewed as Entry[ISING_MERGE_STATIC_MAX] by the kernels.
static __device__ __align__(256) unsigned char s_merge_scratch[sizeof(Entry) * (size_t)ISING_MERGE_STATIC_MAX];

constexpr int MAX_DEVICES = 64;
std::mutex s_setup_mutex;
Entry* s_scratch_on_device[MAX_DEVICES];          // device address of s_merge_scratch, per device; nullptr = not set up

// Once per device, with that device current: resolve the array's device address, and let the sort kernels use their
// 64 KiB shared-memory tile (a per-device function attribute, no allocation). Returns ISING_OK or ISING_ERR_CUDA.
int scratch_for_current_device(Entry** out)
{
    int dev = -1;
    cudaError_t err = cudaGetDevice(&dev);
    if (err != cudaSuccess) { set_last_error(cudaGetErrorString(err)); return ISING_ERR_CUDA; }
    if (dev < 0 || dev >= MAX_DEVICES) { set_last_error("device ordinal beyond the static table of this entry point"); return ISING_ERR_CUDA; }
    std::lock_guard<std::mutex> lock(s_setup_mutex);
    if (!s_scratch_on_device[dev]) {
        void* p = nullptr;
        err = cudaGetSymbolAddress(&p, s_merge_scratch);
        if (err != cudaSuccess || !p) {
            set_last_error(err != cudaSuccess ? cudaGetErrorString(err) : "cudaGetSymbolAddress returned a null address");
            return ISING_ERR_CUDA;
        }
        set_select_attributes();
        err = cudaGetLastError();
        if (err != cudaSuccess) { set_last_error(cudaGetErrorString(err)); return ISING_ERR_CUDA; }
        s_scratch_on_device[dev] = static_cast<Entry*>(p);
    }
    *out = s_scratch_on_device[dev];
    return ISING_OK;
}

}  // namespace
}  // namespace ising

using namespace ising;

extern "C" int ising_merge_lists_static(const uint64_t* states_in_dev, const double* energies_in_dev, int64_t n, int S,
                                        uint64_t* states_out_dev, double* energies_out_dev, void* stream)
{
    set_last_error("");
    if (!states_in_dev || !energies_in_dev || !states_out_dev || !energies_out_dev) {
        set_last_error("null pointer argument");
        return ISING_ERR_NULL;
    }
    if (n > (int64_t)ISING_MERGE_STATIC_MAX) {
        set_last_error("n exceeds ISING_MERGE_STATIC_MAX (131072 entries, the static scratch of ising_merge_lists_static); "
                       "use ising_merge_lists, which allocates");
        return ISING_ERR_BAD_S;
    }
    if (n < 1 || S < 1 || S > n) { set_last_error("bad n or S"); return ISING_ERR_BAD_S; }
    Entry* scratch = nullptr;
    const int rc = scratch_for_current_device(&scratch);
    if (rc != ISING_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    // the same three steps as ising_merge_lists (pack -> bitonic sort by (energy, q) -> emit the first S), on `scratch`
    launch_merge_lists((const unsigned long long*)states_in_dev, energies_in_dev, n, S, scratch,
                       (unsigned long long*)states_out_dev, energies_out_dev, st);
    cudaError_t err = cudaGetLastError();
    if (err == cudaSuccess) err = cudaStreamSynchronize(st);
    if (err != cudaSuccess) { set_last_error(cudaGetErrorString(err)); return ISING_ERR_CUDA; }
    return ISING_OK;
}
