// static_sort.cu — symdel_sort_u64_static: the onesweep LSD radix sort of radix_sort.cu (S2/K2; the sort of the
// sort-merge join, §I.B) for callers that have no way of handing the library device memory.
//
// Who that is.  symdel_stage_sort_u64 wants a ping-pong buffer of n keys and a block of status words from the caller,
// who normally gets them from cudaMalloc or a framework allocator.  Some callers cannot: a plug-in that runs inside a
// host application which claimed the whole device for its own pool at start-up (a raw cudaMalloc then fails, and the
// plug-in was given its input/output buffers and nothing else); a latency-bound service loop in which cudaMalloc /
// cudaFree are banned because both may synchronise the whole device and stall every other stream; code that runs
// after an out-of-memory condition and has to finish with what is already there.  For them the scratch lives in the
// library image itself: `static_scratch` below, a file-scope __device__ array that the driver places on every GPU
// that loads libsymdel.so and keeps there until the process exits (SYMDEL_STATIC_SORT_SCRATCH_BYTES = 11 MiB per GPU,
// which is what bounds the sort at SYMDEL_STATIC_SORT_MAX_KEYS = 2^20 keys).
//
// What to know before calling it.
//   * Nothing in this file, and nothing it calls, allocates or frees: no cudaMalloc* / cudaFree*, no stream, event or
//     context-object creation.  The CUDA calls made are cudaSetDevice, cudaGetSymbolAddress, cudaFuncSetAttribute
//     (first call per device only), cudaMemsetAsync, kernel launches, at most one device-to-device cudaMemcpyAsync,
//     and cudaStreamSynchronize.
//   * The first call on a device does the per-device set-up: it asks the runtime where `static_scratch` lives on that
//     device (in host code the array's name is only a handle for cudaGetSymbolAddress, never an address a kernel could
//     use) and raises the dynamic shared-memory limit of the sort kernels.  Make that first call outside any stream
//     capture; later calls find the address in a table and skip the set-up.
//   * There is ONE array per GPU and every call on that GPU uses it.  It still holds whatever the previous call left,
//     so each call zeroes the part that must start at zero (digit histograms, tile tickets, look-back status words)
//     on the caller's stream before its first kernel.  Two calls whose GPU work can overlap — different streams, or
//     different host threads, on the same device — would clear and count in the same words and overwrite each other's
//     ping-pong buffer: that is a data race with an undefined result.  Run them one after the other.
#include <mutex>

#include "../../include/symdel.h"
#include "kernels.h"

namespace {

constexpr i64 SS_MAX_KEYS = SYMDEL_STATIC_SORT_MAX_KEYS;
constexpr i64 SS_PING_BYTES = SS_MAX_KEYS * 8;                      // the second key buffer of the LSD passes
constexpr i64 SS_CTRL_BYTES = SYMDEL_STATIC_SORT_SCRATCH_BYTES - SS_PING_BYTES;  // histograms, tickets, status words
static_assert(SS_CTRL_BYTES > 0 && SS_PING_BYTES % 256 == 0, "scratch layout");

// [0, SS_PING_BYTES): ping-pong keys | [SS_PING_BYTES, end): control words of sd_sort_* (cleared by every call)
static __device__ __align__(256) unsigned char static_scratch[SYMDEL_STATIC_SORT_SCRATCH_BYTES];

constexpr int SS_MAX_DEVICES = 64;
std::mutex ss_lock;                                  // guards the table below
unsigned char* ss_base_of_device[SS_MAX_DEVICES];    // device address of static_scratch on each GPU; null = set-up not done yet

// Per-device set-up with `device` current.  SYMDEL_OK, SYMDEL_E_CUDA or SYMDEL_E_INTERNAL.
int ss_base(int device, unsigned char** base) {
    std::lock_guard<std::mutex> g(ss_lock);
    if (!ss_base_of_device[device]) {
        if (sd_sort_scratch_bytes(SS_MAX_KEYS, 8) > SS_CTRL_BYTES) return SYMDEL_E_INTERNAL;  // the tile shapes outgrew the array
        unsigned char* p = nullptr;
        if (cudaGetSymbolAddress((void**)&p, static_scratch) != cudaSuccess || !p) return SYMDEL_E_CUDA;
        if (sd_sort_setup() != cudaSuccess) return SYMDEL_E_CUDA;  // what symdel_create does for the sort kernels (idempotent)
        ss_base_of_device[device] = p;
    }
    *base = ss_base_of_device[device];
    return SYMDEL_OK;
}

}  // namespace

extern "C" int symdel_sort_u64_static(int device, uint64_t* keys, int64_t n, int begin_bit, int end_bit, void* cuda_stream) {
    if (n < 0 || begin_bit < 0 || end_bit > 64 || end_bit < begin_bit || (end_bit - begin_bit) % 8 != 0 || device < 0 ||
        device >= SS_MAX_DEVICES)
        return SYMDEL_E_ARG;
    if (n > SS_MAX_KEYS) return SYMDEL_E_STATIC_LIMIT;  // before anything touches the GPU: the array cannot grow
    if (n == 0 || end_bit == begin_bit) return SYMDEL_OK;
    if (!keys) return SYMDEL_E_ARG;
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || device >= count) return SYMDEL_E_CUDA;
    if (cudaSetDevice(device) != cudaSuccess) return SYMDEL_E_CUDA;
    unsigned char* base = nullptr;
    const int rc = ss_base(device, &base);
    if (rc != SYMDEL_OK) return rc;
    u64* ping = reinterpret_cast<u64*>(base);
    void* ctrl = base + SS_PING_BYTES;
    const int npass = (end_bit - begin_bit) / 8;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    u64* res = nullptr;
    // same sequence as symdel_stage_sort_u64, stable, default tile shape; the clear comes first because the
    // array still holds the last call's counts and status words
    if (sd_sort_prepare(ctrl, n, npass, st) != cudaSuccess) return SYMDEL_E_CUDA;
    if (sd_sort_histogram(keys, n, begin_bit, npass, ctrl, st, nullptr) != cudaSuccess) return SYMDEL_E_CUDA;
    if (sd_sort_hist_scan(ctrl, npass, st, nullptr) != cudaSuccess) return SYMDEL_E_CUDA;
    if (sd_sort_passes(keys, ping, n, nullptr, begin_bit, npass, 1, 0, ctrl, st, &res, nullptr) != cudaSuccess) return SYMDEL_E_CUDA;
    if (res != keys && cudaMemcpyAsync(keys, res, (size_t)n * 8, cudaMemcpyDeviceToDevice, st) != cudaSuccess) return SYMDEL_E_CUDA;
    if (cudaStreamSynchronize(st) != cudaSuccess) return SYMDEL_E_CUDA;
    return SYMDEL_OK;
}
