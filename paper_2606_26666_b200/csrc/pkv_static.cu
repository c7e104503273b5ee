// pkv_static.cu -- pkv_decode_static: one decode step that takes NO workspace from the caller and
// makes no device allocation (include/pkv.h "Allocation-free entry point").
//
// The scratch memory of a decode step -- the queue header with its counters, split_offsets, the
// task list and the partial states (m, l, acc) of split rows -- lives in the
// file-scope __device__ array below instead of a caller-provided workspace.  Everything else is
// the existing path: the call ends in pkv_decode(build_queue = 1) on that array's device address.
//
// The array's NAME is not a device address in host code (it is the host-side stand-in the runtime
// registers the symbol under).  The address is looked up once per device, with that device
// current, by cudaGetSymbolAddress in this file, and only that pointer is handed to the kernels.
// Device code in this file names the array directly (pkv_static_clear_kernel).
//
// One array per GPU and per process: all calls on a device share it and it keeps the last call's
// contents.  Every call therefore clears the part of the layout that must start at zero
// (pkv_workspace_init_bytes: queue header, scheduler and completion counters, error word) before
// the decode kernel runs; the queue and the partial states are rewritten by every step before
// they are read.  Two calls that overlap on the GPU (different streams, or two host threads on
// different streams) race on the array: serialise them, or use pkv_decode with workspaces of
// your own.
#include <cuda_runtime.h>

#include <mutex>

#include "pkv_common.h"

namespace pkv {
namespace {

// Held by every GPU that loads the library, from module load until the process exits.
static __device__ __align__(256) unsigned char g_static_workspace[PKV_STATIC_WORKSPACE_BYTES];

constexpr int kMaxDevices = 64;
std::mutex g_static_mutex;
void* g_static_ptr[kMaxDevices] = {};   // device address of g_static_workspace on device i; null = not looked up yet

// Zeroes the first `bytes` (a multiple of 16) of the array.  Not a programmatic-launch primary: it
// never triggers its dependents early, so the decode kernel launched behind it passes its
// dependency wait only after these stores are complete and visible.
__global__ void pkv_static_clear_kernel(unsigned int bytes) {
    uint4* w = reinterpret_cast<uint4*>(g_static_workspace);
    for (unsigned int i = blockIdx.x * blockDim.x + threadIdx.x; i < bytes / 16; i += gridDim.x * blockDim.x)
        w[i] = make_uint4(0u, 0u, 0u, 0u);
}

// Set-up, once per device: the array's address on the CURRENT device.
pkv_status static_workspace_address(void** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        set_error("pkv_decode_static: cudaGetDevice: %s", cudaGetErrorString(e));
        return PKV_ERR_CUDA;
    }
    if (dev < 0 || dev >= kMaxDevices) {
        set_error("pkv_decode_static: device ordinal %d outside 0..%d", dev, kMaxDevices - 1);
        return PKV_ERR_UNSUPPORTED;
    }
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (g_static_ptr[dev] == nullptr) {
        void* ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, g_static_workspace);
        if (e != cudaSuccess || ptr == nullptr) {
            set_error("pkv_decode_static: cudaGetSymbolAddress(static workspace) on device %d: %s", dev,
                      e != cudaSuccess ? cudaGetErrorString(e) : "null address");
            return PKV_ERR_CUDA;
        }
        g_static_ptr[dev] = ptr;
    }
    *out = g_static_ptr[dev];
    return PKV_OK;
}

}  // namespace
}  // namespace pkv

extern "C" {

size_t pkv_static_workspace_bytes(void) { return (size_t)PKV_STATIC_WORKSPACE_BYTES; }

pkv_status pkv_decode_static(const pkv_shape* shape, const pkv_split_policy* policy, const void* q, const void* k_cache,
                             const void* v_cache, const int32_t* block_table, const int32_t* seq_lens, void* out, float* lse,
                             float scale, void* stream) {
    using namespace pkv;
    clear_error();
    if (!shape || !policy) {
        set_error("pkv_decode_static: null shape or policy");
        return PKV_ERR_INVALID_ARG;
    }
    // Size first (host arithmetic only): a step that does not fit is refused before any CUDA call.
    const size_t need = pkv_workspace_bytes(shape, policy);
    if (need == 0) {
        // not a valid shape / policy: let the existing path name the reason (it fails in validation,
        // before it looks at the workspace or launches anything)
        return pkv_decode(shape, policy, q, k_cache, v_cache, block_table, seq_lens, out, lse, scale, 1, nullptr, 0, stream);
    }
    if (need > (size_t)PKV_STATIC_WORKSPACE_BYTES) {
        set_error("pkv_decode_static: this shape and policy need %zu bytes of scratch, the static workspace holds %zu "
                  "(PKV_STATIC_WORKSPACE_BYTES); lower num_splits or B, or call pkv_decode with a workspace of your own",
                  need, (size_t)PKV_STATIC_WORKSPACE_BYTES);
        return PKV_ERR_WORKSPACE;
    }
    void* ws = nullptr;
    pkv_status st = static_workspace_address(&ws);
    if (st != PKV_OK) return st;
    const size_t init = align_up(pkv_workspace_init_bytes(shape, policy), 16);
    cudaStream_t cs = static_cast<cudaStream_t>(stream);
    pkv_static_clear_kernel<<<1, 256, 0, cs>>>((unsigned int)init);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        set_error("pkv_decode_static: clear launch: %s", cudaGetErrorString(e));
        return PKV_ERR_CUDA;
    }
    return pkv_decode(shape, policy, q, k_cache, v_cache, block_table, seq_lens, out, lse, scale, 1, ws,
                      (size_t)PKV_STATIC_WORKSPACE_BYTES, stream);
}

}  // extern "C"
