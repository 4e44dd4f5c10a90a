// rqa_static.cu — rqa_line_hist_static: rqa_line_hist for callers that cannot allocate device memory.
//
// Every heavy call of the library works in a device workspace the CALLER allocates (rqa_workspace_bytes).  Code under
// CUDA-graph capture, a tight serving loop, or a harness that forbids cudaMalloc has nowhere to get one from.  This
// entry point is rqa_line_hist (same kernels, same results) with the workspace in a file-scope
// device array of RQA_STATIC_SCRATCH_BYTES: the caller passes only inputs and outputs, and the call makes no
// cudaMalloc / cudaFree / allocating library call (it launches kernels and cudaMemsetAsync on the given stream).
//
// Cost and limits, also stated in include/rqa.h:
//   * the array is part of this translation unit's device module: every GPU on which the process uses this entry point
//     holds RQA_STATIC_SCRATCH_BYTES of device memory from then until the process exits;
//   * a shape whose scan needs more scratch than that is rejected with RQA_ERR_UNSUPPORTED before anything is launched;
//   * ALL calls on one device share the one array, and it keeps the last call's contents.  The path clears what must
//     start at zero itself (status block, line aggregates, work counters: status_reset_kernel and the cudaMemsetAsync
//     calls at the head of run_line_hist; the segment summaries and carries are written before they are read), so
//     calls in stream order are independent — but two calls that overlap on the GPU (different streams, or threads
//     without ordering between them) race on it.  Serialise them, or use rqa_line_hist with one workspace per stream.
#include <atomic>
#include <mutex>

#include "rqa_common.cuh"

namespace rqa {

namespace {

// The scratch.  In host code the NAME of a __device__ array is a host-side stand-in, not a device address (a kernel
// given `g_static_scratch` from the host would fault or touch unrelated memory): the address comes from
// cudaGetSymbolAddress, asked once per device with that device current.
static __device__ __align__(256) unsigned char g_static_scratch[RQA_STATIC_SCRATCH_BYTES];

constexpr int MAX_DEVICES = 64;
std::atomic<void*> g_scratch_ptr[MAX_DEVICES];
std::mutex g_scratch_mutex;

// Device address of the scratch on the CURRENT device (set-up on first use, then a table read).
rqa_status static_scratch(void** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        cudaGetLastError();
        set_error("rqa_line_hist_static: cudaGetDevice: %s", cudaGetErrorString(e));
        return RQA_ERR_CUDA;
    }
    if (dev < 0 || dev >= MAX_DEVICES) {
        set_error("rqa_line_hist_static: device ordinal %d outside 0..%d", dev, MAX_DEVICES - 1);
        return RQA_ERR_UNSUPPORTED;
    }
    void* p = g_scratch_ptr[dev].load(std::memory_order_acquire);
    if (!p) {
        std::lock_guard<std::mutex> lock(g_scratch_mutex);
        p = g_scratch_ptr[dev].load(std::memory_order_relaxed);
        if (!p) {
            e = cudaGetSymbolAddress((void**)&p, g_static_scratch);     // `dev` is current: its copy of the array
            if (e != cudaSuccess || !p) {
                cudaGetLastError();
                set_error("rqa_line_hist_static: cudaGetSymbolAddress(scratch) on device %d: %s", dev, cudaGetErrorString(e));
                return RQA_ERR_CUDA;
            }
            if (((uintptr_t)p & 255) != 0) {
                set_error("rqa_line_hist_static: scratch at %p is not 256-byte aligned", p);
                return RQA_ERR_CUDA;
            }
            g_scratch_ptr[dev].store(p, std::memory_order_release);
        }
    }
    *out = p;
    return RQA_OK;
}

}  // namespace

}  // namespace rqa

using namespace rqa;

extern "C" rqa_status rqa_line_hist_static(const rqa_points* pts, rqa_norm norm, const float* d_eps, int32_t K,
                                           uint64_t* d_hist, void* stream) {
    rqa_status st = validate_points(pts, "rqa_line_hist_static");
    if (st != RQA_OK) return st;
    if (norm != RQA_NORM_MAX && norm != RQA_NORM_EUCLID) { set_error("rqa_line_hist_static: unknown norm %d", (int)norm); return RQA_ERR_INVALID_ARG; }
    if (K < 1 || K > RQA_MAX_K) { set_error("rqa_line_hist_static: K = %d outside 1..%d", K, RQA_MAX_K); return RQA_ERR_INVALID_ARG; }
    if (!d_eps || !d_hist) { set_error("rqa_line_hist_static: NULL argument"); return RQA_ERR_INVALID_ARG; }
    // the size check comes first: it needs no device and nothing has been launched when it fails
    const View v = make_view(*pts);
    const size_t need = sizeof(WsStatus) + line_workspace_bytes(v, K, Options{});
    if (need > (size_t)RQA_STATIC_SCRATCH_BYTES) {
        set_error("rqa_line_hist_static: n_points = %lld, batch = %d, K = %d needs %zu bytes of scratch, the static "
                  "scratch holds RQA_STATIC_SCRATCH_BYTES = %zu; use rqa_line_hist with a caller workspace",
                  (long long)pts->n_points, pts->batch, K, need, (size_t)RQA_STATIC_SCRATCH_BYTES);
        return RQA_ERR_UNSUPPORTED;
    }
    void* scratch = nullptr;
    st = static_scratch(&scratch);
    if (st != RQA_OK) return st;
    // the scan of rqa_line_hist with every scratch pointer of its kernels carved out of the static array
    return rqa_line_hist_opt(pts, norm, d_eps, K, d_hist, scratch, (size_t)RQA_STATIC_SCRATCH_BYTES, stream, nullptr);
}
