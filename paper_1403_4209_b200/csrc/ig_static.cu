// ig_static.cu - ig_grid_static: ig_grid for callers that have no way of getting a work buffer.
//
// Who this is for. ig_grid wants a work_dev area sized per batch (ig_workspace_bytes), and somebody has to
// cudaMalloc it. Some users of this library cannot: a gridding stage loaded into a correlator's or another
// framework's process gets its grid, bank and visibility buffers handed to it and is told not to touch the
// device heap, because the host application has already reserved the rest of HBM for its own pool (a late
// cudaMalloc then fails or fragments that pool); and a streaming loop with a latency budget cannot afford
// cudaMalloc / cudaFree at all, since both synchronise the whole device and stall every other stream.
// For them the scratch lives in the library image itself: a file-scope __device__ array that the CUDA runtime
// places in device memory when this module is loaded on a GPU and keeps there until the process exits.
//
// What it costs. IG_STATIC_WORK_BYTES (32 MiB) of HBM on every GPU that runs this entry point, for the life of the
// process, whether or not another call follows. There is one array per GPU, not per context: every call on
// that GPU uses the same bytes.
#include <mutex>
#include "ig_internal.h"

#define IG_STATIC_MAX_DEVICES 64

// The scratch itself. In HOST code this name is only a handle for the runtime (a host-side shadow variable):
// taking its address there does not give device memory. Host code must ask the runtime where the array sits
// on the current device (static_work_on_current_device below); device code could name it directly.
static __device__ __align__(256) unsigned char ig_static_work[IG_STATIC_WORK_BYTES];

namespace {
std::mutex g_mutex;                              // guards g_addr (first call per device from several host threads)
char* g_addr[IG_STATIC_MAX_DEVICES] = {};        // device address of ig_static_work, per device ordinal

// Set-up, once per device: the array has its own address on every GPU, so the lookup is made with that GPU
// current and cached under its ordinal. Loads this module on the device if no call has done so yet.
cudaError_t static_work_on_current_device(int* dev_out, char** ptr_out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= IG_STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_mutex);
    if (!g_addr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, ig_static_work);
        if (e != cudaSuccess) return e;
        if (!p || ((uintptr_t)p & 255)) return cudaErrorInvalidSymbol;
        g_addr[dev] = (char*)p;
    }
    *dev_out = dev;
    *ptr_out = g_addr[dev];
    return cudaSuccess;
}
}  // namespace

extern "C" ig_status ig_grid_static(ig_ctx* c, const double* uvw, const int* baseline_id, long long nrow,
                                    const double* freqs, int nchan, const float* vis, const float* wt) {
    if (!c) return IG_EINVAL;
    if (!c->bound || !c->have_bank) { c->err = "ig_grid_static: ig_bind and ig_build_wkernels first"; return IG_ESTATE; }
    if (nrow < 0 || nchan < 1 || !freqs) { c->err = "ig_grid_static: bad nrow/nchan/freqs"; return IG_EINVAL; }
    const size_t need = ig_workspace_bytes(c, nrow, nchan);
    if (need > (size_t)IG_STATIC_WORK_BYTES) {
        c->err = "ig_grid_static: a batch of " + std::to_string(nrow) + " rows x " + std::to_string(nchan) +
                 " channels needs " + std::to_string(need) + " bytes of scratch (ig_workspace_bytes), the built-in area holds " +
                 std::to_string((size_t)IG_STATIC_WORK_BYTES) + " (IG_STATIC_WORK_BYTES): feed smaller batches, or bind a work buffer and call ig_grid";
        return IG_ENOMEM;
    }
    int dev = -1;
    char* scratch = nullptr;
    cudaError_t e = static_work_on_current_device(&dev, &scratch);
    if (e != cudaSuccess) {
        c->err = std::string("ig_grid_static: cannot locate the built-in scratch area on the current device: ") + cudaGetErrorString(e);
        return IG_ECUDA;
    }
    // the array found above belongs to the CURRENT device; the context's buffers must live there too
    cudaPointerAttributes at{};
    e = cudaPointerGetAttributes(&at, c->grid);
    if (e != cudaSuccess) { c->err = std::string("ig_grid_static: ") + cudaGetErrorString(e); return IG_ECUDA; }
    if (at.type == cudaMemoryTypeDevice && at.device != dev) {
        c->err = "ig_grid_static: the bound grid lives on device " + std::to_string(at.device) + " but device " +
                 std::to_string(dev) + " is current";
        return IG_EINVAL;
    }
    // ig_grid, unchanged, with the built-in area in place of the bound work buffer for the length of this call.
    // ig_grid treats its workspace as undefined on entry and clears what it counts in (work-item maxima, gather
    // counts, plan bins), so nothing of the previous call's contents is read.
    char* const bound_work = c->work;
    const size_t bound_bytes = c->work_bytes;
    c->work = scratch;
    c->work_bytes = (size_t)IG_STATIC_WORK_BYTES;
    const ig_status st = ig_grid(c, uvw, baseline_id, nrow, freqs, nchan, vis, wt);
    c->work = bound_work;
    c->work_bytes = bound_bytes;
    return st;
}
