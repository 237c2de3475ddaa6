// static_ws.cu -- polylab_simplify_static: simplify (S0..S5, Table 3, section 6.3) for callers that
// can neither allocate device memory nor hand over a workspace: code under CUDA graph capture set-up, tight serving loops,
// harnesses that forbid cudaMalloc.  The scratch memory every kernel of the pipeline works in (control block, tile states,
// key/coefficient ping-pong buffers, the table path's slots) lives in ONE file-scope __device__ array of
// POLYLAB_STATIC_WORKSPACE_BYTES; every GPU whose context loads the library holds it until the process exits.
//
// In host code `g_static_ws` is a host-side stand-in for the array, not a device address: the address is asked for once per
// device (cudaGetSymbolAddress, with that device current) and cached.  All calls share the array and it keeps the previous
// call's contents: polylab_simplify never assumes a zeroed workspace -- each call clears the control block, the tile states
// and the table region it is about to use -- so nothing else needs clearing here.  Two calls that overlap on one GPU (different
// streams, or two host threads) race on the array; the caller serialises them.
#include <mutex>

#include "kernels.h"

namespace polylab {

__device__ __align__(256) unsigned char g_static_ws[POLYLAB_STATIC_WORKSPACE_BYTES];

constexpr int kMaxStaticDevices = 64;

// device address of g_static_ws on the CURRENT device (nullptr: see *err)
static void* static_workspace(cudaError_t* err)
{
    static std::mutex mu;
    static void* addr[kMaxStaticDevices];          // zero-initialised
    int dev = -1;
    *err = cudaGetDevice(&dev);
    if (*err != cudaSuccess) return nullptr;
    if (dev < 0 || dev >= kMaxStaticDevices) { *err = cudaErrorInvalidDevice; return nullptr; }
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        void* p = nullptr;
        *err = cudaGetSymbolAddress(&p, g_static_ws);
        if (*err != cudaSuccess) return nullptr;
        addr[dev] = p;
    }
    return addr[dev];
}

}  // namespace polylab

using namespace polylab;

extern "C" {

int polylab_simplify_static(const double* coef, const void* exps, int64_t nterms, int32_t nvars, double tol, const polylab_opts* opts,
                            double* out_coef, void* out_exps, int64_t out_capacity, int64_t* out_nterms, void* cuda_stream)
{
    if (nterms < 0 || nvars < 1) return POLYLAB_ERR_INVALID_ARGUMENT;
    if (opts && (opts->flags & POLYLAB_FLAG_TIMING)) return POLYLAB_ERR_INVALID_ARGUMENT;     // stage events would be created
    // the stated limit first, then the layout itself (the static array must hold the worst case of every path)
    if (nterms > POLYLAB_STATIC_MAX_TERMS) return POLYLAB_ERR_WORKSPACE_TOO_SMALL;
    const size_t need = polylab_simplify_workspace_bytes(nterms, nvars, opts);
    if (need == 0 || need > (size_t)POLYLAB_STATIC_WORKSPACE_BYTES) return POLYLAB_ERR_WORKSPACE_TOO_SMALL;
    cudaError_t err = cudaSuccess;
    void* ws = static_workspace(&err);
    if (!ws) { note_cuda_error(err, "cudaGetSymbolAddress(g_static_ws)"); return POLYLAB_ERR_CUDA; }
    return polylab_simplify(coef, exps, nterms, nvars, tol, opts, out_coef, out_exps, out_capacity, out_nterms, ws,
                            (size_t)POLYLAB_STATIC_WORKSPACE_BYTES, cuda_stream);
}

}  // extern "C"
