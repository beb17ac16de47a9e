// nasg_noalloc.cu — nasg_eval_bwd_noalloc (include/nasg.h): the backward pass with the per-camera gradient
// g_campos, for callers that have no device buffer to hand over as `workspace` and no way of making one.
//
// Who that is. nasg_eval_bwd needs nasg_workspace_bytes(N, K, C) of device scratch for the per-block partial sums
// of g_campos, and leaves it to the caller to provide them. Some callers can't: a plug-in that is handed its
// tensors by a host application (a viewer, a trainer with its own caching allocator) and must not call cudaMalloc
// behind that application's memory accounting; a real-time render loop, where cudaMalloc / cudaFree synchronise
// the whole device and would stall the frame; a process whose device memory was carved up and handed out at
// start-up, so that a late cudaMalloc simply fails; a C caller that links this library but not the CUDA runtime
// and has no allocation call to make at all. For them the scratch lives inside the library image: a fixed array
// in device global memory that exists from the moment the module is loaded on a GPU until the process exits.
// No call allocates, frees or resizes anything.
//
// The kernels are the ones nasg_eval_bwd launches (same instantiations, same grids, same fixed summation
// order); only the address of the partial sums differs.
#include "nasg.h"
#include "nasg_internal.h"

#include <atomic>
#include <mutex>

// The scratch itself: NASG_NOALLOC_WS_BYTES (1 MiB) of device memory per GPU that loads the library, held until
// the process exits whether or not nasg_eval_bwd_noalloc is ever called. 256-byte alignment = that of cudaMalloc.
static __device__ __align__(256) float g_noalloc_ws[NASG_NOALLOC_WS_BYTES / sizeof(float)];

namespace {

constexpr int MAX_DEVICES = 64;
std::atomic<float *> g_ws_addr[MAX_DEVICES];      // device address of g_noalloc_ws, per device ordinal (zero-initialised)
std::mutex g_ws_mutex;

// In host code `g_noalloc_ws` is only a handle of the symbol (an address in the HOST image); handing it to a kernel
// makes the kernel fault, or scribble over host memory on systems where the GPU can reach it. The device address
// must be asked for, per device (every GPU has its own copy of the array), with that device current. Done once per
// device on the first call there; it may load the module on that device, which is why the header asks for this
// first call to come before any stream capture.
int noalloc_ws(float **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return nasg::api_cuda_fail(e);
    if (dev < 0 || dev >= MAX_DEVICES) return nasg::api_cuda_fail(cudaErrorInvalidDevice);
    float *p = g_ws_addr[dev].load(std::memory_order_acquire);
    if (!p) {
        std::lock_guard<std::mutex> lock(g_ws_mutex);
        p = g_ws_addr[dev].load(std::memory_order_relaxed);
        if (!p) {
            void *sym = nullptr;
            e = cudaGetSymbolAddress(&sym, g_noalloc_ws);
            if (e != cudaSuccess) return nasg::api_cuda_fail(e);
            if (!sym) return nasg::api_cuda_fail(cudaErrorInvalidSymbol);
            p = static_cast<float *>(sym);
            g_ws_addr[dev].store(p, std::memory_order_release);
        }
    }
    *out = p;
    return NASG_OK;
}

inline bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
inline bool supported_K(int K) { return K == 1 || K == 2 || K == 3 || K == 4 || K == 5 || K == 8; }

} // namespace

extern "C" {

size_t nasg_noalloc_workspace_bytes(void) { return NASG_NOALLOC_WS_BYTES; }

int nasg_eval_bwd_noalloc(const nasg_inputs *in, const float *g_colors, const nasg_grads *out, int norm_mode,
                          void *cuda_stream)
{
    if (!in || !out) return NASG_ERR_NULL;
    if (in->N < 0 || in->C < 1 || in->C > NASG_MAX_CAMERAS) return NASG_ERR_SHAPE;
    if (!supported_K(in->K)) return NASG_ERR_UNSUPPORTED_K;
    if (norm_mode != NASG_NORM_APPROX && norm_mode != NASG_NORM_EXACT && norm_mode != NASG_NORM_NASG) return NASG_ERR_NORM_MODE;
    if (!out->g_campos) return NASG_ERR_NULL;                 // without g_campos there is no scratch: use nasg_eval_bwd
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (in->N == 0) {
        cudaError_t e = cudaMemsetAsync(out->g_campos, 0, sizeof(float) * 3 * in->C, st);
        return e == cudaSuccess ? NASG_OK : nasg::api_cuda_fail(e);
    }
    if (!in->means || !in->quat || !in->shape || !in->amp || !in->dc || !in->campos || !g_colors) return NASG_ERR_NULL;
    if (!aligned16(in->quat) || !aligned16(in->shape) || !aligned16(out->g_quat) || !aligned16(out->g_shape))
        return NASG_ERR_ALIGN;
    // The size test is nasg_eval_bwd's own (rows of partial sums for the largest grid any kernel family launches),
    // against the fixed capacity instead of the caller's workspace_bytes.
    if (nasg_workspace_bytes(in->N, in->K, in->C) > (size_t)NASG_NOALLOC_WS_BYTES) return NASG_ERR_NOALLOC_SIZE;

    float *partial = nullptr;
    int rc = noalloc_ws(&partial);
    if (rc != NASG_OK) return rc;

    // Every row of `partial` the reduction below reads is written, in full, by the backward launch in front of it
    // on the same stream (each block stores its 3 C sums; the reduction reads exactly the blocks launched), so the
    // previous call's contents never show through and nothing has to be cleared first.
    nasg::BwdParams p{in->N, in->C, in->means, in->quat, in->shape, in->amp, in->campos, in->vis, g_colors,
                      out->g_means, out->g_quat, out->g_shape, out->g_amp, out->g_dc, partial};
    const bool pipe = in->C <= 4;                             // the persistent ring kernels; more cameras: the generic ones
    int pipe_blocks = 0;
    cudaError_t e = pipe ? nasg::launch_nasg_bwd_pipe(p, in->K, norm_mode, st, &pipe_blocks)
                         : nasg::launch_nasg_bwd(p, in->K, norm_mode, st);
    if (e != cudaSuccess) return nasg::api_cuda_fail(e);
    nasg::api_count_launches(1);
    e = nasg::launch_campos_reduce(partial, pipe ? pipe_blocks : nasg::grid_blocks(in->N), in->C, out->g_campos, st);
    if (e != cudaSuccess) return nasg::api_cuda_fail(e);
    nasg::api_count_launches(1);
    return NASG_OK;
}

} // extern "C"
