// nasg_api.cu — the extern "C" boundary declared in include/nasg.h: argument validation, dispatch
// to the kernel launchers, and the host-buffer end-to-end entry points. No arithmetic of the
// method lives here.
#include "nasg.h"
#include "nasg_internal.h"

#include <atomic>
#include <cstdlib>

namespace {

std::atomic<int64_t> g_launches{0};
thread_local cudaError_t t_last_cuda = cudaSuccess;

inline bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
inline bool supported_K(int K) { return K == 1 || K == 2 || K == 3 || K == 4 || K == 5 || K == 8; }
inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

// C <= 4 runs the persistent cp.async-pipelined kernels; NASG_FORCE_GENERIC=1 (debug/AB testing) or a
// larger camera batch runs the generic ones.
bool use_pipe(int C)
{
    static const bool force_generic = [] { const char *e = getenv("NASG_FORCE_GENERIC"); return e && e[0] == '1'; }();
    return C <= 4 && !force_generic;
}

int cuda_fail(cudaError_t e) { t_last_cuda = e; return NASG_ERR_CUDA; }

int check_inputs(const nasg_inputs *in)
{
    if (!in) return NASG_ERR_NULL;
    if (in->N < 0 || in->C < 1 || in->C > NASG_MAX_CAMERAS) return NASG_ERR_SHAPE;
    if (!supported_K(in->K)) return NASG_ERR_UNSUPPORTED_K;
    if (in->N == 0) return NASG_OK;
    if (!in->means || !in->quat || !in->shape || !in->amp || !in->dc || !in->campos) return NASG_ERR_NULL;
    return NASG_OK;
}

size_t cam_partial_bytes(int64_t N, int C) { return (size_t)nasg::grid_blocks(N) * (size_t)C * 3 * sizeof(float); }

// carves aligned sub-buffers out of the caller's device scratch (host-buffer entry points)
struct Carver {
    char *base; size_t off, cap;
    template <typename T> T *take(size_t count)
    {
        size_t bytes = align_up(count * sizeof(T));
        if (off + bytes > cap) { off = cap + 1; return nullptr; }
        T *p = reinterpret_cast<T *>(base + off);
        off += bytes;
        return p;
    }
};
#define NASG_TRY_CUDA(expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) return cuda_fail(e_); } while (0)

} // namespace

extern "C" {

int nasg_eval_fwd(const nasg_inputs *in, float *colors, int norm_mode, void *cuda_stream)
{
    int rc = check_inputs(in);
    if (rc != NASG_OK) return rc;
    if (norm_mode != NASG_NORM_APPROX && norm_mode != NASG_NORM_EXACT) return NASG_ERR_NORM_MODE;
    if (in->N == 0) return NASG_OK;
    if (!colors) return NASG_ERR_NULL;
    if (!aligned16(in->quat) || !aligned16(in->shape)) return NASG_ERR_ALIGN;
    nasg::FwdParams p{in->N, in->C, in->means, in->quat, in->shape, in->amp, in->dc, in->campos, in->vis, colors};
    const bool exact = norm_mode == NASG_NORM_EXACT;
    cudaError_t e = use_pipe(in->C) ? nasg::launch_nasg_fwd_pipe(p, in->K, exact, (cudaStream_t)cuda_stream)
                                    : nasg::launch_nasg_fwd(p, in->K, exact, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return NASG_OK;
}

int nasg_eval_bwd(const nasg_inputs *in, const float *g_colors, const nasg_grads *out, int norm_mode,
                  void *cuda_stream)
{
    int rc = check_inputs(in);
    if (rc != NASG_OK) return rc;
    if (norm_mode != NASG_NORM_APPROX && norm_mode != NASG_NORM_EXACT) return NASG_ERR_NORM_MODE;
    if (!out) return NASG_ERR_NULL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (in->N == 0) {
        if (out->g_campos) {
            cudaError_t e = cudaMemsetAsync(out->g_campos, 0, sizeof(float) * 3 * in->C, st);
            if (e != cudaSuccess) return cuda_fail(e);
        }
        return NASG_OK;
    }
    if (!g_colors) return NASG_ERR_NULL;
    if (!aligned16(in->quat) || !aligned16(in->shape) || !aligned16(out->g_quat) || !aligned16(out->g_shape))
        return NASG_ERR_ALIGN;
    float *partial = nullptr;
    if (out->g_campos) {
        if (!out->workspace || out->workspace_bytes < cam_partial_bytes(in->N, in->C)) return NASG_ERR_WORKSPACE;
        partial = static_cast<float *>(out->workspace);
    }
    nasg::BwdParams p{in->N, in->C, in->means, in->quat, in->shape, in->amp, in->campos, in->vis, g_colors,
                      out->g_means, out->g_quat, out->g_shape, out->g_amp, out->g_dc, partial};
    const bool exact = norm_mode == NASG_NORM_EXACT;
    cudaError_t e = (use_pipe(in->C) && !partial) ? nasg::launch_nasg_bwd_pipe(p, in->K, exact, st)
                                                  : nasg::launch_nasg_bwd(p, in->K, exact, st);
    if (e != cudaSuccess) return cuda_fail(e);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    if (partial) {
        e = nasg::launch_campos_reduce(partial, nasg::grid_blocks(in->N), in->C, out->g_campos, st);
        if (e != cudaSuccess) return cuda_fail(e);
        g_launches.fetch_add(1, std::memory_order_relaxed);
    }
    return NASG_OK;
}

int sh_eval_fwd(int64_t N, int32_t C, const float *means, const float *coeffs, const float *campos,
                const uint8_t *vis, float *colors, void *cuda_stream)
{
    if (N < 0 || C < 1 || C > NASG_MAX_CAMERAS) return NASG_ERR_SHAPE;
    if (N == 0) return NASG_OK;
    if (!means || !coeffs || !campos || !colors) return NASG_ERR_NULL;
    nasg::ShParams p{N, C, means, coeffs, campos, vis, nullptr, colors, nullptr, nullptr, nullptr};
    cudaError_t e = use_pipe(C) ? nasg::launch_sh_fwd_pipe(p, (cudaStream_t)cuda_stream) : nasg::launch_sh_fwd(p, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return NASG_OK;
}

int sh_eval_bwd(int64_t N, int32_t C, const float *means, const float *coeffs, const float *campos,
                const uint8_t *vis, const float *g_colors, float *g_means, float *g_coeffs,
                float *g_campos, void *workspace, size_t workspace_bytes, void *cuda_stream)
{
    if (N < 0 || C < 1 || C > NASG_MAX_CAMERAS) return NASG_ERR_SHAPE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (N == 0) {
        if (g_campos) {
            cudaError_t e = cudaMemsetAsync(g_campos, 0, sizeof(float) * 3 * C, st);
            if (e != cudaSuccess) return cuda_fail(e);
        }
        return NASG_OK;
    }
    if (!means || !coeffs || !campos || !g_colors) return NASG_ERR_NULL;
    float *partial = nullptr;
    if (g_campos) {
        if (!workspace || workspace_bytes < cam_partial_bytes(N, C)) return NASG_ERR_WORKSPACE;
        partial = static_cast<float *>(workspace);
    }
    nasg::ShParams p{N, C, means, coeffs, campos, vis, g_colors, nullptr, g_means, g_coeffs, partial};
    cudaError_t e = (use_pipe(C) && !partial) ? nasg::launch_sh_bwd_pipe(p, st) : nasg::launch_sh_bwd(p, st);
    if (e != cudaSuccess) return cuda_fail(e);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    if (partial) {
        e = nasg::launch_campos_reduce(partial, nasg::grid_blocks(N), C, g_campos, st);
        if (e != cudaSuccess) return cuda_fail(e);
        g_launches.fetch_add(1, std::memory_order_relaxed);
    }
    return NASG_OK;
}

size_t nasg_workspace_bytes(int64_t N, int32_t K, int32_t C)
{
    (void)K;
    if (N <= 0 || C < 1) return 0;
    return cam_partial_bytes(N, C);
}

// ---- host-buffer end-to-end entry points ------------------------------------------------------
size_t nasg_host_scratch_bytes(int64_t N, int32_t K, int32_t C)
{
    if (N <= 0 || K < 1 || C < 1) return 0;
    const size_t n = (size_t)N, k = (size_t)K, c = (size_t)C;
    size_t in_b = align_up(n * 3 * 4) + 2 * align_up(k * n * 16) + align_up(k * 3 * n * 4) + align_up(3 * n * 4) +
                  align_up(c * 3 * 4) + align_up(c * n) + align_up(c * n * 3 * 4);            // + g_colors
    size_t out_b = align_up(c * n * 3 * 4) + align_up(n * 3 * 4) + 2 * align_up(k * n * 16) +
                   align_up(k * 3 * n * 4) + align_up(3 * n * 4) + align_up(c * 3 * 4) + align_up(cam_partial_bytes(N, C));
    return in_b + out_b;
}

int nasg_eval_fwd_bwd_host(const nasg_inputs *in, const float *g_colors, float *colors, const nasg_grads *out,
                           int norm_mode, void *dev_scratch, size_t dev_scratch_bytes, void *cuda_stream)
{
    int rc = check_inputs(in);
    if (rc != NASG_OK) return rc;
    if (!out) return NASG_ERR_NULL;
    if (in->N == 0) return NASG_OK;
    if (!g_colors || !colors || !dev_scratch) return NASG_ERR_NULL;
    if (dev_scratch_bytes < nasg_host_scratch_bytes(in->N, in->K, in->C) || !aligned16(dev_scratch))
        return NASG_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t n = (size_t)in->N, k = (size_t)in->K, c = (size_t)in->C;
    Carver cv{static_cast<char *>(dev_scratch), 0, dev_scratch_bytes};
    float *d_means = cv.take<float>(n * 3), *d_quat = cv.take<float>(k * n * 4), *d_shape = cv.take<float>(k * n * 4);
    float *d_amp = cv.take<float>(k * 3 * n), *d_dc = cv.take<float>(3 * n), *d_campos = cv.take<float>(c * 3);
    uint8_t *d_vis = cv.take<uint8_t>(c * n);
    float *d_gcol = cv.take<float>(c * n * 3), *d_col = cv.take<float>(c * n * 3);
    float *d_gm = cv.take<float>(n * 3), *d_gq = cv.take<float>(k * n * 4), *d_gs = cv.take<float>(k * n * 4);
    float *d_ga = cv.take<float>(k * 3 * n), *d_gdc = cv.take<float>(3 * n), *d_gcam = cv.take<float>(c * 3);
    const size_t ws_bytes = cam_partial_bytes(in->N, in->C);
    float *d_ws = cv.take<float>(ws_bytes / sizeof(float));
    if (cv.off > cv.cap) return NASG_ERR_WORKSPACE;

    const cudaMemcpyKind H2D = cudaMemcpyHostToDevice, D2H = cudaMemcpyDeviceToHost;
    NASG_TRY_CUDA(cudaMemcpyAsync(d_means, in->means, n * 12, H2D, st));
    NASG_TRY_CUDA(cudaMemcpyAsync(d_quat, in->quat, k * n * 16, H2D, st));
    NASG_TRY_CUDA(cudaMemcpyAsync(d_shape, in->shape, k * n * 16, H2D, st));
    NASG_TRY_CUDA(cudaMemcpyAsync(d_amp, in->amp, k * n * 12, H2D, st));
    NASG_TRY_CUDA(cudaMemcpyAsync(d_dc, in->dc, n * 12, H2D, st));
    NASG_TRY_CUDA(cudaMemcpyAsync(d_campos, in->campos, c * 12, H2D, st));
    if (in->vis) NASG_TRY_CUDA(cudaMemcpyAsync(d_vis, in->vis, c * n, H2D, st));
    NASG_TRY_CUDA(cudaMemcpyAsync(d_gcol, g_colors, c * n * 12, H2D, st));

    nasg_inputs din = *in;
    din.means = d_means; din.quat = d_quat; din.shape = d_shape; din.amp = d_amp; din.dc = d_dc;
    din.campos = d_campos; din.vis = in->vis ? d_vis : nullptr;
    rc = nasg_eval_fwd(&din, d_col, norm_mode, cuda_stream);
    if (rc != NASG_OK) return rc;
    nasg_grads dg{};
    dg.g_means = out->g_means ? d_gm : nullptr; dg.g_quat = out->g_quat ? d_gq : nullptr;
    dg.g_shape = out->g_shape ? d_gs : nullptr; dg.g_amp = out->g_amp ? d_ga : nullptr;
    dg.g_dc = out->g_dc ? d_gdc : nullptr; dg.g_campos = out->g_campos ? d_gcam : nullptr;
    dg.workspace = d_ws; dg.workspace_bytes = ws_bytes;
    rc = nasg_eval_bwd(&din, d_gcol, &dg, norm_mode, cuda_stream);
    if (rc != NASG_OK) return rc;

    NASG_TRY_CUDA(cudaMemcpyAsync(colors, d_col, c * n * 12, D2H, st));
    if (out->g_means) NASG_TRY_CUDA(cudaMemcpyAsync(out->g_means, d_gm, n * 12, D2H, st));
    if (out->g_quat) NASG_TRY_CUDA(cudaMemcpyAsync(out->g_quat, d_gq, k * n * 16, D2H, st));
    if (out->g_shape) NASG_TRY_CUDA(cudaMemcpyAsync(out->g_shape, d_gs, k * n * 16, D2H, st));
    if (out->g_amp) NASG_TRY_CUDA(cudaMemcpyAsync(out->g_amp, d_ga, k * n * 12, D2H, st));
    if (out->g_dc) NASG_TRY_CUDA(cudaMemcpyAsync(out->g_dc, d_gdc, n * 12, D2H, st));
    if (out->g_campos) NASG_TRY_CUDA(cudaMemcpyAsync(out->g_campos, d_gcam, c * 12, D2H, st));
    return NASG_OK;
}

size_t sh_host_scratch_bytes(int64_t N, int32_t C)
{
    if (N <= 0 || C < 1) return 0;
    const size_t n = (size_t)N, c = (size_t)C;
    return 2 * align_up(n * 12) + 2 * align_up(48 * n * 4) + 2 * align_up(c * 12) + align_up(c * n) +
           2 * align_up(c * n * 12) + align_up(cam_partial_bytes(N, C));
}

int sh_eval_fwd_bwd_host(int64_t N, int32_t C, const float *means, const float *coeffs, const float *campos,
                         const uint8_t *vis, const float *g_colors, float *colors, float *g_means,
                         float *g_coeffs, float *g_campos, void *dev_scratch, size_t dev_scratch_bytes,
                         void *cuda_stream)
{
    if (N < 0 || C < 1 || C > NASG_MAX_CAMERAS) return NASG_ERR_SHAPE;
    if (N == 0) return NASG_OK;
    if (!means || !coeffs || !campos || !g_colors || !colors || !dev_scratch) return NASG_ERR_NULL;
    if (dev_scratch_bytes < sh_host_scratch_bytes(N, C) || !aligned16(dev_scratch)) return NASG_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t n = (size_t)N, c = (size_t)C;
    Carver cv{static_cast<char *>(dev_scratch), 0, dev_scratch_bytes};
    float *d_means = cv.take<float>(n * 3), *d_co = cv.take<float>(48 * n), *d_campos = cv.take<float>(c * 3);
    uint8_t *d_vis = cv.take<uint8_t>(c * n);
    float *d_gcol = cv.take<float>(c * n * 3), *d_col = cv.take<float>(c * n * 3);
    float *d_gm = cv.take<float>(n * 3), *d_gco = cv.take<float>(48 * n), *d_gcam = cv.take<float>(c * 3);
    const size_t ws_bytes = cam_partial_bytes(N, C);
    float *d_ws = cv.take<float>(ws_bytes / sizeof(float));
    if (cv.off > cv.cap) return NASG_ERR_WORKSPACE;
    const cudaMemcpyKind H2D = cudaMemcpyHostToDevice, D2H = cudaMemcpyDeviceToHost;
    NASG_TRY_CUDA(cudaMemcpyAsync(d_means, means, n * 12, H2D, st));
    NASG_TRY_CUDA(cudaMemcpyAsync(d_co, coeffs, 48 * n * 4, H2D, st));
    NASG_TRY_CUDA(cudaMemcpyAsync(d_campos, campos, c * 12, H2D, st));
    if (vis) NASG_TRY_CUDA(cudaMemcpyAsync(d_vis, vis, c * n, H2D, st));
    NASG_TRY_CUDA(cudaMemcpyAsync(d_gcol, g_colors, c * n * 12, H2D, st));
    int rc = sh_eval_fwd(N, C, d_means, d_co, d_campos, vis ? d_vis : nullptr, d_col, cuda_stream);
    if (rc != NASG_OK) return rc;
    rc = sh_eval_bwd(N, C, d_means, d_co, d_campos, vis ? d_vis : nullptr, d_gcol, g_means ? d_gm : nullptr,
                     g_coeffs ? d_gco : nullptr, g_campos ? d_gcam : nullptr, d_ws, ws_bytes, cuda_stream);
    if (rc != NASG_OK) return rc;
    NASG_TRY_CUDA(cudaMemcpyAsync(colors, d_col, c * n * 12, D2H, st));
    if (g_means) NASG_TRY_CUDA(cudaMemcpyAsync(g_means, d_gm, n * 12, D2H, st));
    if (g_coeffs) NASG_TRY_CUDA(cudaMemcpyAsync(g_coeffs, d_gco, 48 * n * 4, D2H, st));
    if (g_campos) NASG_TRY_CUDA(cudaMemcpyAsync(g_campos, d_gcam, c * 12, D2H, st));
    return NASG_OK;
}

const char *nasg_strerror(int code)
{
    switch (code) {
    case NASG_OK: return "ok";
    case NASG_ERR_NULL: return "a required pointer is NULL";
    case NASG_ERR_SHAPE: return "bad shape: need N >= 0 and 1 <= C <= 64";
    case NASG_ERR_UNSUPPORTED_K: return "unsupported lobe count K (supported: 1,2,3,4,5,8)";
    case NASG_ERR_ALIGN: return "quat/shape (or their gradients) must be 16-byte aligned";
    case NASG_ERR_WORKSPACE: return "workspace/scratch missing, misaligned or too small";
    case NASG_ERR_CUDA: return cudaGetErrorString(t_last_cuda);
    case NASG_ERR_NORM_MODE: return "norm_mode must be 0 (approximate) or 1 (exact, eq.10)";
    default: return "unknown error code";
    }
}

const char *nasg_version(void) { return "0.1.0 sm_100a"; }

int64_t nasg_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

} // extern "C"
