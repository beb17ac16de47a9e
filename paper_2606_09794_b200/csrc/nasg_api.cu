// nasg_api.cu — the extern "C" boundary declared in include/nasg.h: argument validation and dispatch
// to the kernel launchers (the host-buffer end-to-end entry points live in nasg_host_pipeline.cu).
// No arithmetic of the method lives here.
#include "nasg.h"
#include "nasg_internal.h"

#include <atomic>

namespace {

std::atomic<int64_t> g_launches{0};
thread_local cudaError_t t_last_cuda = cudaSuccess;

inline bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
inline bool supported_K(int K) { return K == 1 || K == 2 || K == 3 || K == 4 || K == 5 || K == 8; }

// Kernel family: 0 = automatic (tile kernels when their conditions hold, else the cp.async ring kernels for C <= 4,
// else the generic kernels); 1 = generic only; 2 = no tile kernels. Set by nasg_debug_set_path() (a test hook, so
// that every family can be compared with the oracle on the same inputs); never read from the environment.
std::atomic<int> g_path{0};
bool use_pipe(int C) { return C <= 4 && g_path.load(std::memory_order_relaxed) != 1; }
bool use_tile() { return g_path.load(std::memory_order_relaxed) == 0; }

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

} // namespace

namespace nasg {
int api_cuda_fail(cudaError_t e) { return cuda_fail(e); }
void api_count_launches(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }
} // namespace nasg

extern "C" {

int nasg_eval_fwd(const nasg_inputs *in, float *colors, int norm_mode, void *cuda_stream)
{
    int rc = check_inputs(in);
    if (rc != NASG_OK) return rc;
    if (norm_mode != NASG_NORM_APPROX && norm_mode != NASG_NORM_EXACT && norm_mode != NASG_NORM_NASG) return NASG_ERR_NORM_MODE;
    if (in->N == 0) return NASG_OK;
    if (!colors) return NASG_ERR_NULL;
    if (!aligned16(in->quat) || !aligned16(in->shape)) return NASG_ERR_ALIGN;
    nasg::FwdParams p{in->N, in->C, in->means, in->quat, in->shape, in->amp, in->dc, in->campos, in->vis, colors};
    cudaError_t e;
    if (use_tile() && nasg::tile_path_ok(in->N, in->K, in->C, in->means, in->amp, in->dc, nullptr, in->vis))
        e = nasg::launch_nasg_fwd_tile(p, in->K, norm_mode, (cudaStream_t)cuda_stream);
    else
        e = use_pipe(in->C) ? nasg::launch_nasg_fwd_pipe(p, in->K, norm_mode, (cudaStream_t)cuda_stream)
                            : nasg::launch_nasg_fwd(p, in->K, norm_mode, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return NASG_OK;
}

int nasg_eval_bwd(const nasg_inputs *in, const float *g_colors, const nasg_grads *out, int norm_mode,
                  void *cuda_stream)
{
    int rc = check_inputs(in);
    if (rc != NASG_OK) return rc;
    if (norm_mode != NASG_NORM_APPROX && norm_mode != NASG_NORM_EXACT && norm_mode != NASG_NORM_NASG) return NASG_ERR_NORM_MODE;
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
    int pipe_blocks = 0;
    const bool pipe = use_pipe(in->C);
    cudaError_t e;
    if (!partial && use_tile() && nasg::tile_path_ok(in->N, in->K, in->C, in->means, in->amp, nullptr, g_colors, in->vis))
        e = nasg::launch_nasg_bwd_tile(p, in->K, norm_mode, st);
    else
        e = pipe ? nasg::launch_nasg_bwd_pipe(p, in->K, norm_mode, st, &pipe_blocks) : nasg::launch_nasg_bwd(p, in->K, norm_mode, st);
    if (e != cudaSuccess) return cuda_fail(e);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    if (partial) {      // second stage of g_campos: fixed-order sum of the per-block partials
        e = nasg::launch_campos_reduce(partial, pipe ? pipe_blocks : nasg::grid_blocks(in->N), in->C, out->g_campos, st);
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
    int pipe_blocks = 0;
    const bool pipe = use_pipe(C);
    cudaError_t e = pipe ? nasg::launch_sh_bwd_pipe(p, st, &pipe_blocks) : nasg::launch_sh_bwd(p, st);
    if (e != cudaSuccess) return cuda_fail(e);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    if (partial) {
        e = nasg::launch_campos_reduce(partial, pipe ? pipe_blocks : nasg::grid_blocks(N), C, g_campos, st);
        if (e != cudaSuccess) return cuda_fail(e);
        g_launches.fetch_add(1, std::memory_order_relaxed);
    }
    return NASG_OK;
}

// ---- tile-record layout (include/nasg.h: nasg_rec_*) ---------------------------------------------
static bool rec_K_ok(int K) { return K == 2 || K == 4 || K == 8; }
static int norm_ok(int m) { return m == NASG_NORM_APPROX || m == NASG_NORM_EXACT || m == NASG_NORM_NASG; }

size_t nasg_rec_floats(int64_t N, int32_t K)
{
    if (N <= 0 || !rec_K_ok(K)) return 0;
    return (size_t)nasg::rec_total_floats(N, K);
}

int nasg_rec_pack(const nasg_inputs *in, float *params, void *cuda_stream)
{
    if (!in) return NASG_ERR_NULL;
    if (in->N < 0 || in->N > NASG_REC_MAX_N) return NASG_ERR_SHAPE;
    if (!rec_K_ok(in->K)) return NASG_ERR_UNSUPPORTED_K;
    if (in->N == 0) return NASG_OK;
    if (!in->means || !in->quat || !in->shape || !in->amp || !in->dc || !params) return NASG_ERR_NULL;
    if (!aligned16(in->quat) || !aligned16(in->shape) || !aligned16(params)) return NASG_ERR_ALIGN;
    cudaError_t e = nasg::launch_rec_pack(in->N, in->K, in->means, in->quat, in->shape, in->amp, in->dc, params, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return NASG_OK;
}

int nasg_rec_unpack(int64_t N, int32_t K, const float *rec, float *means, float *quat, float *shape, float *amp, float *dc,
                    void *cuda_stream)
{
    if (N < 0 || N > NASG_REC_MAX_N) return NASG_ERR_SHAPE;
    if (!rec_K_ok(K)) return NASG_ERR_UNSUPPORTED_K;
    if (N == 0) return NASG_OK;
    if (!rec) return NASG_ERR_NULL;
    if (!aligned16(quat) || !aligned16(shape) || !aligned16(rec)) return NASG_ERR_ALIGN;
    cudaError_t e = nasg::launch_rec_unpack(N, K, rec, means, quat, shape, amp, dc, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return NASG_OK;
}

static int check_rec_inputs(const nasg_rec_inputs *in, int norm_mode)
{
    if (!in) return NASG_ERR_NULL;
    if (in->N < 0 || in->N > NASG_REC_MAX_N || in->C < 1 || in->C > NASG_REC_MAX_CAMERAS) return NASG_ERR_SHAPE;
    if (!rec_K_ok(in->K)) return NASG_ERR_UNSUPPORTED_K;
    if (!norm_ok(norm_mode & ~NASG_HINT_COHERENT_VIS)) return NASG_ERR_NORM_MODE;
    if (in->N == 0) return NASG_OK;
    if (!in->params || !in->campos) return NASG_ERR_NULL;
    if (!aligned16(in->params)) return NASG_ERR_ALIGN;
    return NASG_OK;
}

static int rec_eval_fwd(const nasg_rec_inputs *in, float *colors, int norm_mode, int pk, void *cuda_stream)
{
    int rc = check_rec_inputs(in, norm_mode);
    if (rc != NASG_OK) return rc;
    if (in->N == 0) return NASG_OK;
    if (!colors) return NASG_ERR_NULL;
    const int bulk_rows = !in->vis || ((in->N & 15) == 0 && aligned16(in->vis));
    nasg::RecFwdParams p{in->N, in->C, bulk_rows, in->params, in->campos, in->vis, colors};
    cudaError_t e = nasg::launch_nasg_rec_fwd(p, in->K, norm_mode, pk, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return NASG_OK;
}

static int rec_eval_bwd(const nasg_rec_inputs *in, const float *g_colors, float *g_params, int norm_mode, int pk, void *cuda_stream)
{
    int rc = check_rec_inputs(in, norm_mode);
    if (rc != NASG_OK) return rc;
    if (in->N == 0) return NASG_OK;
    if (!g_colors || !g_params) return NASG_ERR_NULL;
    if (!aligned16(g_params)) return NASG_ERR_ALIGN;
    const int bulk_rows = (in->N & 3) == 0 && aligned16(g_colors) && (!in->vis || ((in->N & 15) == 0 && aligned16(in->vis)));
    nasg::RecBwdParams p{in->N, in->C, bulk_rows, in->params, in->campos, in->vis, g_colors, g_params};
    cudaError_t e = nasg::launch_nasg_rec_bwd(p, in->K, norm_mode, pk, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return NASG_OK;
}

int nasg_rec_eval_fwd(const nasg_rec_inputs *in, float *colors, int norm_mode, void *cuda_stream)
{
    return rec_eval_fwd(in, colors, norm_mode, 0, cuda_stream);
}
int nasg_rec_eval_bwd(const nasg_rec_inputs *in, const float *g_colors, float *g_params, int norm_mode, void *cuda_stream)
{
    return rec_eval_bwd(in, g_colors, g_params, norm_mode, 0, cuda_stream);
}

// ---- paper-native record (Table 8 activations, Supplementary C frame, no phase): 9 floats per lobe
size_t nasg_paper_floats(int64_t N, int32_t K)
{
    if (N <= 0 || !rec_K_ok(K)) return 0;
    return (size_t)nasg::rec_total_floats(N, K, 1);
}
int nasg_paper_eval_fwd(const nasg_rec_inputs *in, float *colors, int norm_mode, void *cuda_stream)
{
    return rec_eval_fwd(in, colors, norm_mode, 1, cuda_stream);
}
int nasg_paper_eval_bwd(const nasg_rec_inputs *in, const float *g_colors, float *g_params, int norm_mode, void *cuda_stream)
{
    return rec_eval_bwd(in, g_colors, g_params, norm_mode, 1, cuda_stream);
}

// ---- bf16 parameter storage: quaternion and amplitude as bfloat16 (fp32 arithmetic, fp32 gradient records)
size_t nasg_rec16_floats(int64_t N, int32_t K)
{
    if (N <= 0 || !rec_K_ok(K)) return 0;
    return (size_t)nasg::rec_total_floats(N, K, 3);
}
int nasg_rec16_pack(const nasg_inputs *in, float *params, void *cuda_stream)
{
    if (!in) return NASG_ERR_NULL;
    if (in->N < 0 || in->N > NASG_REC_MAX_N) return NASG_ERR_SHAPE;
    if (!rec_K_ok(in->K)) return NASG_ERR_UNSUPPORTED_K;
    if (in->N == 0) return NASG_OK;
    if (!in->means || !in->quat || !in->shape || !in->amp || !in->dc || !params) return NASG_ERR_NULL;
    if (!aligned16(in->quat) || !aligned16(in->shape) || !aligned16(params)) return NASG_ERR_ALIGN;
    cudaError_t e = nasg::launch_rec16_pack(in->N, in->K, in->means, in->quat, in->shape, in->amp, in->dc, params, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return NASG_OK;
}
int nasg_rec16_eval_fwd(const nasg_rec_inputs *in, float *colors, int norm_mode, void *cuda_stream)
{
    return rec_eval_fwd(in, colors, norm_mode, 3, cuda_stream);
}
int nasg_rec16_eval_bwd(const nasg_rec_inputs *in, const float *g_colors, float *g_params, int norm_mode, void *cuda_stream)
{
    return rec_eval_bwd(in, g_colors, g_params, norm_mode, 3, cuda_stream);
}

// ---- isotropic Table-6 functions (Spherical Gaussian / Beta / Cauchy): 7 floats per lobe
size_t nasg_iso_floats(int64_t N, int32_t K)
{
    if (N <= 0 || !rec_K_ok(K)) return 0;
    return (size_t)nasg::rec_total_floats(N, K, 2);
}
int nasg_iso_eval_fwd(const nasg_rec_inputs *in, float *colors, int kind, void *cuda_stream)
{
    return rec_eval_fwd(in, colors, kind, 2, cuda_stream);
}
int nasg_iso_eval_bwd(const nasg_rec_inputs *in, const float *g_colors, float *g_params, int kind, void *cuda_stream)
{
    return rec_eval_bwd(in, g_colors, g_params, kind, 2, cuda_stream);
}

// ---- Anisotropic Spherical Gaussian of Table 6: 9 floats per lobe
size_t nasg_asg_floats(int64_t N, int32_t K)
{
    if (N <= 0 || !rec_K_ok(K)) return 0;
    return (size_t)nasg::rec_total_floats(N, K, 4);
}
int nasg_asg_eval_fwd(const nasg_rec_inputs *in, float *colors, void *cuda_stream)
{
    return rec_eval_fwd(in, colors, 0, 4, cuda_stream);
}
int nasg_asg_eval_bwd(const nasg_rec_inputs *in, const float *g_colors, float *g_params, void *cuda_stream)
{
    return rec_eval_bwd(in, g_colors, g_params, 0, 4, cuda_stream);
}

size_t nasg_workspace_bytes(int64_t N, int32_t K, int32_t C)
{
    (void)K;
    if (N <= 0 || C < 1) return 0;
    return cam_partial_bytes(N, C);
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
    case NASG_ERR_NORM_MODE: return "norm_mode must be 0 (approximate), 1 (exact, eq.10) or 2 (pure NASG, no carrier); nasg_iso_*: kind must be 0, 1 or 2";
    case NASG_ERR_NOALLOC_SIZE: return "nasg_eval_bwd_noalloc: N and C need more scratch than the built-in 1 MiB array (nasg_workspace_bytes(N,K,C) > nasg_noalloc_workspace_bytes()); call nasg_eval_bwd with a workspace of your own";
    default: return "unknown error code";
    }
}

const char *nasg_version(void) { return "0.1.0 sm_100a"; }

int64_t nasg_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

void nasg_debug_set_path(int path) { g_path.store(path < 0 || path > 2 ? 0 : path, std::memory_order_relaxed); }

} // extern "C"
