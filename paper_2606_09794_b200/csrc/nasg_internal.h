// nasg_internal.h — kernel parameter blocks and launcher declarations shared by the .cu files of the
// library (not part of the public ABI; the oracle does not see this file).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace nasg {

struct FwdParams {
    int64_t N;
    int C;
    const float *means, *quat, *shape, *amp, *dc, *campos;
    const uint8_t *vis;
    float *colors;
};

struct BwdParams {
    int64_t N;
    int C;
    const float *means, *quat, *shape, *amp, *campos;
    const uint8_t *vis;
    const float *g_colors;
    float *g_means, *g_quat, *g_shape, *g_amp, *g_dc;
    float *cam_partial;          // [blocks, C, 3] per-block partial sums of g_campos, or nullptr
};

struct ShParams {
    int64_t N;
    int C;
    const float *means, *coeffs, *campos;
    const uint8_t *vis;
    const float *g_colors;       // backward only
    float *colors;               // forward only
    float *g_means, *g_coeffs;   // backward only
    float *cam_partial;
};

// tile-record layout (nasg_rec_kernels.cu; include/nasg.h: nasg_rec_*)
struct RecFwdParams {
    int64_t N;
    int C;
    int bulk_rows;               // vis rows can be moved with bulk copies (N % 16 == 0, 16-byte aligned); else per-lane loads
    const float *params, *campos;
    const uint8_t *vis;
    float *colors;
};
struct RecBwdParams {
    int64_t N;
    int C;
    int bulk_rows;               // g_colors (N % 4 == 0) and vis rows (N % 16 == 0) can be moved with bulk copies
    const float *params, *campos;
    const uint8_t *vis;
    const float *g_colors;
    float *g_params;
};

// Grid of a persistent kernel: min(blocks N needs, blocks resident on the device). The occupancy query and the opt-in to
// `smem` bytes of dynamic shared memory are made once per (kernel instantiation, device) and the resident count is kept
// in `cached` ([64], one slot per device ordinal, zero = not set up yet). Host threads may race on a first call: the
// slot is read and written atomically and every thread would store the same value. A failed opt-in is NOT cached: it is
// retried by the next launch, and the launch that follows here fails and reports it through cudaGetLastError().
template <typename Kernel>
static int resident_grid(Kernel kernel, int threads, size_t smem, int64_t N, int *cached)
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) dev = -1;
    const bool slot = dev >= 0 && dev < 64;
    int resident = slot ? __atomic_load_n(&cached[dev], __ATOMIC_ACQUIRE) : 0;
    if (resident == 0) {
        int sms = 148, per_sm = 1;
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev < 0 ? 0 : dev);
        const cudaError_t opt_in = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, smem) != cudaSuccess || per_sm < 1) per_sm = 1;
        resident = per_sm * sms;
        if (slot && opt_in == cudaSuccess) __atomic_store_n(&cached[dev], resident, __ATOMIC_RELEASE);
    }
    const int64_t need = (N + threads - 1) / threads;
    return (int)(need < resident ? need : resident);
}

int64_t grid_blocks(int64_t N);
int api_cuda_fail(cudaError_t e);     // remembers e for nasg_strerror(), returns NASG_ERR_CUDA (nasg_api.cu)
void api_count_launches(int n);       // adds to nasg_launch_count() (for entry points outside nasg_api.cu)
cudaError_t launch_nasg_fwd(const FwdParams &p, int K, int mode, cudaStream_t st);
cudaError_t launch_nasg_bwd(const BwdParams &p, int K, int mode, cudaStream_t st);
// fast path (nasg_pipe_kernels.cu): C <= 4, persistent threads, cp.async lobe ring
cudaError_t launch_nasg_fwd_pipe(const FwdParams &p, int K, int mode, cudaStream_t st);
cudaError_t launch_nasg_bwd_pipe(const BwdParams &p, int K, int mode, cudaStream_t st, int *grid_out);   // grid_out: blocks launched (= rows of cam_partial)
// row arrays, tile kernels (nasg_tile_kernels.cu): even K, C <= 4, aligned rows, no g_campos: lobe pairs on packed f32x2, TMA bulk-copy tiles
bool tile_path_ok(int64_t N, int K, int C, const void *means, const void *amp, const void *planar, const void *rows, const void *vis);
cudaError_t launch_nasg_fwd_tile(const FwdParams &p, int K, int mode, cudaStream_t st);
cudaError_t launch_nasg_bwd_tile(const BwdParams &p, int K, int mode, cudaStream_t st);
// headline path (nasg_rec_kernels.cu): tile-record parameter layout, even K, C <= 4
int64_t rec_total_floats(int64_t N, int K, int pk = 0);     // pk: 0 = quaternion records (11 floats per lobe), 1 = paper records (9), 2 = isotropic (7), 3 = bf16 quat/amp
cudaError_t launch_nasg_rec_fwd(const RecFwdParams &p, int K, int mode, int pk, cudaStream_t st);
cudaError_t launch_nasg_rec_bwd(const RecBwdParams &p, int K, int mode, int pk, cudaStream_t st);
cudaError_t launch_rec_pack(int64_t N, int K, const float *means, const float *quat, const float *shape, const float *amp, const float *dc,
                            float *rec_out, cudaStream_t st);
cudaError_t launch_rec16_pack(int64_t N, int K, const float *means, const float *quat, const float *shape, const float *amp, const float *dc,
                              float *rec_out, cudaStream_t st);
cudaError_t launch_rec_unpack(int64_t N, int K, const float *rec_in, float *means, float *quat, float *shape, float *amp, float *dc,
                              cudaStream_t st);
cudaError_t launch_campos_reduce(const float *partial, int64_t nblocks, int C, float *out, cudaStream_t st);
cudaError_t launch_sh_fwd(const ShParams &p, cudaStream_t st);
cudaError_t launch_sh_bwd(const ShParams &p, cudaStream_t st);
// fast path (sh_pipe_kernels.cu): C <= 4, same persistent cp.async skeleton
cudaError_t launch_sh_fwd_pipe(const ShParams &p, cudaStream_t st);
cudaError_t launch_sh_bwd_pipe(const ShParams &p, cudaStream_t st, int *grid_out);

} // namespace nasg
