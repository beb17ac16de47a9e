// nasg_host_pipeline.cu — the host-buffer end-to-end entry points of include/nasg.h
// (nasg_eval_fwd_bwd_host, sh_eval_fwd_bwd_host). No arithmetic of the method lives here.
//
// The Gaussians are independent, so the call is cut into chunks of contiguous n-ranges and run as a
// three-stage pipeline over two device buffers: host->device copy of chunk i+1, the two kernels on
// chunk i and device->host copy of chunk i-1 proceed at the same time on three internal streams.
// PCIe is full duplex: with the copies in both directions overlapped the call approaches
// max(H2D, D2H) bytes / link bandwidth instead of their sum (bench.py's `e2e`). Every array keeps the
// layout of the device entry points; a chunk of a planar [rows, N] array is a 2-D copy
// (cudaMemcpy2DAsync: `rows` rows of the chunk's width, source pitch N, destination pitch = chunk).
//
// Stream semantics are those of the device entry points: everything is ordered after the work already
// on `cuda_stream`, the call returns without synchronising, and `cuda_stream` is made to wait for the
// pipeline's last copy. The three internal streams and their events are created once per device on
// first use (the only state the library keeps); calls on one device are serialised by a mutex while
// they enqueue. g_campos sums over all Gaussians, so a call that asks for it runs as a single chunk.
#include "nasg.h"
#include "nasg_internal.h"

#include <mutex>
#include <vector>

namespace {

inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }
inline bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
size_t cam_partial_bytes(int64_t N, int C) { return (size_t)nasg::grid_blocks(N) * (size_t)C * 3 * sizeof(float); }

#define NASG_TRY_CUDA(expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) return nasg::api_cuda_fail(e_); } while (0)
#define NASG_TRY(expr) do { int rc_ = (expr); if (rc_ != NASG_OK) return rc_; } while (0)

#ifndef NASG_HOST_CHUNK_MIN
#define NASG_HOST_CHUNK_MIN 131072
#endif
#ifndef NASG_HOST_MAX_CHUNKS
#define NASG_HOST_MAX_CHUNKS 16
#endif
constexpr int64_t CHUNK_MIN = NASG_HOST_CHUNK_MIN;    // Gaussians per chunk at least (copies of a few MB each)
constexpr int MAX_CHUNKS = NASG_HOST_MAX_CHUNKS;
constexpr size_t SCRATCH_SLOP = 64 * 1024;   // alignment padding of the per-chunk carve-up

// chunk size: a multiple of 256 (keeps rows 16-byte aligned and the visibility rows 4-byte aligned)
int64_t chunk_size(int64_t N, bool single)
{
    if (single || N < 2 * CHUNK_MIN) return N;
    int64_t chunks = N / CHUNK_MIN;
    if (chunks > MAX_CHUNKS) chunks = MAX_CHUNKS;
    const int64_t per = (N + chunks - 1) / chunks;
    return (per + 1023) / 1024 * 1024;
}
// Piece boundaries of the pipeline: full chunks in the middle, and a ramp (chunk/4, chunk/4, chunk/2) at either end so that
// the un-overlapped fill (first host->device copy) and drain (last device->host copy) are a quarter chunk each; every piece
// is a multiple of 256 Gaussians (8 records; rows stay 16-byte aligned) except the last.
std::vector<int64_t> piece_bounds(int64_t N, int64_t chunk)
{
    std::vector<int64_t> b{0};
    if (N >= 4 * chunk && chunk % 1024 == 0) {
        const int64_t middle = N - 2 * chunk, full = middle / chunk, r = middle - full * chunk, r256 = r / 256 * 256;
        for (int64_t u : {chunk / 4, chunk / 4, chunk / 2}) b.push_back(b.back() + u);
        for (int64_t i = 0; i < full; ++i) b.push_back(b.back() + chunk);
        if (r256 > 0) b.push_back(b.back() + r256);
        b.push_back(b.back() + chunk / 2);
        b.push_back(b.back() + chunk / 4);
        b.push_back(N);                                       // chunk/4 + (r - r256) Gaussians
    } else {
        while (N - b.back() > chunk) b.push_back(b.back() + chunk);
        b.push_back(N);
    }
    return b;
}

// carves aligned sub-buffers out of the caller's device scratch
struct Carver {
    char *base; size_t off, cap;
    template <typename T> T *take(size_t count)
    {
        const size_t bytes = align_up(count * sizeof(T));
        if (off + bytes > cap) { off = cap + 1; return nullptr; }
        T *p = reinterpret_cast<T *>(base + off);
        off += bytes;
        return p;
    }
};

// internal streams + events of one device
struct HostPipe {
    bool ready = false;
    cudaStream_t in = nullptr, comp = nullptr, out = nullptr;
    cudaEvent_t start = nullptr, in_done[2] = {nullptr, nullptr}, comp_done[2] = {nullptr, nullptr},
                out_done[2] = {nullptr, nullptr};
    std::mutex mu;
    cudaError_t init()
    {
        if (ready) return cudaSuccess;
        cudaError_t e;
        if ((e = cudaStreamCreateWithFlags(&in, cudaStreamNonBlocking)) != cudaSuccess) return e;
        if ((e = cudaStreamCreateWithFlags(&comp, cudaStreamNonBlocking)) != cudaSuccess) return e;
        if ((e = cudaStreamCreateWithFlags(&out, cudaStreamNonBlocking)) != cudaSuccess) return e;
        cudaEvent_t *evs[] = {&start, &in_done[0], &in_done[1], &comp_done[0], &comp_done[1], &out_done[0], &out_done[1]};
        for (cudaEvent_t *ev : evs)
            if ((e = cudaEventCreateWithFlags(ev, cudaEventDisableTiming)) != cudaSuccess) return e;
        ready = true;
        return cudaSuccess;
    }
};
HostPipe g_pipes[64];

// 2-D chunk copy of a planar [rows, N] array of `elem`-byte items: columns [n0, n0+nc)
cudaError_t copy_rows(void *dst, size_t dst_cols, const void *src, size_t src_cols, size_t col0_dst, size_t col0_src,
                      size_t nc, size_t rows, size_t elem, cudaMemcpyKind kind, cudaStream_t st)
{
    return cudaMemcpy2DAsync(static_cast<char *>(dst) + col0_dst * elem, dst_cols * elem,
                             static_cast<const char *>(src) + col0_src * elem, src_cols * elem, nc * elem, rows, kind, st);
}

// Runs `chunks` chunks through the three-stage pipeline. copy_in/compute/copy_out enqueue the work of
// chunk i (Gaussians [n0, n0+nc)) that uses device buffer b on the given stream.
template <typename CopyIn, typename Compute, typename CopyOut>
int enqueue_chunks(HostPipe &hp, int64_t N, int64_t chunk, cudaStream_t user, CopyIn copy_in, Compute compute, CopyOut copy_out)
{
    const std::vector<int64_t> bounds = piece_bounds(N, chunk);
    const int64_t chunks = (int64_t)bounds.size() - 1;
    for (int64_t i = 0; i < chunks; ++i) {
        const int b = (int)(i & 1);
        const int64_t n0 = bounds[i], nc = bounds[i + 1] - bounds[i];
        if (i >= 2) NASG_TRY_CUDA(cudaStreamWaitEvent(hp.in, hp.comp_done[b], 0));      // inputs of chunk i-2 consumed
        NASG_TRY(copy_in(b, n0, nc, hp.in));
        NASG_TRY_CUDA(cudaEventRecord(hp.in_done[b], hp.in));
        NASG_TRY_CUDA(cudaStreamWaitEvent(hp.comp, hp.in_done[b], 0));
        if (i >= 2) NASG_TRY_CUDA(cudaStreamWaitEvent(hp.comp, hp.out_done[b], 0));     // outputs of chunk i-2 drained
        NASG_TRY(compute(b, nc, hp.comp));
        NASG_TRY_CUDA(cudaEventRecord(hp.comp_done[b], hp.comp));
        NASG_TRY_CUDA(cudaStreamWaitEvent(hp.out, hp.comp_done[b], 0));
        NASG_TRY(copy_out(b, n0, nc, hp.out));
        NASG_TRY_CUDA(cudaEventRecord(hp.out_done[b], hp.out));
    }
    // the caller's stream continues after the last copy-out (which is after everything else)
    NASG_TRY_CUDA(cudaStreamWaitEvent(user, hp.out_done[(chunks - 1) & 1], 0));
    if (chunks >= 2) NASG_TRY_CUDA(cudaStreamWaitEvent(user, hp.out_done[(chunks - 2) & 1], 0));
    return NASG_OK;
}
template <typename CopyIn, typename Compute, typename CopyOut>
int run_pipeline(int64_t N, int64_t chunk, cudaStream_t user, CopyIn copy_in, Compute compute, CopyOut copy_out)
{
    int dev = 0;
    NASG_TRY_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return NASG_ERR_SHAPE;
    HostPipe &hp = g_pipes[dev];
    std::lock_guard<std::mutex> lock(hp.mu);
    NASG_TRY_CUDA(hp.init());
    NASG_TRY_CUDA(cudaEventRecord(hp.start, user));
    NASG_TRY_CUDA(cudaStreamWaitEvent(hp.in, hp.start, 0));
    NASG_TRY_CUDA(cudaStreamWaitEvent(hp.comp, hp.start, 0));
    NASG_TRY_CUDA(cudaStreamWaitEvent(hp.out, hp.start, 0));
    const int rc = enqueue_chunks(hp, N, chunk, user, copy_in, compute, copy_out);
    if (rc != NASG_OK) {
        // an enqueue failed half-way: whatever is already queued on the internal streams may still touch the caller's
        // buffers, so the caller's stream is joined to all three before the error is returned (best effort)
        cudaStream_t ss[3] = {hp.in, hp.comp, hp.out};
        cudaEvent_t es[3] = {hp.in_done[0], hp.comp_done[0], hp.out_done[0]};
        for (int i = 0; i < 3; ++i)
            if (cudaEventRecord(es[i], ss[i]) == cudaSuccess) cudaStreamWaitEvent(user, es[i], 0);
    }
    return rc;
}

} // namespace

// ---- NASGabor ---------------------------------------------------------------------------------
namespace {

struct NasgDev {        // device arrays of one buffer, sized for `cap` Gaussians
    float *means, *quat, *shape, *amp, *dc, *gcol, *col, *gm, *gq, *gs, *ga, *gdc;
    uint8_t *vis;
};
size_t nasg_footprint(size_t n, size_t k, size_t c)
{
    return 2 * align_up(n * 12) /* means, g_means */ + 4 * align_up(k * n * 16) /* quat, shape + grads */ +
           2 * align_up(k * n * 12) /* amp + grad */ + 2 * align_up(n * 12) /* dc + grad */ + align_up(c * n) /* vis */ +
           2 * align_up(c * n * 12) /* g_colors, colors */;
}
bool carve_nasg(Carver &cv, NasgDev &d, size_t n, size_t k, size_t c)
{
    d.means = cv.take<float>(n * 3); d.quat = cv.take<float>(k * n * 4); d.shape = cv.take<float>(k * n * 4);
    d.amp = cv.take<float>(k * 3 * n); d.dc = cv.take<float>(3 * n); d.vis = cv.take<uint8_t>(c * n);
    d.gcol = cv.take<float>(c * n * 3); d.col = cv.take<float>(c * n * 3);
    d.gm = cv.take<float>(n * 3); d.gq = cv.take<float>(k * n * 4); d.gs = cv.take<float>(k * n * 4);
    d.ga = cv.take<float>(k * 3 * n); d.gdc = cv.take<float>(3 * n);
    return cv.off <= cv.cap;
}

} // namespace

extern "C" {

size_t nasg_host_scratch_bytes(int64_t N, int32_t K, int32_t C)
{
    if (N <= 0 || K < 1 || C < 1) return 0;
    const size_t k = (size_t)K, c = (size_t)C;
    const size_t single = nasg_footprint((size_t)N, k, c);
    const size_t chunked = 2 * nasg_footprint((size_t)chunk_size(N, false), k, c);
    return (single > chunked ? single : chunked) + 2 * align_up(c * 12) + align_up(cam_partial_bytes(N, C)) + SCRATCH_SLOP;
}

int nasg_eval_fwd_bwd_host(const nasg_inputs *in, const float *g_colors, float *colors, const nasg_grads *out,
                           int norm_mode, void *dev_scratch, size_t dev_scratch_bytes, void *cuda_stream)
{
    if (!in || !out) return NASG_ERR_NULL;
    if (in->N < 0 || in->C < 1 || in->C > NASG_MAX_CAMERAS) return NASG_ERR_SHAPE;
    if (!(in->K == 1 || in->K == 2 || in->K == 3 || in->K == 4 || in->K == 5 || in->K == 8)) return NASG_ERR_UNSUPPORTED_K;
    if (norm_mode != NASG_NORM_APPROX && norm_mode != NASG_NORM_EXACT && norm_mode != NASG_NORM_NASG) return NASG_ERR_NORM_MODE;
    if (in->N == 0) return NASG_OK;
    if (!in->means || !in->quat || !in->shape || !in->amp || !in->dc || !in->campos || !g_colors || !colors || !dev_scratch)
        return NASG_ERR_NULL;
    if (dev_scratch_bytes < nasg_host_scratch_bytes(in->N, in->K, in->C) || !aligned16(dev_scratch)) return NASG_ERR_WORKSPACE;
    const int64_t N = in->N;
    const size_t k = (size_t)in->K, c = (size_t)in->C, Nn = (size_t)N;
    const int64_t chunk = chunk_size(N, out->g_campos != nullptr);
    const bool two = chunk < N;

    Carver cv{static_cast<char *>(dev_scratch), 0, dev_scratch_bytes};
    float *d_campos = cv.take<float>(c * 3), *d_gcam = cv.take<float>(c * 3);
    const size_t ws_bytes = cam_partial_bytes(chunk, in->C);
    float *d_ws = cv.take<float>(ws_bytes / sizeof(float) + 1);
    NasgDev dev[2];
    if (!carve_nasg(cv, dev[0], (size_t)chunk, k, c)) return NASG_ERR_WORKSPACE;
    if (two && !carve_nasg(cv, dev[1], (size_t)chunk, k, c)) return NASG_ERR_WORKSPACE;
    if (!d_campos || !d_gcam || !d_ws) return NASG_ERR_WORKSPACE;

    const cudaMemcpyKind H2D = cudaMemcpyHostToDevice, D2H = cudaMemcpyDeviceToHost;
    cudaStream_t user = (cudaStream_t)cuda_stream;
    NASG_TRY_CUDA(cudaMemcpyAsync(d_campos, in->campos, c * 12, H2D, user));     // replicated; before the pipeline's start event
    const nasg_inputs host = *in;
    const nasg_grads want = *out;

    auto copy_in = [&](int b, int64_t n0, int64_t nc, cudaStream_t st) -> int {
        const NasgDev &d = dev[b];
        const size_t o = (size_t)n0, w = (size_t)nc;
        NASG_TRY_CUDA(copy_rows(d.means, w, host.means, Nn, 0, o, w, 1, 12, H2D, st));
        NASG_TRY_CUDA(copy_rows(d.quat, w, host.quat, Nn, 0, o, w, k, 16, H2D, st));
        NASG_TRY_CUDA(copy_rows(d.shape, w, host.shape, Nn, 0, o, w, k, 16, H2D, st));
        NASG_TRY_CUDA(copy_rows(d.amp, w, host.amp, Nn, 0, o, w, 3 * k, 4, H2D, st));
        NASG_TRY_CUDA(copy_rows(d.dc, w, host.dc, Nn, 0, o, w, 3, 4, H2D, st));
        if (host.vis) NASG_TRY_CUDA(copy_rows(d.vis, w, host.vis, Nn, 0, o, w, c, 1, H2D, st));
        NASG_TRY_CUDA(copy_rows(d.gcol, w, g_colors, Nn, 0, o, w, c, 12, H2D, st));
        return NASG_OK;
    };
    auto compute = [&](int b, int64_t nc, cudaStream_t st) -> int {
        const NasgDev &d = dev[b];
        nasg_inputs din = host;
        din.N = nc; din.means = d.means; din.quat = d.quat; din.shape = d.shape; din.amp = d.amp; din.dc = d.dc;
        din.campos = d_campos; din.vis = host.vis ? d.vis : nullptr;
        NASG_TRY(nasg_eval_fwd(&din, d.col, norm_mode, st));
        nasg_grads dg{};
        dg.g_means = want.g_means ? d.gm : nullptr; dg.g_quat = want.g_quat ? d.gq : nullptr;
        dg.g_shape = want.g_shape ? d.gs : nullptr; dg.g_amp = want.g_amp ? d.ga : nullptr;
        dg.g_dc = want.g_dc ? d.gdc : nullptr; dg.g_campos = want.g_campos ? d_gcam : nullptr;
        dg.workspace = d_ws; dg.workspace_bytes = ws_bytes + sizeof(float);
        return nasg_eval_bwd(&din, d.gcol, &dg, norm_mode, st);
    };
    auto copy_out = [&](int b, int64_t n0, int64_t nc, cudaStream_t st) -> int {
        const NasgDev &d = dev[b];
        const size_t o = (size_t)n0, w = (size_t)nc;
        NASG_TRY_CUDA(copy_rows(colors, Nn, d.col, w, o, 0, w, c, 12, D2H, st));
        if (want.g_means) NASG_TRY_CUDA(copy_rows(want.g_means, Nn, d.gm, w, o, 0, w, 1, 12, D2H, st));
        if (want.g_quat) NASG_TRY_CUDA(copy_rows(want.g_quat, Nn, d.gq, w, o, 0, w, k, 16, D2H, st));
        if (want.g_shape) NASG_TRY_CUDA(copy_rows(want.g_shape, Nn, d.gs, w, o, 0, w, k, 16, D2H, st));
        if (want.g_amp) NASG_TRY_CUDA(copy_rows(want.g_amp, Nn, d.ga, w, o, 0, w, 3 * k, 4, D2H, st));
        if (want.g_dc) NASG_TRY_CUDA(copy_rows(want.g_dc, Nn, d.gdc, w, o, 0, w, 3, 4, D2H, st));
        if (want.g_campos) NASG_TRY_CUDA(cudaMemcpyAsync(want.g_campos, d_gcam, c * 12, D2H, st));   // single chunk only
        return NASG_OK;
    };
    return run_pipeline(N, chunk, user, copy_in, compute, copy_out);
}

} // extern "C"

// ---- SH degree 3 --------------------------------------------------------------------------------
namespace {

struct ShDev { float *means, *co, *gcol, *col, *gm, *gco; uint8_t *vis; };
size_t sh_footprint(size_t n, size_t c)
{
    return 2 * align_up(n * 12) + 2 * align_up(48 * n * 4) + align_up(c * n) + 2 * align_up(c * n * 12);
}
bool carve_sh(Carver &cv, ShDev &d, size_t n, size_t c)
{
    d.means = cv.take<float>(n * 3); d.co = cv.take<float>(48 * n); d.vis = cv.take<uint8_t>(c * n);
    d.gcol = cv.take<float>(c * n * 3); d.col = cv.take<float>(c * n * 3);
    d.gm = cv.take<float>(n * 3); d.gco = cv.take<float>(48 * n);
    return cv.off <= cv.cap;
}

} // namespace

extern "C" {

size_t sh_host_scratch_bytes(int64_t N, int32_t C)
{
    if (N <= 0 || C < 1) return 0;
    const size_t c = (size_t)C;
    const size_t single = sh_footprint((size_t)N, c), chunked = 2 * sh_footprint((size_t)chunk_size(N, false), c);
    return (single > chunked ? single : chunked) + 2 * align_up(c * 12) + align_up(cam_partial_bytes(N, C)) + SCRATCH_SLOP;
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
    const size_t c = (size_t)C, Nn = (size_t)N;
    const int64_t chunk = chunk_size(N, g_campos != nullptr);
    const bool two = chunk < N;

    Carver cv{static_cast<char *>(dev_scratch), 0, dev_scratch_bytes};
    float *d_campos = cv.take<float>(c * 3), *d_gcam = cv.take<float>(c * 3);
    const size_t ws_bytes = cam_partial_bytes(chunk, C);
    float *d_ws = cv.take<float>(ws_bytes / sizeof(float) + 1);
    ShDev dev[2];
    if (!carve_sh(cv, dev[0], (size_t)chunk, c)) return NASG_ERR_WORKSPACE;
    if (two && !carve_sh(cv, dev[1], (size_t)chunk, c)) return NASG_ERR_WORKSPACE;
    if (!d_campos || !d_gcam || !d_ws) return NASG_ERR_WORKSPACE;

    const cudaMemcpyKind H2D = cudaMemcpyHostToDevice, D2H = cudaMemcpyDeviceToHost;
    cudaStream_t user = (cudaStream_t)cuda_stream;
    NASG_TRY_CUDA(cudaMemcpyAsync(d_campos, campos, c * 12, H2D, user));

    auto copy_in = [&](int b, int64_t n0, int64_t nc, cudaStream_t st) -> int {
        const ShDev &d = dev[b];
        const size_t o = (size_t)n0, w = (size_t)nc;
        NASG_TRY_CUDA(copy_rows(d.means, w, means, Nn, 0, o, w, 1, 12, H2D, st));
        NASG_TRY_CUDA(copy_rows(d.co, w, coeffs, Nn, 0, o, w, 48, 4, H2D, st));
        if (vis) NASG_TRY_CUDA(copy_rows(d.vis, w, vis, Nn, 0, o, w, c, 1, H2D, st));
        NASG_TRY_CUDA(copy_rows(d.gcol, w, g_colors, Nn, 0, o, w, c, 12, H2D, st));
        return NASG_OK;
    };
    auto compute = [&](int b, int64_t nc, cudaStream_t st) -> int {
        const ShDev &d = dev[b];
        NASG_TRY(sh_eval_fwd(nc, C, d.means, d.co, d_campos, vis ? d.vis : nullptr, d.col, st));
        return sh_eval_bwd(nc, C, d.means, d.co, d_campos, vis ? d.vis : nullptr, d.gcol, g_means ? d.gm : nullptr,
                           g_coeffs ? d.gco : nullptr, g_campos ? d_gcam : nullptr, d_ws, ws_bytes + sizeof(float), st);
    };
    auto copy_out = [&](int b, int64_t n0, int64_t nc, cudaStream_t st) -> int {
        const ShDev &d = dev[b];
        const size_t o = (size_t)n0, w = (size_t)nc;
        NASG_TRY_CUDA(copy_rows(colors, Nn, d.col, w, o, 0, w, c, 12, D2H, st));
        if (g_means) NASG_TRY_CUDA(copy_rows(g_means, Nn, d.gm, w, o, 0, w, 1, 12, D2H, st));
        if (g_coeffs) NASG_TRY_CUDA(copy_rows(g_coeffs, Nn, d.gco, w, o, 0, w, 48, 4, D2H, st));
        if (g_campos) NASG_TRY_CUDA(cudaMemcpyAsync(g_campos, d_gcam, c * 12, D2H, st));
        return NASG_OK;
    };
    return run_pipeline(N, chunk, user, copy_in, compute, copy_out);
}

} // extern "C"

// ---- NASGabor, tile-record layout: a chunk of Gaussians is a contiguous range of records ---------------
namespace {
struct RecDev { float *params, *gparams, *gcol, *col; uint8_t *vis; };
size_t rec_footprint(size_t n, int K, size_t c, int pk)
{
    return 2 * align_up((size_t)nasg::rec_total_floats((int64_t)n, K, pk) * 4) + align_up(c * n) + 2 * align_up(c * n * 12);
}
bool carve_rec(Carver &cv, RecDev &d, size_t n, int K, size_t c, int pk)
{
    const size_t rf = (size_t)nasg::rec_total_floats((int64_t)n, K, pk);
    d.params = cv.take<float>(rf); d.gparams = cv.take<float>(rf); d.vis = cv.take<uint8_t>(c * n);
    d.gcol = cv.take<float>(c * n * 3); d.col = cv.take<float>(c * n * 3);
    return cv.off <= cv.cap;
}
size_t rec_host_scratch(int64_t N, int32_t K, int32_t C, int pk)
{
    if (N <= 0 || !(K == 2 || K == 4 || K == 8) || C < 1) return 0;
    const size_t c = (size_t)C;
    const size_t single = rec_footprint((size_t)N, K, c, pk), chunked = 2 * rec_footprint((size_t)chunk_size(N, false), K, c, pk);
    return (single > chunked ? single : chunked) + align_up(c * 12) + SCRATCH_SLOP;
}

int rec_host(const nasg_rec_inputs *in, const float *g_colors, float *colors, float *g_params, int norm_mode, void *dev_scratch,
             size_t dev_scratch_bytes, int pk, void *cuda_stream)
{
    if (!in) return NASG_ERR_NULL;
    if (in->N < 0 || in->N > NASG_REC_MAX_N || in->C < 1 || in->C > NASG_REC_MAX_CAMERAS) return NASG_ERR_SHAPE;
    if (!(in->K == 2 || in->K == 4 || in->K == 8)) return NASG_ERR_UNSUPPORTED_K;
    if (norm_mode != NASG_NORM_APPROX && norm_mode != NASG_NORM_EXACT && norm_mode != NASG_NORM_NASG) return NASG_ERR_NORM_MODE;
    if (in->N == 0) return NASG_OK;
    if (!in->params || !in->campos || !g_colors || !colors || !g_params || !dev_scratch) return NASG_ERR_NULL;
    if (dev_scratch_bytes < rec_host_scratch(in->N, in->K, in->C, pk) || !aligned16(dev_scratch)) return NASG_ERR_WORKSPACE;
    const int64_t N = in->N;
    const int K = in->K;
    const size_t c = (size_t)in->C, Nn = (size_t)N;
    const int64_t chunk = chunk_size(N, false);              // a multiple of 256 Gaussians = 8 records (or all of N)
    const bool two = chunk < N;

    Carver cv{static_cast<char *>(dev_scratch), 0, dev_scratch_bytes};
    float *d_campos = cv.take<float>(c * 3);
    RecDev dev[2];
    if (!carve_rec(cv, dev[0], (size_t)chunk, K, c, pk)) return NASG_ERR_WORKSPACE;
    if (two && !carve_rec(cv, dev[1], (size_t)chunk, K, c, pk)) return NASG_ERR_WORKSPACE;
    if (!d_campos) return NASG_ERR_WORKSPACE;

    const cudaMemcpyKind H2D = cudaMemcpyHostToDevice, D2H = cudaMemcpyDeviceToHost;
    cudaStream_t user = (cudaStream_t)cuda_stream;
    NASG_TRY_CUDA(cudaMemcpyAsync(d_campos, in->campos, c * 12, H2D, user));     // replicated; before the pipeline's start event
    const nasg_rec_inputs host = *in;
    const size_t rec_f = (size_t)nasg::rec_total_floats(32, K, pk);              // floats per record

    auto copy_in = [&](int b, int64_t n0, int64_t nc, cudaStream_t st) -> int {
        const RecDev &d = dev[b];
        const size_t o = (size_t)n0, w = (size_t)nc;
        // the chunk's records are one contiguous block: a single copy
        NASG_TRY_CUDA(cudaMemcpyAsync(d.params, host.params + (o / 32) * rec_f, (size_t)nasg::rec_total_floats(nc, K, pk) * 4, H2D, st));
        if (host.vis) NASG_TRY_CUDA(copy_rows(d.vis, w, host.vis, Nn, 0, o, w, c, 1, H2D, st));
        NASG_TRY_CUDA(copy_rows(d.gcol, w, g_colors, Nn, 0, o, w, c, 12, H2D, st));
        return NASG_OK;
    };
    auto compute = [&](int b, int64_t nc, cudaStream_t st) -> int {
        const RecDev &d = dev[b];
        nasg_rec_inputs din = host;
        din.N = nc; din.params = d.params; din.campos = d_campos; din.vis = host.vis ? d.vis : nullptr;
        if (pk) {
            NASG_TRY(nasg_paper_eval_fwd(&din, d.col, norm_mode, st));
            return nasg_paper_eval_bwd(&din, d.gcol, d.gparams, norm_mode, st);
        }
        NASG_TRY(nasg_rec_eval_fwd(&din, d.col, norm_mode, st));
        return nasg_rec_eval_bwd(&din, d.gcol, d.gparams, norm_mode, st);
    };
    auto copy_out = [&](int b, int64_t n0, int64_t nc, cudaStream_t st) -> int {
        const RecDev &d = dev[b];
        const size_t o = (size_t)n0, w = (size_t)nc;
        NASG_TRY_CUDA(copy_rows(colors, Nn, d.col, w, o, 0, w, c, 12, D2H, st));
        NASG_TRY_CUDA(cudaMemcpyAsync(g_params + (o / 32) * rec_f, d.gparams, (size_t)nasg::rec_total_floats(nc, K, pk) * 4, D2H, st));
        return NASG_OK;
    };
    return run_pipeline(N, chunk, user, copy_in, compute, copy_out);
}

} // namespace

extern "C" {

size_t nasg_rec_host_scratch_bytes(int64_t N, int32_t K, int32_t C) { return rec_host_scratch(N, K, C, 0); }
int nasg_rec_eval_fwd_bwd_host(const nasg_rec_inputs *in, const float *g_colors, float *colors, float *g_params,
                               int norm_mode, void *dev_scratch, size_t dev_scratch_bytes, void *cuda_stream)
{
    return rec_host(in, g_colors, colors, g_params, norm_mode, dev_scratch, dev_scratch_bytes, 0, cuda_stream);
}
size_t nasg_paper_host_scratch_bytes(int64_t N, int32_t K, int32_t C) { return rec_host_scratch(N, K, C, 1); }
int nasg_paper_eval_fwd_bwd_host(const nasg_rec_inputs *in, const float *g_colors, float *colors, float *g_params,
                                 int norm_mode, void *dev_scratch, size_t dev_scratch_bytes, void *cuda_stream)
{
    return rec_host(in, g_colors, colors, g_params, norm_mode, dev_scratch, dev_scratch_bytes, 1, cuda_stream);
}

} // extern "C"
