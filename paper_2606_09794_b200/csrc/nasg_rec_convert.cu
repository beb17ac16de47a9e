// nasg_rec_convert.cu — row arrays <-> tile records for EVERY record kind (include/nasg.h: nasg_kind_pack,
// nasg_kind_unpack, nasg_rec16_unpack), so that a C caller never has to build [T][6 + M K][32] records by hand from the
// header comment and can decode a gradient record without the Python helpers. Pure re-ordering: no arithmetic of the method.
// Not on the hot path (records are the persistent layout); one thread per record lane, plain loads and stores.
#include "nasg.h"
#include "nasg_internal.h"

namespace {

constexpr int WT = 32;             // Gaussians per record
constexpr int HDR = 192;           // header floats: means x[32] y[32] z[32], dc r[32] g[32] b[32]

inline bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
inline bool even_K(int K) { return K == 2 || K == 4 || K == 8; }

// components per lobe of a record kind, and which component the padding lanes of the last record get as 1
// (a unit quaternion / the axis (0,0,1): nothing divides by zero in lanes that are never stored); 0 = unknown kind
inline int kind_components(int kind) { return kind == NASG_KIND_QUAT ? 11 : kind == NASG_KIND_PAPER ? 9 : kind == NASG_KIND_ISO ? 7 : kind == NASG_KIND_ASG ? 9 : 0; }
inline int kind_pad_one(int kind) { return kind == NASG_KIND_QUAT || kind == NASG_KIND_ASG ? 0 : kind == NASG_KIND_ISO ? 2 : -1; }

// record float of (pair j, component c, lane, half h):  192 + 64 M j + 64 c + 2 lane + h
__global__ void __launch_bounds__(256) kind_pack_kernel(int64_t N, int K, int M, int pad_one, const float *means, const float *dc, const float *comp, float *rec)
{
    const int64_t n = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t T = (N + WT - 1) / WT;
    if (n >= T * WT) return;
    const int lane = (int)(n & 31);
    float *r = rec + (n >> 5) * (int64_t)(HDR + M * K * WT);
    const bool valid = n < N;
    for (int c = 0; c < 3; ++c) {
        r[c * WT + lane] = valid ? means[3 * n + c] : 0.f;
        r[(3 + c) * WT + lane] = valid ? dc[(int64_t)c * N + n] : 0.f;
    }
    for (int l = 0; l < K; ++l) {
        float *o = r + HDR + (l >> 1) * (2 * WT * M) + 2 * lane + (l & 1);
        const float *src = comp + ((int64_t)l * N + n) * M;
        for (int c = 0; c < M; ++c) o[2 * WT * c] = valid ? src[c] : (c == pad_one ? 1.f : 0.f);
    }
}

__global__ void __launch_bounds__(256) kind_unpack_kernel(int64_t N, int K, int M, const float *rec, float *means, float *dc, float *comp)
{
    const int64_t n = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= N) return;
    const int lane = (int)(n & 31);
    const float *r = rec + (n >> 5) * (int64_t)(HDR + M * K * WT);
    for (int c = 0; c < 3; ++c) {
        if (means) means[3 * n + c] = r[c * WT + lane];
        if (dc) dc[(int64_t)c * N + n] = r[(3 + c) * WT + lane];
    }
    if (!comp) return;
    for (int l = 0; l < K; ++l) {
        const float *o = r + HDR + (l >> 1) * (2 * WT * M) + 2 * lane + (l & 1);
        float *dst = comp + ((int64_t)l * N + n) * M;
        for (int c = 0; c < M; ++c) dst[c] = o[2 * WT * c];
    }
}

// bf16 parameter record (480 words per pair: quat words [32 c + lane], shape [128 + 64 c + 2 lane + h], amp [384 + 32 c + lane];
// a bf16 pair = lobe 2j in the low half, lobe 2j+1 in the high half) -> fp32 row arrays. bf16 -> fp32 is exact.
__global__ void __launch_bounds__(256) rec16_unpack_kernel(int64_t N, int K, const unsigned *rec, float *means, float *quat, float *shape, float *amp, float *dc)
{
    const int64_t n = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= N) return;
    const int lane = (int)(n & 31);
    const unsigned *r = rec + (n >> 5) * (int64_t)(HDR + (K / 2) * 480);
    for (int c = 0; c < 3; ++c) {
        if (means) means[3 * n + c] = __uint_as_float(r[c * WT + lane]);
        if (dc) dc[(int64_t)c * N + n] = __uint_as_float(r[(3 + c) * WT + lane]);
    }
    for (int l = 0; l < K; ++l) {
        const unsigned *o = r + HDR + (l >> 1) * 480;
        const int h = l & 1;
        for (int c = 0; c < 4; ++c) {
            const unsigned w = o[32 * c + lane];
            if (quat) quat[((int64_t)l * N + n) * 4 + c] = __uint_as_float(h ? (w & 0xffff0000u) : (w << 16));
            if (shape) shape[((int64_t)l * N + n) * 4 + c] = __uint_as_float(o[128 + 64 * c + 2 * lane + h]);
        }
        for (int c = 0; c < 3; ++c) {
            const unsigned w = o[384 + 32 * c + lane];
            if (amp) amp[((int64_t)l * 3 + c) * N + n] = __uint_as_float(h ? (w & 0xffff0000u) : (w << 16));
        }
    }
}

int done(cudaError_t e)
{
    if (e != cudaSuccess) return nasg::api_cuda_fail(e);
    nasg::api_count_launches(1);
    return NASG_OK;
}

} // namespace

extern "C" {

int32_t nasg_kind_components(int kind) { return kind_components(kind); }

size_t nasg_kind_floats(int kind, int64_t N, int32_t K)
{
    const int M = kind_components(kind);
    if (M == 0 || N <= 0 || !even_K(K)) return 0;
    return (size_t)((N + WT - 1) / WT) * (size_t)(HDR + M * K * WT);
}

int nasg_kind_pack(int kind, int64_t N, int32_t K, const float *means, const float *dc, const float *comp, float *rec, void *cuda_stream)
{
    const int M = kind_components(kind);
    if (M == 0) return NASG_ERR_NORM_MODE;
    if (N < 0 || N > NASG_REC_MAX_N) return NASG_ERR_SHAPE;
    if (!even_K(K)) return NASG_ERR_UNSUPPORTED_K;
    if (N == 0) return NASG_OK;
    if (!means || !dc || !comp || !rec) return NASG_ERR_NULL;
    if (!aligned16(rec)) return NASG_ERR_ALIGN;
    const int64_t lanes = ((N + WT - 1) / WT) * WT;
    kind_pack_kernel<<<(unsigned)((lanes + 255) / 256), 256, 0, (cudaStream_t)cuda_stream>>>(N, K, M, kind_pad_one(kind), means, dc, comp, rec);
    return done(cudaGetLastError());
}

int nasg_kind_unpack(int kind, int64_t N, int32_t K, const float *rec, float *means, float *dc, float *comp, void *cuda_stream)
{
    const int M = kind_components(kind);
    if (M == 0) return NASG_ERR_NORM_MODE;
    if (N < 0 || N > NASG_REC_MAX_N) return NASG_ERR_SHAPE;
    if (!even_K(K)) return NASG_ERR_UNSUPPORTED_K;
    if (N == 0) return NASG_OK;
    if (!rec) return NASG_ERR_NULL;
    if (!aligned16(rec)) return NASG_ERR_ALIGN;
    kind_unpack_kernel<<<(unsigned)((N + 255) / 256), 256, 0, (cudaStream_t)cuda_stream>>>(N, K, M, rec, means, dc, comp);
    return done(cudaGetLastError());
}

int nasg_rec16_unpack(int64_t N, int32_t K, const float *rec16, float *means, float *quat, float *shape, float *amp, float *dc,
                      void *cuda_stream)
{
    if (N < 0 || N > NASG_REC_MAX_N) return NASG_ERR_SHAPE;
    if (!even_K(K)) return NASG_ERR_UNSUPPORTED_K;
    if (N == 0) return NASG_OK;
    if (!rec16) return NASG_ERR_NULL;
    if (!aligned16(rec16)) return NASG_ERR_ALIGN;
    rec16_unpack_kernel<<<(unsigned)((N + 255) / 256), 256, 0, (cudaStream_t)cuda_stream>>>(
        N, K, reinterpret_cast<const unsigned *>(rec16), means, quat, shape, amp, dc);
    return done(cudaGetLastError());
}

} // extern "C"
