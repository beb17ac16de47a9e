/* nasg.h — C ABI of the B200-native (sm_100a) NASGabor / SH-3 per-Gaussian colour evaluation.
 *
 * What the library computes (arxiv/paper_2606_09794; citations are /root/reference/PAPER.md lines):
 *
 *   d_cn      = normalize(means[n] - campos[c])          central-ray direction, one evaluation per
 *                                                        primitive per frame
 *   colour    = c0 + sum_{l<K} w_l G_l(d)                appearance model, eq.(6)
 *   G         = H p E / I                                NASGabor lobe, eq.(9)
 *               kappa = (d.z+1)/2, tau = a (d.x)^2/(1-(d.z)^2), E = kappa^tau,
 *               p = exp(2 lambda (E kappa - 1)), H = (1+cos(k d.x + phi))/2
 *   I         = pi(1-e^{-2 lambda})/(lambda sqrt(1+a)) (1+Psi),                       eq.(10)
 *               Psi = 2 Lambda e^{-Lambda} sinhc(sqrt(Lambda^2-k^2))/(1-e^{-2 Lambda}), Lambda = lambda(1+a)
 *               (norm_mode 0: the NASG normaliser 2 pi(1-e^{-2 lambda})/(lambda sqrt(1+a)),
 *                what the paper trained with)
 *   SH path   = sum_{j<16} coeff_j Y_j(d), real SH of degree 3, eq.(5)
 *   backward  = exact gradient of sum(g_colors * colors) w.r.t. every parameter and the mean
 *               (through d); eqs.(50)-(65) PAPER.md:754-861 plus the terms derived in DESIGN.md §4.
 *
 * Parameterisation (DESIGN.md §3 readings R1, R5, R12): the frame [x y z] is R(q/|q|) of a per-lobe
 * quaternion q = (w,x,y,z), x = column 0 (carrier axis), z = column 2 (lobe axis); the two
 * log-bandwidths are l1 = log Lambda >= l2 = log lambda, a = Lambda/lambda - 1 >= 0; the phase phi
 * enters the carrier only. No activation is applied to k, phi, w or c0 (Table 8 activations are the
 * caller's); no clamp or +0.5 on the output.
 *
 * Conventions
 *   - Every pointer of the device entry points is a DEVICE pointer, fp32 unless typed otherwise,
 *     row-major with the shape written beside it. The caller owns every buffer; the library never
 *     allocates, never synchronises, keeps no global state, and is CUDA-graph capturable. Work is
 *     enqueued on `cuda_stream` (a cudaStream_t passed as void*; NULL = legacy default stream).
 *   - Outputs are overwritten, never accumulated. colors[c,n,:] of a culled pair (vis[c,n]==0) is 0;
 *     every gradient of a Gaussian culled in all C cameras is 0.
 *   - Return value: 0 (NASG_OK) or a negative NASG_ERR_* code. Nothing is thrown or printed.
 *     Device-side faults (bad pointers) surface at the caller's next synchronisation.
 *   - Inputs are not validated on the device: a zero quaternion or means[n]==campos[c] yields NaN.
 *   - N == 0 is a successful no-op.
 */
#ifndef NASG_H_
#define NASG_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NASG_OK                  0
#define NASG_ERR_NULL           -1  /* a required pointer is NULL                                   */
#define NASG_ERR_SHAPE          -2  /* N < 0, C < 1, C > NASG_MAX_CAMERAS                           */
#define NASG_ERR_UNSUPPORTED_K  -3  /* K not in {1,2,3,4,5,8} (paper: 1..5; cfg4: 8)  */
#define NASG_ERR_ALIGN          -4  /* quat/shape (or their gradients) not 16-byte aligned          */
#define NASG_ERR_WORKSPACE      -5  /* g_campos requested but workspace NULL or too small           */
#define NASG_ERR_CUDA           -6  /* launch / copy failed: cudaGetLastError()                     */
#define NASG_ERR_NORM_MODE      -7  /* norm_mode not 0, 1 or 2                                      */
#define NASG_ERR_NOALLOC_SIZE   -8  /* nasg_eval_bwd_noalloc: the problem needs more scratch than   */
                                    /* the built-in NASG_NOALLOC_WS_BYTES (use nasg_eval_bwd)       */

#define NASG_MAX_CAMERAS 64

#define NASG_NORM_APPROX 0          /* NASG normaliser, carrier ignored              */
#define NASG_NORM_EXACT  1          /* eq.(10) as printed                        */
#define NASG_NORM_NASG   2          /* pure NASG lobe: no Gabor carrier. k and phi   */
                                    /* (shape[...,2:4]) are ignored = taken as 0, their gradients   */
                                    /* are written as 0; at k = 0 both normalisers above coincide   */

/* Inputs of one evaluation: N Gaussians, K lobes each, C cameras. */
typedef struct {
    int64_t N;
    int32_t K;
    int32_t C;
    const float   *means;   /* [N,3]                                                                */
    const float   *quat;    /* [K,N,4]  (w,x,y,z), any non-zero norm; 16-byte aligned               */
    const float   *shape;   /* [K,N,4]  (log Lambda, log lambda, k, phi), log Lambda >= log lambda;  */
                            /*          16-byte aligned                                             */
    const float   *amp;     /* [K,3,N]  RGB amplitude w_l (planar)                                   */
    const float   *dc;      /* [3,N]    c0 (planar)                                                  */
    const float   *campos;  /* [C,3]                                                                */
    const uint8_t *vis;     /* [C,N] non-zero = visible, or NULL = all visible                      */
} nasg_inputs;

/* Gradient outputs of nasg_eval_bwd; same shapes as the inputs. Any pointer may be NULL = skip. */
typedef struct {
    float *g_means;         /* [N,3]                                                                */
    float *g_quat;          /* [K,N,4]  w.r.t. the raw (unnormalised) quaternion; 16-byte aligned   */
    float *g_shape;         /* [K,N,4]  (d/dlogLambda, d/dloglambda, d/dk, d/dphi); 16-byte aligned */
    float *g_amp;           /* [K,3,N]                                                              */
    float *g_dc;            /* [3,N]                                                                */
    float *g_campos;        /* [C,3]    optional per-camera term (needs workspace)                  */
    void  *workspace;       /* device scratch, >= nasg_workspace_bytes(N,K,C); only for g_campos    */
    size_t workspace_bytes;
} nasg_grads;

/* colors[C,N,3] = c0 + sum_l w_l G_l(d)   (eq.(6), eq.(9), eq.(10)). Asynchronous on cuda_stream. */
int nasg_eval_fwd(const nasg_inputs *in, float *colors, int norm_mode, void *cuda_stream);

/* Gradients of sum(g_colors[C,N,3] * colors) (Supplementary F + DESIGN.md §4). Nothing saved by the
 * forward is needed: the lobe values are recomputed. Each gradient element is written exactly once
 * by one thread (no atomics); g_campos is a per-thread partial -> warp-shuffle -> block -> second-stage
 * reduction through `workspace`, in a fixed order: bit-reproducible for a given N and device. */
int nasg_eval_bwd(const nasg_inputs *in, const float *g_colors, const nasg_grads *out, int norm_mode,
                  void *cuda_stream);

/* Comparison path: real SH degree 3, coeffs [16,3,N] (j = l^2+l+m, Condon-Shortley sign kept,
 * DESIGN.md R15), colors[C,N,3] = sum_j coeffs[j,:,n] Y_j(d). */
int sh_eval_fwd(int64_t N, int32_t C, const float *means, const float *coeffs, const float *campos,
                const uint8_t *vis, float *colors, void *cuda_stream);
int sh_eval_bwd(int64_t N, int32_t C, const float *means, const float *coeffs, const float *campos,
                const uint8_t *vis, const float *g_colors, float *g_means, float *g_coeffs,
                float *g_campos, void *workspace, size_t workspace_bytes, void *cuda_stream);

/* ---- tile-record parameter layout ("layout v2"): the fast path ---------------------------------------
 * The per-Gaussian evaluation is issue-bound on B200 once C > 1, and with the row arrays above a
 * warp's 32 Gaussians are 24-29 separate row segments whose addressing alone is 17-20 % of the executed instructions.
 * The record layout stores everything a warp tile needs as ONE contiguous 16-byte aligned block, lobes interleaved in
 * pairs so that they load as packed f32x2 operands:
 *
 *   params: float [T][6 + 11 K][32],  T = ceil(N / 32);  record of tile t (Gaussians n = 32 t + lane), floats:
 *     [  0 ..  95]   means, planar:  x[32] y[32] z[32]
 *     [ 96 .. 191]   dc (c0), planar: r[32] g[32] b[32]
 *     [192 + 704 j + 64 c + 2 lane + h]   component c of lobe 2 j + h   (lobe pair j < K/2, h = 0,1)
 *                    c = 0..3 quaternion (w,x,y,z) | 4..7 (log Lambda, log lambda, k, phi) | 8..10 amplitude (r,g,b)
 *
 * The same 6 + 11 K floats per Gaussian as the row arrays (the algorithmic bytes do not change); lanes past N in the
 * last record are padding (written by nasg_rec_pack as a unit quaternion and zeros; never read back as results).
 * Gradient records have the same layout (g_means, g_dc, then per pair the gradients of the 11 components); padding
 * lanes of the last gradient record are not written. colors / g_colors [C,N,3] and vis [C,N] keep their shapes: they
 * belong to the neighbouring stages (rasteriser). Restrictions of these entry points: K in {2, 4, 8}, C <= 4 (more
 * cameras: call per batch of 4 and add the gradient records, or use the row-array entry points), no g_campos.
 * g_colors / vis rows are moved with bulk copies when N % 4 == 0 (N % 16 == 0 with a mask) and the pointers are
 * 16-byte aligned; otherwise they are loaded per lane (correct, slower). Everything else is as above: device
 * pointers, caller-owned, asynchronous on cuda_stream, outputs overwritten, CUDA-graph capturable. */
/* Optional hint, OR-ed into norm_mode of nasg_rec_eval_fwd / nasg_rec_eval_bwd: the visibility mask is spatially coherent
 * (the scene is stored in spatial order, so frustum culling removes runs of consecutive Gaussians). The kernels then test per
 * warp of 32 Gaussians which cameras ANY of them sees, skip the lobe evaluations of the others, and skip all lobe arithmetic of
 * a tile culled in every camera (step F0). Results are identical with and without the hint; with iid masks it only costs time
 * (~5 % of the forward), which is why it is a hint and not the default. Ignored by the other record kinds and for C = 1. */
#define NASG_HINT_COHERENT_VIS 0x100
#define NASG_REC_MAX_CAMERAS 4
#define NASG_REC_MAX_N ((int64_t)1 << 35)

typedef struct {
    int64_t N;
    int32_t K;              /* 2, 4 or 8                                                            */
    int32_t C;              /* 1..4                                                                 */
    const float   *params;  /* nasg_rec_floats(N, K) floats, 16-byte aligned                        */
    const float   *campos;  /* [C,3]                                                                */
    const uint8_t *vis;     /* [C,N] or NULL                                                        */
} nasg_rec_inputs;

/* Floats in a parameter (or gradient) record array for N Gaussians of K lobes; 0 if K is unsupported. */
size_t nasg_rec_floats(int64_t N, int32_t K);
/* Row arrays -> records (reads means, quat, shape, amp, dc of `in`; campos, vis, C are ignored). */
int nasg_rec_pack(const nasg_inputs *in, float *params, void *cuda_stream);
/* Records -> row arrays (parameters or gradients alike); any output pointer may be NULL = skip. */
int nasg_rec_unpack(int64_t N, int32_t K, const float *rec, float *means, float *quat, float *shape,
                    float *amp, float *dc, void *cuda_stream);
/* nasg_eval_fwd / nasg_eval_bwd on records: same function, same gradient (eq.(6), (9), (10)). */
int nasg_rec_eval_fwd(const nasg_rec_inputs *in, float *colors, int norm_mode, void *cuda_stream);
int nasg_rec_eval_bwd(const nasg_rec_inputs *in, const float *g_colors, float *g_params, int norm_mode,
                      void *cuda_stream);

/* ---- the paper's own parameter record --------------------------------------
 * 3 + 9 K appearance floats per primitive (Table 5) instead of 3 + 11 K: per lobe
 * the RAW (pre-activation) values of Table 8, activations applied inside the kernels:
 *     (c_theta, c_phi, c_tau) = tanh(raw), sines = +sqrt(1 - c^2)       frame of Supplementary C:
 *     z = (c_theta s_phi, s_theta s_phi, c_phi),  x = (c_theta c_phi c_tau - s_theta s_tau, s_theta c_phi c_tau + c_theta s_tau, -s_phi c_tau)
 *     lambda = exp(raw), a = exp(raw), k = 20 (tanh(raw) + 1), w = tanh(raw); no phase; c0 (dc) has no activation.
 * Stored as tile records like the layout above with 9 components per lobe:
 *     [192 + 576 j + 64 c + 2 lane + h],  c = 0..2 (theta, phi, tau) | 3..5 (lambda, a, k) | 6..8 amplitude (r,g,b)
 * nasg_paper_floats(N, K) floats. The lobe function and the normaliser are those of nasg_eval_fwd (eq.(9), eq.(10)
 * / norm_mode); the gradient record holds dL/d(raw) (the chain rule of eqs.(37)-(44), and of the
 * activations, is applied inside the backward kernel). Same restrictions as nasg_rec_eval_*. */
size_t nasg_paper_floats(int64_t N, int32_t K);
int nasg_paper_eval_fwd(const nasg_rec_inputs *in, float *colors, int norm_mode, void *cuda_stream);
int nasg_paper_eval_bwd(const nasg_rec_inputs *in, const float *g_colors, float *g_params, int norm_mode,
                        void *cuda_stream);

/* ---- reduced-precision parameter STORAGE: bfloat16 quaternion and amplitude ----------
 * The record of nasg_rec_* with the quaternion and the amplitude of every lobe stored as bfloat16 (the arithmetic stays fp32;
 * the (log Lambda, log lambda, k, phi) group stays fp32 because it feeds the exponent; means and dc stay fp32). Per pair:
 *     words [32 c + lane]           c = 0..3   quaternion: bf16 of lobe 2j | bf16 of lobe 2j+1 << 16
 *     words [128 + 64 c + 2 lane + h]  c = 0..3  shape, fp32
 *     words [384 + 32 c + lane]     c = 0..2   amplitude, bf16 pair
 * = 480 32-bit words per pair after the 192-word header: 36 instead of 50 words per Gaussian at K = 4 (-28 % parameter bytes).
 * nasg_rec16_pack rounds to nearest even. The GRADIENT record is the fp32 record of nasg_rec_eval_bwd (nasg_rec_floats).
 * What bf16 storage does to the colours (oracle on the rounded values against the fp32 values, cfg2 recipe): DESIGN.md 11. */
size_t nasg_rec16_floats(int64_t N, int32_t K);          /* 32-bit words of a bf16 parameter record array */
int nasg_rec16_pack(const nasg_inputs *in, float *params, void *cuda_stream);
int nasg_rec16_eval_fwd(const nasg_rec_inputs *in, float *colors, int norm_mode, void *cuda_stream);
int nasg_rec16_eval_bwd(const nasg_rec_inputs *in, const float *g_colors, float *g_params, int norm_mode,
                        void *cuda_stream);

/* ---- other spherical functions of the paper's Table 6 in the same skeleton ---------
 * colour = c0 + sum_l w_l c_l G_l(d . zhat_l) (eq.(6)) with an ISOTROPIC, normalised lobe:
 *     NASG_ISO_SG      0   Spherical Gaussian  G = exp{lambda (z.d - 1)},  c = lambda/(2 pi (1 - e^{-2 lambda})),  lambda = e^raw
 *     NASG_ISO_BETA    1   Spherical Beta      G = max(z.d, 0)^beta,       c = (beta + 1)/(2 pi),                  beta = e^raw
 *     NASG_ISO_CAUCHY  2   Spherical Cauchy    G = ((1 - rho^2)/(1 + rho^2 - 2 rho z.d))^2,  c = 1/(4 pi),          rho = 1/(1 + e^-raw)
 * (Table 6 prints the Cauchy denominator as 1 - rho^2 - 2 rho z.d; only 1 + rho^2 - 2 rho z.d integrates to 1/c: DESIGN.md R19.)
 * zhat = z/|z| of a free 3-vector per lobe (gradient through the normalisation). Tile records with 7 components per lobe:
 *     [192 + 448 j + 64 c + 2 lane + h],  c = 0..2 axis (x,y,z) | 3 shape (raw) | 4..6 amplitude (r,g,b);  [T][6 + 7 K][32]
 * nasg_iso_floats(N, K) floats; the gradient record has the same layout (dL/d axis, dL/d raw, dL/d w). Same restrictions
 * and conventions as nasg_rec_eval_* (`kind` takes the place of norm_mode; a bad kind returns NASG_ERR_NORM_MODE). */
#define NASG_ISO_SG     0
#define NASG_ISO_BETA   1
#define NASG_ISO_CAUCHY 2
size_t nasg_iso_floats(int64_t N, int32_t K);
int nasg_iso_eval_fwd(const nasg_rec_inputs *in, float *colors, int kind, void *cuda_stream);
int nasg_iso_eval_bwd(const nasg_rec_inputs *in, const float *g_colors, float *g_params, int kind, void *cuda_stream);

/* Anisotropic Spherical Gaussian (Table 6, [XSD*13]), not normalised (Table 6: "Not analytical"):
 *     G(d) = max(d.z, 0) exp{-mu (d.x)^2 - lambda (d.y)^2},   [x y z] = R(q/|q|) (Hamilton (w,x,y,z), as nasg_inputs.quat),
 *     mu = e^raw0, lambda = e^raw1;   colour = c0 + sum_l w_l G_l(d) (eq.(6)).
 * At d.z = 0 the lobe has a kink; the derivative there is taken as 0 (the far side). Tile records with 9 components per lobe:
 *     [192 + 576 j + 64 c + 2 lane + h],  c = 0..3 quaternion (w,x,y,z) | 4 raw mu | 5 raw lambda | 6..8 amplitude (r,g,b);
 *     [T][6 + 9 K][32] floats = nasg_asg_floats(N, K); the gradient record has the same layout (dL/dq through the
 * normalisation, dL/draw, dL/dw). Same restrictions and conventions as nasg_rec_eval_* (no norm_mode). */
size_t nasg_asg_floats(int64_t N, int32_t K);
int nasg_asg_eval_fwd(const nasg_rec_inputs *in, float *colors, void *cuda_stream);
int nasg_asg_eval_bwd(const nasg_rec_inputs *in, const float *g_colors, float *g_params, void *cuda_stream);

/* ---- building and decoding records of EVERY kind from C (no Python helper needed) ------------------------------------
 * All record kinds share one skeleton: [T][6 + M K][32] floats, T = ceil(N / 32), the 192-float header (means planar,
 * dc planar) and then, per lobe pair j, M components of 64 floats each: float [192 + 64 M j + 64 c + 2 lane + h] is
 * component c of lobe 2 j + h of Gaussian 32 t + lane. The kinds differ in M and in what the components are:
 *     NASG_KIND_QUAT   0   M = 11   q_w q_x q_y q_z | log Lambda, log lambda, k, phi | w_r w_g w_b        (nasg_rec_*)
 *     NASG_KIND_PAPER  1   M =  9   raw theta, phi, tau | raw lambda, a, k | raw w_r w_g w_b                (nasg_paper_*)
 *     NASG_KIND_ISO    2   M =  7   axis x y z | raw shape | w_r w_g w_b                                    (nasg_iso_*)
 *     NASG_KIND_ASG    4   M =  9   q_w q_x q_y q_z | raw mu, raw lambda | w_r w_g w_b                      (nasg_asg_*)
 * nasg_kind_pack builds such a record array from means [N,3], dc [3,N] and ONE row array comp [K,N,M] that holds the M
 * components of every lobe in the order above (note: the amplitude sits per lobe row here, not planar as nasg_inputs.amp).
 * Padding lanes of the last record are written as zeros, except a 1 in q_w (kinds 0, 4) or axis z (kind 2), so that the
 * never-stored padding lanes divide by nothing. nasg_kind_unpack is the inverse, for parameter and gradient records alike
 * (any output pointer may be NULL = skip). nasg_rec16_unpack decodes the bf16 parameter record of nasg_rec16_pack into
 * fp32 row arrays (exact; shapes as nasg_inputs; any output may be NULL); the gradient record of the bf16 kind is a
 * kind-0 record. A bad kind returns NASG_ERR_NORM_MODE; K must be 2, 4 or 8; rec must be 16-byte aligned. Device pointers,
 * asynchronous on cuda_stream, nothing allocated. These kernels re-order only and are not tuned: records are the
 * persistent layout, conversion is not a per-step operation.
 * The host-buffer end-to-end calls below exist for the quaternion and the paper record only; the isotropic, ASG and bf16
 * kinds are device-only by design (their records are built on the device with the calls above and stay there). */
#define NASG_KIND_QUAT  0
#define NASG_KIND_PAPER 1
#define NASG_KIND_ISO   2
#define NASG_KIND_ASG   4
int32_t nasg_kind_components(int kind);                          /* M, or 0 for an unknown kind */
size_t nasg_kind_floats(int kind, int64_t N, int32_t K);        /* floats of a record array (= nasg_rec/paper/iso/asg_floats) */
int nasg_kind_pack(int kind, int64_t N, int32_t K, const float *means, const float *dc, const float *comp, float *rec,
                   void *cuda_stream);
int nasg_kind_unpack(int kind, int64_t N, int32_t K, const float *rec, float *means, float *dc, float *comp,
                     void *cuda_stream);
int nasg_rec16_unpack(int64_t N, int32_t K, const float *rec16, float *means, float *quat, float *shape, float *amp,
                      float *dc, void *cuda_stream);

/* End-to-end with HOST buffers, as nasg_eval_fwd_bwd_host below: params / g_params are HOST record arrays, campos, vis,
 * g_colors, colors HOST arrays. A chunk of Gaussians is a contiguous block of records, so each chunk moves with one
 * copy per direction for the parameters / gradients plus one strided copy each for vis, g_colors and colors. Padding
 * lanes of the last gradient record are copied back as whatever the device buffer held (never results). */
size_t nasg_rec_host_scratch_bytes(int64_t N, int32_t K, int32_t C);
int nasg_rec_eval_fwd_bwd_host(const nasg_rec_inputs *in, const float *g_colors, float *colors, float *g_params,
                               int norm_mode, void *dev_scratch, size_t dev_scratch_bytes, void *cuda_stream);
/* the same for paper-native records (nasg_paper_floats(N, K) floats) */
size_t nasg_paper_host_scratch_bytes(int64_t N, int32_t K, int32_t C);
int nasg_paper_eval_fwd_bwd_host(const nasg_rec_inputs *in, const float *g_colors, float *colors, float *g_params,
                                 int norm_mode, void *dev_scratch, size_t dev_scratch_bytes, void *cuda_stream);

/* Bytes of device scratch nasg_eval_bwd / sh_eval_bwd need when g_campos != NULL (pass K = 0 for SH). */
size_t nasg_workspace_bytes(int64_t N, int32_t K, int32_t C);

/* ---- backward with g_campos for callers that cannot allocate device memory ----------------------------------
 * nasg_eval_bwd asks the caller for `workspace` when g_campos is wanted. Not every caller can produce one: a plug-in
 * that lives inside a host application (a viewer, a trainer with its own caching allocator) and must not call
 * cudaMalloc behind that application's back; a real-time render loop, where cudaMalloc / cudaFree synchronise the
 * device and drop frames; a process whose device memory was handed out completely at start-up; a C caller that links
 * this library without the CUDA runtime. nasg_eval_bwd_noalloc is nasg_eval_bwd for them: same inputs, same outputs,
 * same kernels and summation order (so the same values), but the per-block partial sums of g_campos go to a fixed
 * array of NASG_NOALLOC_WS_BYTES that is part of the library image in device memory. The call allocates and frees
 * nothing (no cudaMalloc / cudaFree, no allocating library routine); out->workspace and out->workspace_bytes are
 * ignored. What to know before using it:
 *   - Cost: every GPU on which the library is loaded holds NASG_NOALLOC_WS_BYTES (1 MiB) from module load until the
 *     process exits, used or not.
 *   - Limit: nasg_workspace_bytes(N, K, C) <= nasg_noalloc_workspace_bytes(), i.e. ceil(N / 256) * C <= 87,381 (for
 *     example N <= 5.59 million at C = 4, N <= 22.3 million at C = 1). Larger problems are refused with
 *     NASG_ERR_NOALLOC_SIZE and nothing is launched; use nasg_eval_bwd with your own workspace for those.
 *   - out->g_campos is required (NASG_ERR_NULL otherwise): without it the backward needs no scratch and nasg_eval_bwd
 *     already serves the caller. The other gradient pointers stay optional.
 *   - First call on a device: the library looks up the array's device address there (cudaGetSymbolAddress, once per
 *     device, with the calling thread's current device; this may load the module on that device). Make that first
 *     call on each device outside of any stream capture; later calls only launch the two kernels.
 *   - One array per device, shared by every call: two calls whose kernels can overlap on the GPU (different streams
 *     without an ordering between them, or two host threads on different streams) race on it and both g_campos
 *     results are garbage. Calls on one stream, or ordered by events, are safe. The array keeps the last call's
 *     partial sums; the next call overwrites every entry it later reads, so nothing has to be cleared in between. */
#define NASG_NOALLOC_WS_BYTES (1u << 20)
size_t nasg_noalloc_workspace_bytes(void);            /* = NASG_NOALLOC_WS_BYTES */
int nasg_eval_bwd_noalloc(const nasg_inputs *in, const float *g_colors, const nasg_grads *out, int norm_mode,
                          void *cuda_stream);

/* ---- end-to-end entry points with HOST buffers -------------------------------------------------
 * Same computation, forward then backward, but every array pointer in `in`, `colors`, `g_colors`
 * and `out` is a HOST pointer (pinned memory makes the copies asynchronous and fast; pageable works).
 * The call copies the inputs to `dev_scratch` (a DEVICE buffer of >= *_host_scratch_bytes), runs the
 * two kernels and copies colours and gradients back. Gaussians are independent, so a large call is cut
 * into chunks of contiguous n-ranges that run as a three-stage pipeline (H2D of chunk i+1, kernels on
 * chunk i, D2H of chunk i-1) on three streams the library creates once per device on first use: PCIe is
 * full duplex, so the copies in the two directions overlap. Ordering is that of cuda_stream: the work
 * starts after what is already queued there, cuda_stream waits for the last copy, and the call returns
 * without synchronising; host buffers must stay valid until cuda_stream reaches that point.
 * A call that asks for g_campos (a sum over all Gaussians) runs as one chunk. Not CUDA-graph capturable.
 * Calls on one device are serialised while they enqueue. out->workspace is ignored (carved from
 * dev_scratch). */
size_t nasg_host_scratch_bytes(int64_t N, int32_t K, int32_t C);
int nasg_eval_fwd_bwd_host(const nasg_inputs *in, const float *g_colors, float *colors,
                           const nasg_grads *out, int norm_mode, void *dev_scratch,
                           size_t dev_scratch_bytes, void *cuda_stream);
size_t sh_host_scratch_bytes(int64_t N, int32_t C);
int sh_eval_fwd_bwd_host(int64_t N, int32_t C, const float *means, const float *coeffs,
                         const float *campos, const uint8_t *vis, const float *g_colors,
                         float *colors, float *g_means, float *g_coeffs, float *g_campos,
                         void *dev_scratch, size_t dev_scratch_bytes, void *cuda_stream);

/* Human-readable text for a return code (static string; for NASG_ERR_CUDA the last CUDA error). */
const char *nasg_strerror(int code);

/* Library version, e.g. "0.1.0 sm_100a". */
const char *nasg_version(void);

/* Number of kernels the library has launched since load (all entry points; for bench accounting). */
int64_t nasg_launch_count(void);

/* Test hook: which kernel family the device entry points dispatch to. 0 (default) = automatic: the tile kernels
 * (even K, C <= 4, N % 4 == 0 — N % 16 == 0 with a mask —, 16-byte aligned arrays, no g_campos), else the
 * cp.async ring kernels (C <= 4), else the generic kernels; 1 = generic kernels only; 2 = never the tile kernels.
 * Process-wide; exists so that the parity tests can compare every family with the oracle on the same inputs.
 * The library never reads the environment. */
void nasg_debug_set_path(int path);

#ifdef __cplusplus
}
#endif
#endif /* NASG_H_ */
