/*
 * nvfp4.h -- C ABI of the B200-native NVFP4 GEMV hot path of arxiv/paper_2606_13233.
 *
 * What the library computes (citations are PAPER.md lines; "R<n>" = a reading in DESIGN.md):
 *   - the format: NVFP4 = E2M1 4-bit elements, one FP8-E4M3 scale per block of 16
 *     consecutive K, one FP32 global scale per tensor (PAPER.md:344-349 Table 7, :359, :175);
 *   - the operation: the small-M linear projection  Y[M,N] = X[M,K] * W[N,K]^T
 *     (Sec. 5 "Y = XW ... at small M", stored here by output channel, R7),
 *     executed on CUDA cores as a single streaming pass over W (Sec. 5.2);
 *   - the activation quantizer "Q" that feeds it (Table 3 :209-217).
 *
 * Conventions common to every call
 *   - extern "C"; every function returns an int status (0 = NVFP4_OK, negative = error)
 *     unless it returns a size or a string.
 *   - Every pointer marked [device] is CUDA device memory owned by the CALLER and must be
 *     16-byte aligned; the library never allocates, frees or retains caller memory.
 *     Pinned, device-mapped HOST memory (cudaHostAlloc / cudaHostRegister under unified addressing) qualifies
 *     for the BF16 activation inputs and the y outputs: the kernels then read / write it over PCIe themselves
 *     ("zero-copy"; each activation element is read once, each output written once).  Weights, workspaces and
 *     the NVFP4 intermediates belong in device memory.
 *   - Calls are ASYNCHRONOUS: they enqueue kernels on `stream` (a cudaStream_t passed as
 *     void*, NULL = the legacy default stream) and return; they never synchronise, never
 *     read device data on the host, and are capturable in a CUDA graph.
 *   - There is no CPU fallback. On a machine with no usable CUDA device every compute call
 *     returns NVFP4_ERR_CUDA.
 *   - Canonical NVFP4 layout of a tensor T[R,K] (the oracle's layout):
 *       codes  uint8 [R, K/2]  byte j of a row = element k=2j in the LOW nibble, k=2j+1 in
 *                              the HIGH nibble; a nibble is sign-magnitude E2M1 `s e1 e0 m`
 *       scales uint8 [R, K/16] E4M3 ("fn"), one per 16 consecutive k, always 0x00..0x7E
 *       g      float           per-tensor global scale;  value = g * E4M3(scale) * E2M1(code)
 *   - Shape limits: 1 <= M <= 8, N >= 1, K >= 16 and K % 16 == 0, N*K < 2^40.
 *     Anything else -> NVFP4_ERR_UNSUPPORTED_SHAPE.
 *   - Non-finite inputs (NaN/Inf activations): behaviour undefined (documented, untested).
 */
#ifndef NVFP4_B200_H_
#define NVFP4_B200_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NVFP4_ABI_VERSION 2

/* status codes */
#define NVFP4_OK                      0
#define NVFP4_ERR_INVALID_ARG        -1   /* NULL pointer, bad enum value, workspace too small */
#define NVFP4_ERR_UNSUPPORTED_SHAPE  -2   /* M, N, K or a leading dimension outside the limits */
#define NVFP4_ERR_ALIGNMENT          -3   /* a device pointer is not 16-byte aligned */
#define NVFP4_ERR_CUDA               -4   /* a CUDA runtime call failed; see nvfp4_last_cuda_error */

/* nvfp4_gemv `mode` */
#define NVFP4_MODE_W4A4   0   /* x = NVFP4 codes + scales + global scale ("W4A4") */
#define NVFP4_MODE_W4A16  1   /* x = BF16 activations consumed directly (BASELINE.json configs[3]) */

/* nvfp4_gemv `y_dtype` */
#define NVFP4_DTYPE_F32   0
#define NVFP4_DTYPE_BF16  1   /* round-to-nearest-even of the FP32 result */

/* nvfp4_quantize_act `gscale_mode` */
#define NVFP4_GSCALE_DYNAMIC 0 /* g = max|X| / 2688 over the whole [M,K] call argument; WRITTEN to *gscale (R3) */
#define NVFP4_GSCALE_STATIC  1 /* *gscale is READ (a calibrated value, the paper's deployed flow) */
#define NVFP4_GSCALE_DYNAMIC_PER_ROW 2 /* per-token variant (R3): gscale[m] = max|X[m,:]| / 2688, M floats WRITTEN;
                                         feeds nvfp4_gemv_rowscale.  Single-launch sizes only (M*K <= 524288). */

/* ABI version == repacked-blob format version. */
int nvfp4_version(void);

/* Text of the last CUDA error seen by the calling thread's library calls ("" if none).
 * The pointer stays valid until the next library call on this thread. */
const char* nvfp4_last_cuda_error(void);

/*
 * Activation quantizer, steps a1+a2 of SURVEY.md 8(a) (the paper's kernel "Q").
 * BF16 X[M,K] -> canonical NVFP4.  Bit-exact contract (R1, R2; every op one IEEE binary32
 * round-to-nearest-even op, in this order):
 *   g = max|X| / 2688;  per 16-block: t = amax_b / 6; u = t / g; scale = E4M3_RNE(min(u,448));
 *   d = g * E4M3(scale);  code = sign(x) | E2M1_RNE_sat(|x / d|);  g == 0 or d == 0 -> codes 0.
 *
 *   x_bf16   [device] BF16 bits, row m at x_bf16 + m*ldx elements; ldx >= K, ldx % 8 == 0
 *   codes    [device] out, uint8 [M, K/2] contiguous
 *   scales   [device] out, uint8 [M, K/16] contiguous (row-major, "non-swizzled")
 *   gscale   [device] one float; written (DYNAMIC) or read (STATIC)
 *   workspace/ws_bytes: unused by this version (may be NULL / 0); kept for ABI stability.
 * One kernel launch for M*K <= 524288 (a thread-block cluster does the tensor-wide amax on chip,
 * X is read once); larger tensors take two launches.
 */
int nvfp4_quantize_act(const void* x_bf16, int M, int K, int64_t ldx,
                       uint8_t* codes, uint8_t* scales, float* gscale, int gscale_mode,
                       void* workspace, size_t ws_bytes, void* stream);

/*
 * Offline weight repack, step a0.  The blob holds exactly the information of the canonical
 * (codes, scales) pair, permuted into the order the GEMV's 128-bit loads consume
 * (a 128-byte versioned header {magic "NVF4", ABI version << 16 | KP,
 * N, K, cell bytes, tiles, cells} followed by 4608-byte cells of 32/KP rows x 256*KP k, where the
 * number of K parts KP in {1,2,4,..,32} is a fixed function of (N, K) unless overridden with
 * nvfp4_set_layout_kparts); rows are padded to a multiple of 32/KP and K to a multiple of 256*KP
 * with zero codes / zero scales (<= 3% extra for K).  nvfp4_repacked_bytes returns 0 for an
 * unsupported shape.
 *   codes  [device] uint8 [N, K/2];  scales [device] uint8 [N, K/16];  blob_out [device].
 * nvfp4_unpack_weight is the exact inverse (blob -> canonical, byte-identical).
 * The blob is the library's only persistent artefact: nvfp4_gemv validates the header on the
 * device against the (N, K, KP, ABI version) of its own call and writes NaN to EVERY output element
 * if they differ (a stale or foreign blob never yields plausible numbers).
 * Ordering: nvfp4_gemv starts streaming the blob before it waits for its stream predecessor
 * (programmatic dependent launch), so the blob must not be WRITTEN by the kernel launched
 * immediately before nvfp4_gemv on the same stream; nvfp4_repack_weight itself ends with an empty
 * kernel that makes repack -> gemv safe.
 */
size_t nvfp4_repacked_bytes(int N, int K);
int nvfp4_repack_weight(const uint8_t* codes, const uint8_t* scales, int N, int K,
                        void* blob_out, void* stream);
int nvfp4_unpack_weight(const void* blob, int N, int K,
                        uint8_t* codes_out, uint8_t* scales_out, void* stream);

/*
 * The GEMV / skinny GEMM, steps a3..a7:  Y[m,n] = sum_k vX[m,k] * vW[n,k],
 * one pass over the repacked W, each decoded weight reused for all M rows (PAPER.md:161,
 * challenge C1 :151), products exact inside a 16-block, FP32 accumulation across blocks (R8).
 *   mode      NVFP4_MODE_W4A4 or NVFP4_MODE_W4A16
 *   w_blob    [device] from nvfp4_repack_weight for this (N, K)
 *   w_gscale  [device] one float, the weight tensor's global scale
 *   x         [device] W4A4: uint8 codes, row m at x + m*ldx BYTES'-worth of elements, i.e.
 *                      ldx counts code bytes (>= K/2, % 8 == 0);
 *                      W4A16: BF16 bits, ldx counts elements (>= K, % 8 == 0)
 *   x_scales  [device] W4A4 only: uint8 [M, K/16] contiguous;  NULL for W4A16
 *   x_gscale  [device] W4A4 only: one float (e.g. the quantizer's output);  NULL for W4A16
 *   y         [device] out, row m at y + m*ldy elements of y_dtype; ldy >= N
 *   workspace [device] REQUIRED, at least nvfp4_gemv_workspace_bytes(M,N,K) bytes (never 0: the
 *             weight stream is cut into equal shares per SM wherever that falls, so row tiles at
 *             the cuts are completed through it): arrival counters and FP32 partials of the
 *             row tiles cut between CTAs / K slices.  It must be ZERO-FILLED once before its first use; every
 *             call leaves it zero-filled where that matters (the counters), so it can be
 *             reused by any later call on the same stream, and by CUDA-graph replays.  Calls
 *             that may run concurrently need separate workspaces.  The size depends on the
 *             launch shape in effect (query again after nvfp4_gemv_set_config).
 * Acceptance (BASELINE.json north_star): |y - y_ref| <= 1e-3 * sum_k|w_k x_k| + 1e-6.
 */
size_t nvfp4_gemv_workspace_bytes(int M, int N, int K);
int nvfp4_gemv(int mode, const void* w_blob, const float* w_gscale, int N, int K,
               const void* x, const uint8_t* x_scales, const float* x_gscale, int M, int64_t ldx,
               void* y, int y_dtype, int64_t ldy,
               void* workspace, size_t ws_bytes, void* stream);

/*
 * Any-M entry point (the paper's runtime dispatches per (M, shape) between its CUDA-core kernel and a tensor-core GEMM,
 * PAPER.md:526-532 App. C.3; this library has only the CUDA-core kernel): M <= 8 is nvfp4_gemv; larger M runs as
 * ceil(M/8) consecutive GEMV passes over 8-row chunks of x / y on the same stream (W is streamed once per chunk:
 * correct and deterministic, but not a prefill kernel).  x_scales is [M, K/16] contiguous, x_gscale one float for
 * the whole [M, K] tensor; rows must be 16-byte aligned (ldx % 16 == 0 for codes, ldx % 8 == 0 for BF16; ldy * element size % 16 == 0).
 * workspace >= nvfp4_linear_workspace_bytes(M, N, K), zero-filled once.
 */
size_t nvfp4_linear_workspace_bytes(int M, int N, int K);
int nvfp4_linear(int mode, const void* w_blob, const float* w_gscale, int N, int K,
                 const void* x, const uint8_t* x_scales, const float* x_gscale, int M, int64_t ldx,
                 void* y, int y_dtype, int64_t ldy,
                 void* workspace, size_t ws_bytes, void* stream);

/*
 * Per-token (row-wise) activation global scales (R3): the same W4A4 GEMV
 * with x_gscales = M floats, row m of Y scaled by w_gscale * x_gscales[m].  Feed it from
 * nvfp4_quantize_act(..., NVFP4_GSCALE_DYNAMIC_PER_ROW): a row's codes then no longer depend on the other
 * rows of the batch (batch invariance).  Other arguments as for nvfp4_gemv(NVFP4_MODE_W4A4).
 */
int nvfp4_gemv_rowscale(const void* w_blob, const float* w_gscale, int N, int K,
                        const void* x_codes, const uint8_t* x_scales, const float* x_gscales, int M, int64_t ldx,
                        void* y, int y_dtype, int64_t ldy,
                        void* workspace, size_t ws_bytes, void* stream);

/*
 * Fused variant of the two calls above: W4A4 GEMV on BF16 activations with the
 * activation quantizer (dynamic global scale, same bit-exact op sequence as nvfp4_quantize_act) run inside
 * the GEMV kernel -- one launch instead of two.  The result equals nvfp4_quantize_act followed by
 * nvfp4_gemv(NVFP4_MODE_W4A4) on the same inputs (same arithmetic path per M; bit-identical outputs are
 * tested at M = 1).  Every CTA re-quantises the activations it needs, so this pays only at M = 1 (measured:
 * DESIGN.md 6.4); the canonical codes / scales are not materialised.
 *   x_bf16        [device] BF16 bits, row m at x_bf16 + m*ldx elements; ldx >= K, ldx % 8 == 0
 *   x_gscale_out  [device] optional (may be NULL): receives the activation global scale amax/2688
 * Other arguments as for nvfp4_gemv; workspace as returned by nvfp4_gemv_workspace_bytes.
 */
int nvfp4_gemv_fused_quant(const void* w_blob, const float* w_gscale, int N, int K,
                           const void* x_bf16, int M, int64_t ldx, float* x_gscale_out,
                           void* y, int y_dtype, int64_t ldy,
                           void* workspace, size_t ws_bytes, void* stream);

/*
 * Launch-shape override for sweeps (process-wide host state behind a mutex; 0 = use the tuned table):
 *   ksplit = number of K slices (grid.y, 1..64), warps = consumer warps per CTA (1..20),
 *   rows   = row tiles per warp step (1 or 2; 2 exists for the integer W4A4 path, M >= 2),
 *   stages = depth of each warp's bulk-copy ring (1..16),
 *   ctas_per_sm = persistent CTAs per SM (1..3; with >= 2 the CTAs of the NEXT kernel on the stream become
 *            resident and prefetch their first weight cells while this kernel still runs),
 *   balance = 1: every CTA owns units/CTAs whole row-tile units plus an equal share of the leftover units'
 *            cells (data-parallel + stream-K, equal bytes per SM); 2: whole units only (the first CTAs own one
 *            unit more; no partial sums between CTAs).
 * Values the kernels cannot run (shared memory, launch bounds) are clamped; nvfp4_gemv_get_config reports
 * what nvfp4_gemv would use for (mode, M, N, K).  Returns NVFP4_ERR_INVALID_ARG if out of range.
 * nvfp4_set_layout_kparts overrides the K-part count KP of the repacked layout (0 = the default function
 * of (N, K); else a power of two <= 32) for every later size query, repack, unpack and GEMV of this
 * process; the header records KP, so a blob repacked under another value is rejected (NaN outputs), never
 * misread.  nvfp4_get_layout_kparts returns the KP in effect for (N, K).
 */
int nvfp4_gemv_set_config(int ksplit, int warps, int rows, int stages, int ctas_per_sm, int balance);
int nvfp4_gemv_get_config(int mode, int M, int N, int K, int* ksplit, int* warps, int* rows, int* stages,
                          int* ctas_per_sm, int* balance);
int nvfp4_set_layout_kparts(int kparts);
int nvfp4_get_layout_kparts(int N, int K);

/*
 * Quantizer -> GEMV through the GEMV's own activation records (M = 1; the decode step, BASELINE.json configs[1]).
 * nvfp4_gemv stages its activations by loading codes and scales, expanding them and storing them to shared memory after
 * it has waited for the quantizer; here the quantizer writes that shared-memory image itself (per 32 k: the 2 x 16 E2M1
 * values as FP16 -- exact --, then the two block scales as FP32; 80 bytes) and the GEMV fetches its K range with ONE
 * bulk copy.  Same arithmetic, same bits: y equals nvfp4_gemv(NVFP4_MODE_W4A4) on nvfp4_quantize_act's output.
 *   nvfp4_gemv_xrecord_bytes(N, K)  size of the record buffer for a weight of this shape (K padded to the repacked
 *                                   layout's cell; depends on the layout's K parts, so query it per weight shape).  The
 *                                   buffer must be ZERO-FILLED once: the quantizer writes the blocks below K only.
 *   nvfp4_quantize_act_records      x_bf16 [device] BF16 [1, K]; xrec_out [device] the records; gscale / gscale_mode as for
 *                                   nvfp4_quantize_act (NVFP4_GSCALE_DYNAMIC or _STATIC); M must be 1
 *   nvfp4_silu_mul_quantize_records nvfp4_silu_mul_quantize writing the records (down_proj's input from gate_up's BF16 output
 *                                   [1, 2I]; h_bf16_opt as there); M must be 1
 *   nvfp4_gemv_records              w_blob / w_gscale / y / workspace as for nvfp4_gemv (same workspace size); xrec from
 *                                   nvfp4_quantize_act_records for the same K; x_gscale [device] one float; M must be 1
 * Errors as for nvfp4_gemv; M != 1 -> NVFP4_ERR_UNSUPPORTED_SHAPE.
 */
size_t nvfp4_gemv_xrecord_bytes(int N, int K);
int nvfp4_quantize_act_records(const void* x_bf16, int M, int K, int64_t ldx, void* xrec_out, float* gscale, int gscale_mode,
                               void* stream);
int nvfp4_silu_mul_quantize_records(const void* gu_bf16, int M, int I, void* xrec_out, float* gscale, int gscale_mode,
                                    void* h_bf16_opt, void* stream);
int nvfp4_gemv_records(const void* w_blob, const float* w_gscale, int N, int K, const void* xrec, const float* x_gscale, int M,
                       void* y, int y_dtype, int64_t ldy, void* workspace, size_t ws_bytes, void* stream);

/*
 * SiLU*mul + activation quantizer in ONE launch (the producer of down_proj's input in
 * BASELINE.json configs[4]):  h[m,j] = RN_bf16(silu(gu[m,j]) * gu[m,I+j])  (same FP32 expression and BF16 rounding
 * as nvfp4_silu_mul), then the NVFP4 quantizer of nvfp4_quantize_act on h[M,I].  codes / scales / gscale are
 * bit-identical to nvfp4_silu_mul followed by nvfp4_quantize_act; the BF16 intermediate is not written unless
 * h_bf16_opt is given.
 *   gu_bf16 [device] BF16 [M, 2I], row stride 2I;  I % 16 == 0;  M*I <= 524288 unless gscale_mode is NVFP4_GSCALE_STATIC
 *           (a given scale needs no tensor-wide amax: plain wide grid instead of one thread-block cluster, any size)
 *   codes [device] out uint8 [M, I/2];  scales [device] out uint8 [M, I/16];  gscale as for nvfp4_quantize_act
 *   h_bf16_opt [device] optional (may be NULL): BF16 [M, I] copy of the intermediate
 */
int nvfp4_silu_mul_quantize(const void* gu_bf16, int M, int I, uint8_t* codes, uint8_t* scales, float* gscale,
                            int gscale_mode, void* h_bf16_opt, void* stream);

/*
 * Glue of the decode chain (step a8, BASELINE.json configs[4]; not part of the paper's kernel):
 *   h[m,j] = silu(gu[m,j]) * gu[m,I+j],  gu BF16 [M,2I] (row stride 2I), h BF16 [M,I];  I % 8 == 0.
 */
int nvfp4_silu_mul(const void* gu_bf16, int M, int I, void* h_bf16, void* stream);

/*
 * The ReSET sampler step (Sec. 4 :107-139, the paper's titular method): for each of B
 * sequences, one decoding position in ONE launch --
 *   H_t = entropy of softmax(z_t) (nats, :54)  ->  H_bar (running global mean) and H_step (hybrid step-entropy
 *   estimator HSE, Eq. 3 :134: mean of the min(w, t+1) most recent H_i while t - t0 < w, else the mean over the
 *   current step)  ->  tau_t = tau0 if H_step <= H_bar else H_step (SAT, Eq. 2 :113)  ->  T_t = t_low if H_t < tau_t
 *   else t_high (Eq. 1 :90)  ->  top-p sample from softmax(z_t / T_t): the kept set is every token whose strictly more
 *   probable mass is < top_p, the draw is the exponential race argmax z_v/T_t - log(-log u_v) with u_v from
 *   Philox4x32-10 (counter (v, t, 0, 0), key = seed), u = ((x0 >> 9) + 0.5) * 2^-23, ties to the lowest index
 *   ->  if the sampled token is `delimiter_token` ("\n\n", :367) the next step starts at t + 1.
 *   logits [device] F32 or BF16 (NVFP4_DTYPE_*), row b at logits + b*ld elements; V <= 163840, ld >= V
 *   state  [device] B * reset_sampler_state_bytes() bytes, 8-byte aligned, ZERO-FILLED before the first token of a
 *          sequence; read and updated by every call (ring of the last 32 entropies, sums, t, t0)
 *   w in 1..32 (paper: 32, :139);  tau0 per model (Table 8 :414-423);  t_low / t_high / top_p as in :139, :412
 *   token_out [device] int32 [B];  diag_out [device] optional float [B][8]: H_t, H_step, H_bar, tau_t, T_t,
 *          size of the kept set, t + 1, t0 after the step
 * Asynchronous on `stream`, graph capturable, deterministic (fixed-order reductions); one thread-block cluster of
 * 8 CTAs per sequence keeps the vocabulary in registers (the logits are read once).
 */
size_t reset_sampler_state_bytes(void);
int reset_sampler_step(const void* logits, int logits_dtype, int B, int V, int64_t ld, void* state,
                       float tau0, float t_low, float t_high, float top_p, int w, int delimiter_token,
                       unsigned long long seed, int* token_out, float* diag_out, void* stream);

/*
 * Tensor-core NVFP4 GEMM (App. C.3 :526-532, Table 16 :560-575: the paper dispatches
 * large M to a tensor-core GEMM).  Y[M,N] = X[M,K] . W[N,K]^T, both operands NVFP4, on tcgen05 block-scaled MMAs
 * (kind::mxf4nvf4, scale_vec::4X: E2M1 codes and E4M3 block scales go to the tensor core as they are, FP32
 * accumulation in tensor memory).  The weight tile is the MMA's A operand (128 weight rows) and the tokens are its N
 * dimension, so W is streamed from HBM once per 128 tokens for ANY M >= 1 (M <= 128: exactly once).
 *
 *   nvfp4_gemm_repacked_bytes   size of the tensor-core blob for (N, K); 0 if the shape is unsupported
 *                               (requires K % 256 == 0, K >= 256, N >= 1).  Same 0.5625 B per weight as the GEMV blob,
 *                               rows padded to a multiple of 128.
 *   nvfp4_gemm_repack_weight    canonical codes [N,K/2] + scales [N,K/16] (device) -> blob (device, 128-byte aligned
 *                               recommended, 16 required): a pure byte permutation into the shared-memory image of
 *                               the MMA operands (8-row x 16-byte core matrices; scale chunks in tcgen05.cp order)
 *                               behind a versioned 128-byte header.  Offline, once.  nvfp4_gemm_unpack_weight is its
 *                               exact inverse.  The blob is NOT interchangeable with nvfp4_repack_weight's: the GEMM
 *                               writes NaN outputs when handed a blob whose header does not match (N, K).
 *   nvfp4_gemm                  x_codes [M, K/2] (row stride ldx bytes, ldx % 16 == 0), x_scales [M, K/16] contiguous,
 *                               x_gscale one device float (gscale_per_row = 0) or M floats (= 1); y F32 or BF16
 *                               [M, N] (row stride ldy elements).  Launches a small activation re-layout kernel and
 *                               the GEMM (per 128-token chunk) on `stream`; graph capturable, deterministic
 *                               (fixed-order stream-K fix-up), programmatic dependent launch.
 *                               workspace >= nvfp4_gemm_workspace_bytes(M, N, K), 16-byte aligned, zero-filled once
 *                               before first use (the kernel leaves its counters zero).
 * Acceptance as for nvfp4_gemv: |y - y_ref| <= 1e-3 * sum_k|w_k x_k| + 1e-6.
 */
size_t nvfp4_gemm_repacked_bytes(int N, int K);
int nvfp4_gemm_repack_weight(const uint8_t* codes, const uint8_t* scales, int N, int K, void* blob_out, void* stream);
int nvfp4_gemm_unpack_weight(const void* blob, int N, int K, uint8_t* codes, uint8_t* scales, void* stream);
size_t nvfp4_gemm_workspace_bytes(int M, int N, int K);
int nvfp4_gemm(const void* w_blob_tc, const float* w_gscale, int N, int K,
               const void* x_codes, const uint8_t* x_scales, const float* x_gscale, int gscale_per_row, int M, int64_t ldx,
               void* y, int y_dtype, int64_t ldy,
               void* workspace, size_t ws_bytes, void* stream);

/*
 * The same GEMM fed without the re-layout kernel (the decode chain's form: quantizer -> GEMM, two launches per
 * projection like the GEMV path).  The activations of M <= 128 tokens live in the GEMM's own record layout
 * ("packed": per 256 k one record of MT*128 code bytes in 8-token x 16-byte core matrices followed by four 512-byte
 * scale chunks, MT = 8, 16, 32, 64 or 128 >= M), nvfp4_gemm_packed_act_bytes(M, K) bytes, 16-byte aligned; the buffer
 * need not be initialised (columns of tokens >= M are computed and never stored).
 *   nvfp4_gemm_pack_act             canonical codes / scales -> packed
 *   nvfp4_quantize_act_packed       nvfp4_quantize_act writing the packed layout directly: the same binary32 sequence,
 *                                   so pack_act(quantize_act(x)) == quantize_act_packed(x) byte for byte.  M <= 128 for
 *                                   NVFP4_GSCALE_DYNAMIC / _STATIC, M <= 8 for _DYNAMIC_PER_ROW.
 *   nvfp4_silu_mul_quantize_packed  nvfp4_silu_mul_quantize writing the packed layout (M * I <= 524288 unless _STATIC)
 *   nvfp4_gemm_packed               the GEMM on packed activations; workspace >= nvfp4_gemm_packed_workspace_bytes,
 *                                   zero-filled once; other arguments as for nvfp4_gemm
 *   nvfp4_gemm_set_config           tuning knobs (0 = table), process-wide like nvfp4_gemv_set_config: depth of the
 *                                   kernel's shared-memory ring of weight stages (2..16, clamped to what fits) and
 *                                   the number of persistent CTAs the stage list is cut into (clamped to 148)
 */
int nvfp4_gemm_set_config(int stages, int ctas);
size_t nvfp4_gemm_packed_act_bytes(int M, int K);
int nvfp4_gemm_pack_act(const void* x_codes, const uint8_t* x_scales, int M, int K, int64_t ldx, void* xpack_out, void* stream);
int nvfp4_quantize_act_packed(const void* x_bf16, int M, int K, int64_t ldx, void* xpack_out, float* gscale, int gscale_mode,
                              void* stream);
int nvfp4_silu_mul_quantize_packed(const void* gu_bf16, int M, int I, void* xpack_out, float* gscale, int gscale_mode,
                                   void* h_bf16_opt, void* stream);
size_t nvfp4_gemm_packed_workspace_bytes(int M, int N, int K);
int nvfp4_gemm_packed(const void* w_blob_tc, const float* w_gscale, int N, int K, const void* xpack, const float* x_gscale,
                      int gscale_per_row, int M, void* y, int y_dtype, int64_t ldy, void* workspace, size_t ws_bytes,
                      void* stream);

/*
 * nvfp4_gemv for callers that cannot allocate device memory (CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): same arguments and results as nvfp4_gemv, but the scratch (arrival counters + split partials)
 * is a built-in array of NVFP4_NOALLOC_SCRATCH_BYTES bytes of device memory that every GPU loading the library holds
 * until the process exits.  The call allocates nothing (no cudaMalloc / cudaFree): it clears the bytes it is going to
 * use on `stream`, then launches the same kernel as nvfp4_gemv on that array.
 *   - shapes whose workspace (nvfp4_gemv_workspace_bytes(M, N, K)) exceeds NVFP4_NOALLOC_SCRATCH_BYTES return
 *     NVFP4_ERR_UNSUPPORTED_SHAPE (text in nvfp4_last_cuda_error()); 4 MiB covers every Qwen3-8B/14B/32B projection at
 *     M <= 8 (largest: gate_up 51200 x 5120, M = 8: 3.3 MB), not a 151936-row output head at M = 8
 *   - EVERY call on a device shares the one array: calls that overlap on the GPU (different streams) race; issue them
 *     on one stream or order them with events
 *   - the first call on each device looks up the array's device address (cudaGetSymbolAddress, which may load the
 *     module): make it outside stream capture
 */
#define NVFP4_NOALLOC_SCRATCH_BYTES (4u << 20)
int nvfp4_gemv_noalloc(int mode, const void* w_blob, const float* w_gscale, int N, int K,
                       const void* x, const uint8_t* x_scales, const float* x_gscale, int M, int64_t ldx,
                       void* y, int y_dtype, int64_t ldy, void* stream);

/*
 * nvfp4_gemm_packed with the NEXT projection's activation quantizer fused into its epilogue (SURVEY.md 8(f) item 1:
 * "quantize fused into the previous kernel's epilogue when the output tile holds whole 16-blocks and a static global
 * scale is used"; the paper's deployed flow uses static, calibrated activation scales).  The first
 * n_quant output columns (n_quant % 256 == 0, <= N) are rounded to BF16 and quantised with the STATIC global scale
 * *out_gscale (device float, read) by the same binary32 sequence as nvfp4_quantize_act, and written as packed
 * activation records for a following nvfp4_gemm_packed with K = n_quant and the same M:
 *   xpack_out == nvfp4_gemm_pack_act(nvfp4_quantize_act(STATIC, RN_bf16(y)[:, :n_quant]))  byte for byte (tokens < M).
 * xpack_out: nvfp4_gemm_packed_act_bytes(M, n_quant) bytes, 16-byte aligned.  y_opt may be NULL (no BF16 / FP32 output is
 * written then: the quantised records are the only result).  Values beyond the static scale's range saturate
 * (block scale clamps at 448, codes at +-6), as in nvfp4_quantize_act(STATIC).  Other arguments as for nvfp4_gemm_packed.
 */
int nvfp4_gemm_packed_quant_out(const void* w_blob_tc, const float* w_gscale, int N, int K, const void* xpack,
                                const float* x_gscale, int gscale_per_row, int M, void* y_opt, int y_dtype, int64_t ldy,
                                void* xpack_out, const float* out_gscale, int n_quant, void* workspace, size_t ws_bytes,
                                void* stream);

/*
 * W4A16 on the tensor cores (BASELINE.json configs[3]: NVFP4 weights, BF16 activations consumed directly, FP32
 * accumulation), any M >= 1:  Y[M,N] = X_bf16[M,K] . W[N,K]^T  with W in the tensor-core blob of nvfp4_gemm_repack_weight.
 * The weights are expanded to FP16 in shared memory ONCE per 128-row x 256-k stage (exact: E2M1 value x E4M3 block scale),
 * whatever M is, and multiplied with the BF16 activations by tcgen05.mma kind::f16 (FP32 accumulator in tensor memory);
 * the global weight scale is applied in the epilogue.  Same result as nvfp4_gemv(NVFP4_MODE_W4A16) up to FP32 summation
 * order; acceptance |y - y_ref| <= 1e-3 * sum_k|w_k x_k| + 1e-6.  Deterministic (fixed-order split-K fix-up).
 *   x_bf16 [M, K] BF16, row stride ldx elements (ldx % 8 == 0, 16-byte aligned rows); K % 256 == 0
 *   workspace >= nvfp4_gemm_w4a16_workspace_bytes(M, N, K), 16-byte aligned, zero-filled once (counters are left zero)
 * Launches a small re-layout kernel for the activations and the GEMM per chunk of 32 tokens (W is streamed once per chunk).
 */
size_t nvfp4_gemm_w4a16_workspace_bytes(int M, int N, int K);
int nvfp4_gemm_w4a16(const void* w_blob_tc, const float* w_gscale, int N, int K, const void* x_bf16, int M, int64_t ldx,
                     void* y, int y_dtype, int64_t ldy, void* workspace, size_t ws_bytes, void* stream);

/*
 * The gate_up projection with SiLU * mul AND the down projection's STATIC-scale quantizer in its epilogue (SURVEY.md
 * 8(f) item 1, step a8 fused): no BF16 gate_up output, no separate SiLU * mul / quantizer launch.
 *   nvfp4_gemm_repack_weight_gate_up   the tensor-core blob of the fused gate_up weight [N = 2I, K] (gate = rows [0, I),
 *                                      up = rows [I, 2I), R11) with the rows INTERLEAVED per 128-row tile: 64
 *                                      gate rows followed by the 64 matching up rows, so one tile owns both factors.
 *                                      N % 128 == 0; same size as nvfp4_gemm_repacked_bytes(N, K); the header records
 *                                      the interleaving (a plain nvfp4_gemm on this blob, or this call on a plain blob,
 *                                      writes NaN).  nvfp4_gemm_unpack_weight_gate_up is its exact inverse.
 *   nvfp4_gemm_packed_silu_quant_out   h[m, j] = RN_bf16(silu(RN_bf16(gate[m, j])) * RN_bf16(up[m, j])), j < I = N/2 (the
 *                                      arithmetic of nvfp4_silu_mul on the BF16 GEMM output), quantised with the STATIC
 *                                      global scale *out_gscale into packed activation records for a following
 *                                      nvfp4_gemm_packed with K = I (I % 256 == 0): byte-identical to
 *                                      nvfp4_silu_mul_quantize_packed(STATIC) applied to the plain GEMM's BF16 output.
 *                                      h_opt (optional, [M, I], row stride ldh) receives h.  Other arguments as for
 *                                      nvfp4_gemm_packed_quant_out.
 */
int nvfp4_gemm_repack_weight_gate_up(const uint8_t* codes, const uint8_t* scales, int N, int K, void* blob_out, void* stream);
int nvfp4_gemm_unpack_weight_gate_up(const void* blob, int N, int K, uint8_t* codes, uint8_t* scales, void* stream);
int nvfp4_gemm_packed_silu_quant_out(const void* w_blob_gate_up, const float* w_gscale, int N, int K, const void* xpack,
                                     const float* x_gscale, int gscale_per_row, int M, void* h_opt, int h_dtype, int64_t ldh,
                                     void* xpack_out, const float* out_gscale, void* workspace, size_t ws_bytes, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* NVFP4_B200_H_ */
