/*
 * hq.h — C ABI of libhq.so: HyperQuant's inference-time hot path on one NVIDIA B200 (sm_100a).
 *
 * Citations are /root/reference/PAPER.md line numbers (arxiv/paper_2606_23406); "FORMAT" is
 * docs/FORMAT.md (bitstream layout and the canonical fp32 arithmetic); "G<n>" are the readings of
 * the paper listed in DESIGN.md §3.
 *
 * Conventions
 *  - Every pointer says "dev" (CUDA device memory on the context's device) or "host".
 *  - Caller-owned buffers are never retained past the call; work is enqueued on `stream`
 *    (a cudaStream_t passed as void*) and is asynchronous unless the call says it synchronizes.
 *  - Handles (hq_ctx, hq_weight, hq_kv) own only memory obtained from the hq_allocator given to
 *    hq_create; the library never calls cudaMalloc itself.
 *  - Every call returns an hq_status; nothing throws or aborts.  hq_last_error() gives the text.
 *  - There is no CPU fallback: a device that is not compute capability 10.x gives HQ_ERR_UNSUPPORTED.
 *  - A context serializes its work: hq_linear / hq_linear_group share one context-owned workspace (activation
 *    operand tiles, split-K partial sums, arrival counters), so calls on one hq_ctx must be issued to one stream at a
 *    time.  The workspace grows on demand (which synchronizes the device): call each shape once eagerly before
 *    capturing the calls into a CUDA graph.  Results are deterministic (fixed summation order).
 */
#ifndef HQ_H_
#define HQ_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    HQ_OK = 0,
    HQ_ERR_INVALID_ARG = 1, /* NULL pointer, bad enum, bad handle */
    HQ_ERR_SHAPE = 2,       /* n_in not a multiple of n_tile, head_dim not a supported tile, batch too large ... */
    HQ_ERR_UNSUPPORTED = 3, /* not an sm_100 device, rotation qjl, ... */
    HQ_ERR_ALLOC = 4,       /* the caller's allocator returned NULL */
    HQ_ERR_CUDA = 5,        /* a CUDA runtime call failed; text in hq_last_error */
    HQ_ERR_FORMAT = 6       /* a tile's U-section exceeds the container's bound (FORMAT §4, §5); a KV cache whose U stream
                               ran out of capacity (sticky: every later call on that cache returns it); a blob that fails
                               hq_weight_import's layout checks */
} hq_status;

typedef enum { HQ_Z = 1, HQ_A2 = 2, HQ_D4 = 4, HQ_E8 = 8 } hq_lattice;     /* §3.2, §4.5; value = dimension */
typedef enum { HQ_F32 = 0, HQ_BF16 = 1 } hq_dtype;
typedef enum { HQ_ROT_NONE = 0, HQ_ROT_SIGNS = 1, HQ_ROT_QJL = 2 } hq_rotation; /* §4.2, §3.4; QJL = a dense Haar matrix given in hq_kv_config.qjl_dev */

/* Device-memory allocator supplied by the caller (the Python binding backs it with torch). */
typedef struct {
    void* (*alloc)(void* user, size_t bytes); /* returns a dev pointer aligned to >= 256 bytes, or NULL */
    void (*free)(void* user, void* dev_ptr);
    void* user;
} hq_allocator;

/* The codec operating point (Table 4). */
typedef struct {
    int32_t lattice;   /* hq_lattice */
    int32_t n_tile;    /* RHT tile = normalization tile: 64, 128 or 256 (§4.1, §7.2) */
    float snr_db;      /* target SNR; alpha = sqrt(10^(snr/10) * G V^(2/N)), eq.(9) */
    int32_t rice_k[2]; /* Rice parameter per symbol class (FORMAT §3); -1 = auto (argmin of total bits) */
    uint64_t seed;     /* seeds the RHT signs D (and, for KV, the rotation S and the dither) — FORMAT §1 */
} hq_codec_config;

typedef struct hq_ctx hq_ctx;
typedef struct hq_weight hq_weight;
typedef struct hq_kv hq_kv;

/* ---- context ------------------------------------------------------------------------------- */
hq_status hq_create(hq_ctx** out, const hq_allocator* alloc, int cuda_device);
void hq_destroy(hq_ctx* ctx);
const char* hq_last_error(const hq_ctx* ctx); /* never NULL; valid until the next call on ctx */

/* Measurement aid: when enabled, hq_linear and hq_attend bracket their dominant kernel (the fused
 * decode+MMA kernel / the split attention kernel) with CUDA events on the caller's stream.
 * hq_profile_read synchronizes those events, returns their summed duration and count, and clears them. */
hq_status hq_profile_enable(hq_ctx* ctx, int32_t on);
hq_status hq_profile_read(hq_ctx* ctx, double* total_ms, int64_t* launches);

/* Measurement aid: the issue-slot ceiling of the E8 Rice decode on this device.  Every warp of a
 * full grid (one CTA per SM, the fused kernel's CTA shape) keeps one sub-group of `w` in registers and runs the fused
 * kernel's decode phases on it `reps` times - no global loads in the loop, no MMA, no split-K.  Returns decoded
 * scalars per second (CUDA events on `stream`, synchronizes).  w must be E8 / tile 128 / k <= 3 (HQ_ERR_UNSUPPORTED). */
hq_status hq_measure_decode_ceiling(hq_ctx* ctx, const hq_weight* w, int32_t reps, void* stream, double* scalars_per_s);

/* alpha of eq.(9) L871 for (lattice, snr_db), as the library computes it (host, double). */
double hq_alpha(int32_t lattice, double snr_db);

/*
 * Calibration lookup (§5.4, App. B.1, reading G17): the SNR at which `lattice` realizes
 * `target_bps` payload bits per scalar (Rice code at the best k, no metadata) on iid Gaussian tiles of 128, by linear
 * interpolation in a cached table b(SNR) (1e5 tiles, seed 42, 0.25 dB grid over 5..35 dB).  The table is data, committed
 * as csrc/hq_calib_table.inc and written by oracle/make_calib_table.py (which calls only oracle/); the paper's printed
 * anchors pin it (tests/test_abi.py).  Pure host function: ctx may be NULL.  target_bps outside the table's range ->
 * HQ_ERR_INVALID_ARG.  rice_k_out (may be NULL) receives the table's best k-set at the grid point below the answer.
 */
hq_status hq_snr_for_bps(const hq_ctx* ctx, int32_t lattice, double target_bps, float* snr_db_out, int32_t* rice_k_out);

/* ---- weights: encode (§5.1; SURVEY §8(a) B1,B3,B5-B7) ------------------------------ */
/*
 * Quantize W [m_out, n_in] (row-major, leading dimension ld elements, dev, F32 or BF16): per
 * (row, column tile) RHT -> l2-normalize to radius alpha*sqrt(n) (norm stored as fp16) -> nearest
 * lattice point -> strip + zig-zag -> Rice code, packed into the FORMAT §5 container with per-tile
 * lengths and per-group offsets from a device prefix sum.  Synchronizes `stream` (the container
 * size is data dependent).  *out owns its device memory; free with hq_weight_free.
 */
hq_status hq_encode_weights(hq_ctx* ctx, const void* W_dev, int32_t dtype, int64_t m_out, int64_t n_in,
                            int64_t ld, const hq_codec_config* cfg, void* stream, hq_weight** out);
void hq_weight_free(hq_ctx* ctx, hq_weight* w);

typedef struct {
    int64_t m_out, n_in;
    int32_t lattice, n_tile, rice_k[2];
    float snr_db;
    double alpha;
    uint64_t seed;
    int64_t payload_bits;  /* sum over tiles of Rbits + ulen = the Rice code's length */
    int64_t norm_bits;     /* 16 per tile (L500) */
    int64_t length_bits;   /* 16 per tile (G12) */
    int64_t blob_bytes;    /* whole container incl. padding */
    int64_t n_groups;      /* sub-groups of 32 rows x one tile: 4 * ceil(m_out/128) * n_in/n_tile (FORMAT §5) */
    int64_t clamp_count;   /* quantizer inputs limited by the INT8 pre-clamp (G8, L236) */
} hq_weight_info;
hq_status hq_weight_get_info(const hq_weight* w, hq_weight_info* out);

/* dev pointers into the handle (valid until hq_weight_free): the FORMAT §5 blob and sub_off[n_groups+1]. */
hq_status hq_weight_export(const hq_weight* w, const void** blob_dev, const uint32_t** group_off_dev);

/* Rate and range statistics of an encoded weight (SURVEY §5 "metrics": Figs 10-11 report realized bps and overflow).
 * Host values recorded at encode / import time; no device work. */
typedef struct {
    int64_t payload_bits, norm_bits, length_bits;  /* as hq_weight_info */
    int64_t offset_bits;                           /* 32 per sub-group (sub_off, FORMAT §5) */
    int64_t padding_bits;                          /* 8 * blob_bytes - payload - norm - length: word / 16-byte alignment */
    int64_t clamp_count;                           /* INT8 pre-clamp events (G8) */
    int64_t n_tiles;                               /* m_out * n_in / n_tile */
    int32_t tile_bits_min, tile_bits_max;          /* Rice code length of the shortest / longest tile (Rbits + ulen) */
    double bits_per_scalar_payload, bits_per_scalar_total; /* total = payload + norm + length */
} hq_stats;
hq_status hq_weight_stats(const hq_weight* w, hq_stats* out);

/*
 * The encoded weight as a host artefact ("store integer codes and per-tile scales", §5.1; SURVEY §5 checkpoint).
 * hq_weight_export_host copies the FORMAT §5 container to caller-owned HOST buffers (blob_host: header.blob_bytes
 * bytes, sub_off_host: header.n_groups + 1 words; pass both NULL to get the header and the sizes only) and
 * synchronizes `stream`.  hq_weight_import rebuilds a handle from them: it checks the header, that sub_off is
 * increasing and ends at blob_bytes / 16, and that every sub-group's size equals what its ulen header implies
 * (HQ_ERR_FORMAT otherwise, nothing is launched on a bad blob), uploads on `stream`, regenerates the RHT signs from
 * the seed.  An imported handle gives bit-identical hq_linear / hq_decode_int8 results.
 */
typedef struct {
    uint32_t magic, version;      /* 'HQW1', 2 */
    int64_t m_out, n_in;
    int32_t lattice, n_tile, rice_k[2];
    float snr_db;
    uint64_t seed;
    int64_t blob_bytes, n_groups;
    int64_t payload_bits, clamp_count;
    int32_t ulen_min, ulen_max;   /* shortest / longest U-section over the present rows, bits */
} hq_weight_header;
hq_status hq_weight_export_host(hq_ctx* ctx, const hq_weight* w, hq_weight_header* header, void* blob_host,
                                uint32_t* sub_off_host, void* stream);
hq_status hq_weight_import(hq_ctx* ctx, const hq_weight_header* header, const void* blob_host,
                           const uint32_t* sub_off_host, void* stream, hq_weight** out);

/* Parity / debug: the INT8 lattice points c [m_out, n_in] (row-major, dev) and fp16 norms
 * [m_out, n_in/n_tile] (dev, may be NULL) decoded from the container (O2; §4.5-4.7 inverse). */
hq_status hq_decode_int8(hq_ctx* ctx, const hq_weight* w, int8_t* codes_dev, uint16_t* norms_dev, void* stream);

/* ---- activations (FORMAT R1, R7) ---------------------------------------- */
/*
 * x [batch, n_in] (dev, leading dimension ldx) -> per (row, tile): u = RHT(x) with the weight's sign
 * vector (§3.1 eq.(1)), amax-scaled INT8 cast q = rint(u*127/amax), s_x = amax/127.
 * q [batch, n_in] int8, s_x [batch, n_in/n_tile] f32, u (optional, may be NULL) [batch, n_in] f32.
 */
hq_status hq_act_quant(hq_ctx* ctx, const hq_weight* w, const void* x_dev, int32_t dtype, int64_t batch,
                       int64_t ldx, int8_t* q_dev, float* s_x_dev, float* u_dev_or_null, void* stream);

/* ---- linear: fused Rice decode -> INT8 points -> tcgen05 INT8 MMA ------- */
/*
 * y[b, r] = sum_kt (rho[r,kt] / (alpha sqrt(n))) * s_x[b,kt] * acc[kt,b,r],
 * acc[kt,b,r] = sum_{i in tile kt} c[r,i] * q[b,i]  (INT32, tcgen05.mma kind::i8).
 * x [batch, n_in] dev (ldx), y [batch, m_out] bf16 dev (ldy).  Optional debug outputs (dev, may be
 * NULL): y_f32 [batch, m_out] (the value before the bf16 cast), acc_i32 [n_kt, batch, m_out].
 * Where the decoded weights live (north_star (d)):
 *   batch 1, E8 / tile 128 / k <= 3 (k_gemv_e8): registers -> tensor memory (tcgen05.st) -> MMA A operand; never in
 *     shared or global memory.  The kernel also does the activation RHT + INT8 cast itself: one launch per call.
 *   batch 2..63 (k_linear_e8) and every other lattice / tile (k_linear_generic): a shared-memory operand tile.
 *   batch >= 64, E8 at tile 128 or 256 (large-M path): decoded ONCE per call into a scratch copy in operand layout in
 *     the context's workspace (global memory, L2 resident: 69 MB for a 16384 x 4096 weight), streamed by TMA into a
 *     warp-specialised tcgen05 GEMM.  This is the one place decoded weights leave the SM (DESIGN.md §6.4 says why).
 * Any batch >= 1.  Limits of the fused kernels (HQ_ERR_SHAPE beyond them): n_in / n_tile < 4096, m_out < 8388608,
 * ceil(m_out / 128) * (n_in / n_tile) < 2^31.
 */
hq_status hq_linear(hq_ctx* ctx, const hq_weight* w, const void* x_dev, int32_t dtype, int64_t batch,
                    int64_t ldx, void* y_bf16_dev, int64_t ldy, float* y_f32_dev_or_null,
                    int32_t* acc_i32_dev_or_null, void* stream);

/*
 * hq_linear with the MMA cast of §4.8 chosen by the caller ("cast at the matmul boundary to FP8-E4M3/INT8";
 * §6.3 L433-448 compares the two).  HQ_CAST_INT8 is hq_linear.  HQ_CAST_FP8_E4M3 (docs/FORMAT.md R12): the
 * decoded integer coordinates and the RHT'd activations (per-tile amax -> 448) are rounded to E4M3 and contracted by
 * tcgen05.mma kind::f8f6f4 into an fp32 accumulator; y = sum_kt (rho / (alpha sqrt n)) s_x acc as for INT8.  Built for the
 * compute-bound regime on the large-M pipeline: E8, tile 128 or 256, k <= 3, batch >= 64 - anything else ->
 * HQ_ERR_UNSUPPORTED.  The accumulation order inside the tensor core is the hardware's: y meets the 1e-3 bar against
 * the reference, it is not bit-reproducible across GPU generations.  NVFP4 / MXFP4 (§6.4) are not built.
 * acc_dev_or_null: parity / debug copy of every RHT tile's accumulator, [n_in / n_tile, batch, m_out]: int32 for
 * HQ_CAST_INT8, float (the fp32 tensor-core accumulator) for HQ_CAST_FP8_E4M3.
 */
typedef enum { HQ_CAST_INT8 = 0, HQ_CAST_FP8_E4M3 = 1 } hq_cast;
hq_status hq_linear_cast(hq_ctx* ctx, const hq_weight* w, const void* x_dev, int32_t dtype, int64_t batch, int64_t ldx,
                         void* y_bf16_dev, int64_t ldy, float* y_f32_dev_or_null, void* acc_dev_or_null, int32_t cast,
                         void* stream);

/*
 * Several weights applied to the SAME x in one fused launch (q/k/v or gate/up of a decoder layer: §5.1 L309 quantizes
 * every nn.Linear separately, the forward shares the input).  ws[i] -> ys_bf16[i] [batch, m_i] (leading dimension
 * ldys[i]).  From 2 activation rows the results are bit-identical to n_w separate hq_linear calls; at batch 1 the K range of
 * a row block is summed in the segments the launch's flat tile partition cuts it into, so grouped and separate calls
 * agree to fp32 rounding (each call is deterministic: same call, same bits).  1 <= n_w <= 4.  Weights that cannot share
 * a launch (different n_in / lattice / tile / Rice k / seed / snr_db, or not on the E8 fast path) are run one by one.
 * ys_f32_or_null: optional array of n_w dev pointers (entries may be NULL) for the fp32 pre-cast outputs.
 */
hq_status hq_linear_group(hq_ctx* ctx, const hq_weight* const* ws, int32_t n_w, const void* x_dev, int32_t dtype,
                          int64_t batch, int64_t ldx, void* const* ys_bf16_dev, const int64_t* ldys,
                          float* const* ys_f32_or_null, void* stream);

/*
 * hq_linear for ONE activation row that allocates nothing: for callers that cannot call cudaMalloc (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid it).  Same kernel and same result as hq_linear at batch 1 on
 * the E8 / tile 128 / k <= 3 path (k_gemv_e8: x [n_in] dev -> y [m_out] bf16 dev and/or y_f32 [m_out] dev, at least one
 * non-NULL); the kernel's scratch (split-K arrival counters and partial sums) lives in a file-scope device array of
 * HQ_LINEAR_STATIC_SCRATCH_BYTES inside the library instead of the allocator-backed workspace.  Every GPU that loads the
 * library holds that array until the process exits.  The call makes no cudaMalloc / cudaFree / allocator call: it
 * enqueues one cudaMemsetAsync (the counters must start at zero; the array keeps the previous call's contents) and one
 * kernel on `stream`.  ALL calls on a device share the array: calls that overlap on the GPU (two streams, two contexts,
 * two threads) race on it - serialize them.  Limits: other lattices / tiles / k > 3 / n_in > 16384 -> HQ_ERR_UNSUPPORTED;
 * a weight whose scratch does not fit -> HQ_ERR_SHAPE, hq_last_error says by how much.  The array holds 32 KiB of
 * counters (16 bytes per 128 rows: m_out <= 262144) and 2 064 384 bytes of partial sums (slots * m_out * 4, slots = the
 * segments the launch's tile partition cuts a row block's K range into, <= n_in / 128 + 1): on a 148-SM device every
 * weight with m_out <= 160 000 fits, whatever its n_in.  The array's device address is taken once per device at hq_create (cudaGetSymbolAddress); if that failed the
 * call returns HQ_ERR_CUDA.
 */
#define HQ_LINEAR_STATIC_SCRATCH_BYTES (2u * 1024u * 1024u)
hq_status hq_linear_static(hq_ctx* ctx, const hq_weight* w, const void* x_dev, int32_t dtype, void* y_bf16_dev,
                           float* y_f32_dev_or_null, void* stream);

/* ---- a decoder layer's decode step: the glue between the linears folded into their kernels ---- */
/*
 * PAPER.md:L212 (§4.1): "the butterfly folds into the preceding LayerNorm"; Table 10's decode shape
 * (L496-511).  At batch 1 the fused kernel (k_gemv_e8) quantizes the activation vector itself, so the element-wise steps
 * that precede a linear run inside its prologue and the residual add inside its epilogue - no kernel of their own, no
 * round trip of the normalised vector through HBM.  Canonical arithmetic: docs/FORMAT.md R8 (RMSNorm), R9 (SiLU.mul),
 * R10 (residual); each fold is bit-identical to a separate kernel that writes its result in bf16.
 *   HQ_FOLD_RMSNORM : x_dev = residual stream h [n_in] bf16, aux_dev = gain g [n_in] bf16:  x_i = bf16((h_i r) g_i),
 *                     r = 1 / sqrt(mean(h^2) + eps).  Every CTA recomputes r from the 2 n_in bytes of h (L2 hits).
 *   HQ_FOLD_SILU_MUL: x_dev = gate a [n_in] bf16, aux_dev = up b [n_in] bf16:  x_i = bf16(silu(a_i) b_i).
 *   residuals_dev   : NULL, or n_w device pointers (entries may be NULL): bf16 [m_i] added to output i before the bf16
 *                     cast (y_f32 then carries the sum).  A residual may alias its output.
 * x_dev and aux_dev must be 8-byte aligned.  Batch 1, bf16, E8 / tile 128 / k <= 3 weights that can share a launch
 * (as hq_linear_group), n_in <= 16384: anything else -> HQ_ERR_UNSUPPORTED (there is no unfused fallback).
 */
typedef enum { HQ_FOLD_NONE = 0, HQ_FOLD_RMSNORM = 1, HQ_FOLD_SILU_MUL = 2 } hq_fold_mode;
typedef struct {
    int32_t mode;                      /* hq_fold_mode */
    float eps;                         /* HQ_FOLD_RMSNORM */
    const void* aux_dev;               /* gain (RMSNORM) or second factor (SILU_MUL); NULL for HQ_FOLD_NONE */
    const void* const* residuals_dev;  /* NULL or n_w pointers */
} hq_fold;
hq_status hq_linear_group_fold(hq_ctx* ctx, const hq_weight* const* ws, int32_t n_w, const void* x_dev,
                               const hq_fold* fold, void* const* ys_bf16_dev, float* const* ys_f32_or_null, void* stream);

/*
 * One decode step (one token) of a Llama-style decoder layer on compressed weights and a compressed KV cache, seven
 * launches in stream order, no host synchronisation, no allocation after the first call at a given shape:
 *   q,k,v = W_{q,k,v} RMSNorm(h; g_attn)      hq_linear_group_fold, RMSNorm in the prologue        (1 launch)
 *   cache <- (k, v)                            hq_kv_append                                         (1 launch)
 *   a = attend(q)                              hq_attend                                            (2 launches)
 *   h2 = h + W_o a                             hq_linear_group_fold, residual in the epilogue       (1 launch)
 *   gate, up = W_{gate,up} RMSNorm(h2; g_mlp)  hq_linear_group_fold, RMSNorm in the prologue        (1 launch)
 *   h_out = h2 + W_down (silu(gate) * up)      hq_linear_group_fold, SiLU.mul prologue + residual   (1 launch)
 * Rotary position embedding is not part of the paper's method and is not applied (the weights are synthetic).
 * h_in, h_out [hidden] bf16 dev (may alias).  scratch_dev: hq_layer_scratch_bytes() bytes, 256-byte aligned, holds q, k, v,
 * a, h2, gate, up (bf16); hq_layer_scratch_view returns their offsets for parity tests.  With a cache created with
 * hq_kv_config.device_position = 1 the call can be captured into ONE CUDA graph after one eager warm-up call (which sizes
 * the library's workspaces) and every replay is the next token; with a host-position cache a captured graph replays the
 * SAME position.
 * Shapes: wq [q_heads d, hidden], wk / wv [kv_heads d, hidden], wo [hidden, q_heads d], wgate / wup [ffn, hidden],
 * wdown [hidden, ffn]; d = the cache's head_dim.  Mismatch -> HQ_ERR_SHAPE.
 */
typedef struct {
    const hq_weight *wq, *wk, *wv, *wo, *wgate, *wup, *wdown;
    const void* g_attn_dev;   /* [hidden] bf16 */
    const void* g_mlp_dev;    /* [hidden] bf16 */
    float eps;
    hq_kv* kv;
    int32_t q_heads;
} hq_layer;
typedef struct { size_t q, k, v, a, h2, gate, up, total; } hq_layer_scratch;   /* byte offsets into scratch_dev */
hq_status hq_layer_scratch_view(const hq_layer* layer, hq_layer_scratch* out);
hq_status hq_layer_decode(hq_ctx* ctx, const hq_layer* layer, const void* h_in_dev, void* h_out_dev, void* scratch_dev,
                          size_t scratch_bytes, void* stream);

/* bytes of scratch hq_linear needs for this (weight, batch); it is taken from the ctx allocator and cached. */
hq_status hq_linear_workspace_bytes(const hq_weight* w, int64_t batch, size_t* bytes);

/* ---- KV cache (§5.2, attend C1-C5) ------------------------------ */
typedef struct {
    int32_t kv_heads, head_dim; /* head_dim is the RHT tile (L639): 64, 128 or 256 */
    int64_t max_tokens;
    hq_codec_config codec;      /* n_tile must equal head_dim; rice_k must be given (>= 0) */
    int32_t rotation;           /* hq_rotation: S applied after the RHT (§4.2, G14) */
    int32_t dither;             /* 1: subtractive dither U ~ Unif(V(Lambda)) per token (§4.4, A.6 L843) */
    int32_t window;             /* exact bf16 residual window, tokens (§6.7.2); 0 <= window <= head_dim */
    int64_t una_capacity_bits;  /* capacity of each (role, head) U stream; 0 = auto: max_tokens * head_dim *
                                   max(4, 1.3 * (1 + (0.8 alpha + 0.5) / 2^k)) bits (E|zz| ~ 0.8 alpha on a normalized vector).
                                   A vector that does not fit is NOT written; the cache turns sticky HQ_ERR_FORMAT. */
    const float* qjl_dev;       /* HQ_ROT_QJL (§3.4 L184-188 eq.(2); the paper's default KV rotation at >= 2 bps, Table 4):
                                   the orthogonal matrix S [head_dim][head_dim], fp32 row-major, DEVICE memory, drawn
                                   Haar-uniform once per layer by the caller (the library draws no matrices; orthogonality is
                                   not checked).  Copied at hq_kv_create: the caller may free it afterwards.  Encode applies
                                   u' = S u after the RHT (FORMAT R11: canonical fma accumulation in column order, so the
                                   codes are reproducible bit for bit); hq_attend rotates the query by S and un-rotates the code-domain sum by S^T, one
                                   head_dim x head_dim matvec per QUERY head instead of the paper's O(T D^2) per layer (L502).
                                   Must be NULL for the other rotations. */
    int32_t device_position;    /* 1: the number of held tokens lives in DEVICE memory.  A single-token hq_kv_append reads
                                   its token index there and advances it, hq_attend reads the context length there and is
                                   launched over a split count fixed by max_tokens - so a CUDA graph that captured
                                   hq_kv_append(1 token) / hq_attend / hq_layer_decode stays correct on every replay (each
                                   replay is the next token).  A replayed append past max_tokens writes nothing and turns the
                                   cache sticky HQ_ERR_FORMAT.  The host's own count is refreshed from the device (one
                                   blocking 4-byte copy) by multi-token hq_kv_append, hq_kv_export, hq_kv_decode_int8 and
                                   hq_kv_sync_position.  0: the count is host state (a captured graph replays one position). */
} hq_kv_config;

hq_status hq_kv_create(hq_ctx* ctx, const hq_kv_config* cfg, hq_kv** out);
void hq_kv_free(hq_ctx* ctx, hq_kv* kv);

/* Append n_tok tokens: k, v [n_tok, kv_heads, head_dim] bf16 dev.  Encodes every vector (RHT ->
 * rotate -> normalize -> dither -> nearest point -> strip -> Rice) into the FORMAT §6 container and
 * writes the bf16 ring.  Token indices continue from the tokens already held. */
hq_status hq_kv_append(hq_ctx* ctx, hq_kv* kv, const void* k_dev, const void* v_dev, int64_t n_tok, void* stream);

/* device_position caches only: wait for the stream work issued so far and read the held-token count back (returned in
 * *n_tokens_out, may be NULL).  A no-op that returns the host count for other caches. */
hq_status hq_kv_sync_position(hq_ctx* ctx, hq_kv* kv, int64_t* n_tokens_out);

/* One decode step of attention (L178) for q [q_heads, head_dim] bf16 dev over all held tokens:
 * tokens [0, T-window) from the bitstream (decoded in the code domain), [T-window, T) from the ring.
 * out [q_heads, head_dim] bf16 dev; out_f32 optional. q_heads must be a multiple of kv_heads, q_heads <= 64,
 * q_heads / kv_heads <= 8 (HQ_ERR_SHAPE otherwise). */
hq_status hq_attend(hq_ctx* ctx, const hq_kv* kv, const void* q_dev, int32_t q_heads, void* out_bf16_dev,
                    float* out_f32_dev_or_null, void* stream);

typedef struct {
    int64_t n_tokens;
    int64_t rbits;               /* R-section bits per vector */
    const uint32_t* rem_dev;     /* [2][kv_heads][rem_words]   */
    const uint32_t* una_dev;     /* [2][kv_heads][una_words]   */
    const uint16_t* ulen_dev;    /* [2][kv_heads][max_tokens]  */
    const uint16_t* norm_dev;    /* [2][kv_heads][max_tokens]  */
    const uint32_t* blk_off_dev; /* [2][kv_heads][max_tokens/128 + 1] */
    const uint32_t* upos_dev;    /* [2][kv_heads] current U-stream length in bits */
    int64_t rem_words, una_words;
    int64_t clamp_count;
} hq_kv_view;
/* Synchronizes the device. Pointers stay valid until hq_kv_free. */
hq_status hq_kv_export(hq_ctx* ctx, const hq_kv* kv, hq_kv_view* out);

/* Parity / debug: decode tokens [t0, t0+n) of one role to INT8 codes [n, kv_heads, head_dim] (dev). */
hq_status hq_kv_decode_int8(hq_ctx* ctx, const hq_kv* kv, int32_t role, int64_t t0, int64_t n,
                            int8_t* codes_dev, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* HQ_H_ */
