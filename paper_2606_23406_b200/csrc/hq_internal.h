// hq_internal.h — host-side declarations shared by the translation units of libhq.so (not installed).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/hq.h"

struct hq_ctx {
    hq_allocator alloc;
    int device;
    int sm_count;
    std::string err;
    // cached scratch for hq_linear (activation operand, split-K partials)
    void* ws = nullptr;
    size_t ws_bytes = 0;
    uint32_t* e8_lut = nullptr;  // dev: phase-1 table of the E8 fast decoder (hq_e8_decode.cuh)
    // dev: split-arrival counters of the E8 kernel's in-kernel split-K reduction; all zero whenever no hq_linear is
    // in flight (the last arrival resets its counter), cleared when (re)allocated
    unsigned int* e8_cnt = nullptr;
    size_t e8_cnt_bytes = 0;
    // optional kernel timing (hq_profile_*): event pairs around the dominant kernel of each call
    bool prof = false;
    std::vector<cudaEvent_t> prof_ev;
    // fork / join inside one call (large-M path: the weight decode runs beside the activation cast): a side stream and
    // two timing-free events; everything stays ordered with respect to the caller's stream (graph-capturable)
    cudaStream_t side = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    // device address of the library's file-scope scratch array on this device (hq_linear_static), from
    // cudaGetSymbolAddress at hq_create; null if that failed
    uint8_t* static_scratch = nullptr;
};

struct hq_weight {
    hq_ctx* ctx;
    int64_t m, n_in;
    int lattice, n, k0, k1;
    float snr_db;
    double alpha;
    float A;  // (float)(alpha*sqrt(n))
    uint64_t seed;
    int64_t n_kt, n_rb, G;
    int rbits;
    uint8_t* blob;        // dev
    uint32_t* group_off;  // dev [4G+1]  sub-group offsets (FORMAT §5)
    int8_t* dsign;        // dev [n_in]  RHT signs (+1/-1)
    int64_t blob_bytes, payload_bits, clamp_count;
    uint32_t max_group16;  // largest sub-group size in 16-byte units
    uint32_t min_ulen;     // shortest U-section (bits) over the present rows of all tiles
    uint32_t max_ulen;     // longest
};

struct hq_kv {
    hq_ctx* ctx;
    hq_kv_config cfg;
    int k0, k1, rbits;
    double alpha;
    float A;
    int64_t n_tokens;  // host-side count
    int64_t rem_words, una_words, n_blk;
    uint32_t* rem;      // [2][H][rem_words]
    uint32_t* una;      // [2][H][una_words]
    uint16_t* ulen;     // [2][H][max_tokens]
    uint16_t* norm;     // [2][H][max_tokens]
    uint32_t* blk_off;  // [2][H][n_blk+1]
    uint32_t* upos;     // [2][H]
    __nv_bfloat16* ring;  // [2][window][H][d]
    int8_t* dsign;      // [d]
    int8_t* ssign;      // [d]
    uint32_t* pos_dev;  // device_position caches: [0] tokens held, [1] arrival counter of the single-token append (null otherwise)
    float* qjl;         // HQ_ROT_QJL: [2][d][d] - S row-major, then S transposed (null otherwise)
    unsigned long long* counters;  // [0] clamp count
    int* flag_host;                // mapped pinned host word: 0 ok, 1 a U-section past 65534 bits, 2 U stream full (sticky)
    int* flag_dev;                 // its device alias (the append kernels raise it, the host polls it without a sync)
    int8_t* scratch_codes;         // [2][chunk][H][d]
    int64_t scratch_tokens;
    float* att_ws;                 // split partials
    size_t att_ws_bytes;
};

namespace hq {

// launch with the programmatic-stream-serialization attribute (PDL): the kernel may begin while its
// predecessor in the stream drains; it synchronizes with griddepcontrol.wait (hq_tc.cuh)
template <class... KArgs, class... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

#define HQ_CUDA_CHECK(ctx, call)                                                        \
    do {                                                                                \
        cudaError_t e__ = (call);                                                       \
        if (e__ != cudaSuccess) {                                                       \
            (ctx)->err = std::string(#call) + ": " + cudaGetErrorString(e__);           \
            return HQ_ERR_CUDA;                                                         \
        }                                                                               \
    } while (0)

// ---- encode (hq_encode.cu) ----
void launch_signs(uint64_t seed, uint32_t stream_id, int64_t n, int8_t* out, cudaStream_t st);
// weights: W [m, n_in] -> codes [m, n_in] int8, norms [m, n_kt] u16; counters[0] += clamps,
// counters[1 + a*8 + k] += total bits of class a at Rice parameter k (auto-k, FORMAT §3)
void launch_quantize_weights(const void* W, int dtype, int64_t m, int64_t n_in, int64_t ld, int lattice, int n,
                             float A, const int8_t* dsign, int8_t* codes, uint16_t* norms,
                             unsigned long long* counters, cudaStream_t st);
// KV: x [n_tok, H, d] bf16 -> codes [n_tok, H, d], norm written to norm_out[h*max_tokens + token0 + t]
void launch_quantize_kv(const void* x, int64_t n_tok, int H, int d, int64_t token0, int role, int lattice,
                        float A, int rotation, int dither, uint64_t seed, const int8_t* dsign,
                        const int8_t* ssign, int8_t* codes, uint16_t* norm_out, int64_t max_tokens,
                        unsigned long long* counters, cudaStream_t st, const float* qjl_t = nullptr);
void launch_set_u32(uint32_t* dst, uint32_t v, cudaStream_t st);
void launch_transpose_f32(const float* a, float* at, int n, cudaStream_t st);
// activations: x [B, n_in] -> q int8 [B, n_in], s_x [B, n_kt], optional u
void launch_act_quant(const void* x, int dtype, int64_t B, int64_t n_in, int64_t ldx, int lattice, int n,
                      const int8_t* dsign, int8_t* q, float* s_x, float* u, cudaStream_t st);
// activations as the E8 fused kernel's B operand tiles (UMMA layout, permuted K, + scales); n_tile = 128
void launch_act_blob(const void* x, int dtype, int64_t B, int64_t n_in, int64_t ldx, const int8_t* dsign, int NB,
                     uint8_t* bblob, cudaStream_t st, int fp8 = 0);
// the same for RHT tiles of 256: two operand chunks of 128 K-bytes per tile (large-M path at n_tile = 256)
void launch_act_blob256(const void* x, int dtype, int64_t B, int64_t n_in, int64_t ldx, const int8_t* dsign, int NB,
                        uint8_t* bblob, cudaStream_t st, int fp8 = 0);
// ulen_tmp[sg*32 + i] for all sub-groups (0 for absent rows); err_flag[0] set if a tile exceeds 8160 bits,
// err_flag[4] = max over present rows of 65535 - ulen, err_flag[5] = max over present rows of ulen
void launch_tile_ulen(const int8_t* codes, int64_t m, int64_t n_in, int lattice, int n, int k0, int k1,
                      uint16_t* ulen_tmp, int* err_flag, cudaStream_t st);
// group_off[G4+1] (sub-group offsets, 16-byte units) by a device prefix sum; totals[0] = sum of ulen over all tiles
void launch_group_offsets(const uint16_t* ulen_tmp, int64_t G4, int rw_words, uint32_t* group_off,
                          unsigned long long* totals, uint32_t* max_group16, cudaStream_t st);
void launch_pack_groups(const int8_t* codes, const uint16_t* norms, const uint16_t* ulen_tmp, int64_t m,
                        int64_t n_in, int lattice, int n, int k0, int k1, const uint32_t* group_off,
                        uint8_t* blob, cudaStream_t st);
// KV pack: per (role, head) prefix over the new tokens' ulen, then bit-pack into rem/una
void launch_kv_pack(const int8_t* codes /*[n_tok,H,d]*/, int64_t n_tok, int H, int d, int64_t token0, int role,
                    int lattice, int k0, int k1, int rbits, int64_t max_tokens, int64_t rem_words,
                    int64_t una_words, int64_t n_blk, uint32_t* rem, uint32_t* una, uint16_t* ulen,
                    uint32_t* blk_off, uint32_t* upos, int* err_flag, cudaStream_t st);
// one token, one launch: the whole append chain incl. the ring (bit-identical to the bulk kernels)
void launch_kv_append1(const hq_kv* kv, const void* k, const void* v, cudaStream_t st);
void launch_kv_ring(const void* k, const void* v, int64_t n_tok, int H, int d, int64_t token0, int window,
                    __nv_bfloat16* ring, cudaStream_t st);

// ---- decode + linear (hq_linear.cu) ----
void launch_decode_int8(const hq_weight* w, int8_t* codes, uint16_t* norms, cudaStream_t st);
// the whole of hq_linear after argument checks: activation cast, fused decode + MMA, split-K finalize
hq_status launch_linear(hq_ctx* ctx, const hq_weight* w, const void* x, int dtype, int64_t B, int64_t ldx,
                        void* y_bf16, int64_t ldy, float* y_f32, int32_t* acc_i32, uint8_t* ws, cudaStream_t st);
size_t linear_workspace_bytes(const hq_ctx* ctx, const hq_weight* w, int64_t B);
// several weights that share x in ONE fused launch (hq_linear_group)
bool linear_group_compatible(const hq_weight* const* ws, int n_w);
size_t linear_group_workspace_bytes(const hq_ctx* ctx, const hq_weight* const* ws, int n_w, int64_t B);
hq_status launch_linear_group(hq_ctx* ctx, const hq_weight* const* ws, int n_w, const void* x, int dtype, int64_t B,
                              int64_t ldx, void* const* ys_bf16, const int64_t* ldys, float* const* ys_f32,
                              int32_t* acc_i32, uint8_t* wsbuf, cudaStream_t st, const hq_fold* fold = nullptr);
bool linear_uses_e8_fast(const hq_weight* w);
hq_status launch_linear_fp8(hq_ctx* ctx, const hq_weight* w, const void* x, int dtype, int64_t B, int64_t ldx, void* y_bf16,
                            int64_t ldy, float* y_f32, float* acc_f32, uint8_t* wsbuf, cudaStream_t st);
hq_status launch_decode_ceiling(hq_ctx* ctx, const hq_weight* w, int reps, cudaStream_t st, double* scalars_per_s);
// hq_linear_static: the address of the static scratch array (once per device, that device current), and the launch
hq_status linear_static_setup(hq_ctx* ctx);
hq_status launch_linear_static(hq_ctx* ctx, const hq_weight* w, const void* x, int dtype, void* y_bf16, float* y_f32,
                               cudaStream_t st);

// ---- KV decode + attend (hq_attend.cu) ----
void launch_kv_decode_int8(const hq_kv* kv, int role, int64_t t0, int64_t n, int8_t* codes, cudaStream_t st);
hq_status launch_attend(hq_ctx* ctx, const hq_kv* kv, const void* q, int q_heads, void* out_bf16,
                        float* out_f32, cudaStream_t st);
size_t attend_workspace_bytes(const hq_ctx* ctx, const hq_kv* kv);

}  // namespace hq
