// hq_api.cu — the C ABI of libhq.so (include/hq.h): argument checking, memory through the caller's
// allocator, kernel sequencing.  No compute happens on the host; there is no CPU fallback.
#include <math.h>
#include <string.h>

#include <new>
#include <vector>

#include "hq_common.cuh"
#include "hq_e8_decode.cuh"
#include "hq_internal.h"

using namespace hq;

namespace {

bool valid_lattice(int l) { return l == HQ_Z || l == HQ_A2 || l == HQ_D4 || l == HQ_E8; }
bool valid_tile(int n) { return n == 64 || n == 128 || n == 256; }

void* ctx_alloc(hq_ctx* ctx, size_t bytes) {
    if (bytes == 0) bytes = 16;
    void* p = ctx->alloc.alloc(ctx->alloc.user, bytes);
    if (!p) ctx->err = "allocator returned NULL for " + std::to_string(bytes) + " bytes";
    return p;
}
void ctx_free(hq_ctx* ctx, void* p) {
    if (p) ctx->alloc.free(ctx->alloc.user, p);
}

hq_status fail(hq_ctx* ctx, hq_status s, const char* msg) {
    if (ctx) ctx->err = msg;
    return s;
}

// every entry point that launches work makes the context's device current (two contexts on two GPUs in one process)
#define HQ_ENTER(ctx) HQ_CUDA_CHECK(ctx, cudaSetDevice((ctx)->device))

// sticky error state of a KV cache: the append kernels raise the flag in mapped host memory (no synchronization here)
hq_status kv_flag_status(hq_ctx* ctx, const hq_kv* kv) {
    const int f = *(volatile int*)kv->flag_host;
    if (f == 1) return fail(ctx, HQ_ERR_FORMAT, "a vector's U-section exceeds 65534 bits (FORMAT §4); the cache is unusable");
    if (f == 2) return fail(ctx, HQ_ERR_FORMAT, "U-stream capacity exceeded (hq_kv_config.una_capacity_bits); the cache is unusable");
    if (f == 3) return fail(ctx, HQ_ERR_FORMAT, "a replayed append ran past max_tokens (device_position cache); the cache is unusable");
    return HQ_OK;
}

// device_position caches: the host's token count follows the device's (blocking)
static hq_status kv_refresh_position(hq_ctx* ctx, hq_kv* kv) {
    if (!kv->pos_dev) return HQ_OK;
    uint32_t t = 0;
    HQ_CUDA_CHECK(ctx, cudaDeviceSynchronize());
    HQ_CUDA_CHECK(ctx, cudaMemcpy(&t, kv->pos_dev, 4, cudaMemcpyDeviceToHost));
    kv->n_tokens = (int64_t)t;
    return HQ_OK;
}

// calibration table b(SNR) written by oracle/make_calib_table.py (G17): HQ_CALIB_N grid points from HQ_CALIB_SNR0 in
// steps of HQ_CALIB_STEP dB; per lattice (Z, A2, D4, E8) the payload bits per scalar and the best k-set
#include "hq_calib_table.inc"
int calib_index(int lattice) { return lattice == HQ_Z ? 0 : lattice == HQ_A2 ? 1 : lattice == HQ_D4 ? 2 : 3; }

constexpr uint32_t HQW_MAGIC = 0x31575148u;   // "HQW1"
constexpr uint32_t HQW_VERSION = 2u;           // FORMAT v2 (sub-group container)

}  // namespace

extern "C" {

hq_status hq_create(hq_ctx** out, const hq_allocator* alloc, int cuda_device) {
    if (!out || !alloc || !alloc->alloc || !alloc->free) return HQ_ERR_INVALID_ARG;
    *out = nullptr;
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || cuda_device < 0 || cuda_device >= count) return HQ_ERR_UNSUPPORTED;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, cuda_device) != cudaSuccess) return HQ_ERR_CUDA;
    if (prop.major != 10) return HQ_ERR_UNSUPPORTED;  // tcgen05 / TMEM: sm_100a only, no fallback
    if (cudaSetDevice(cuda_device) != cudaSuccess) return HQ_ERR_CUDA;
    hq_ctx* ctx = new (std::nothrow) hq_ctx();
    if (!ctx) return HQ_ERR_ALLOC;
    ctx->alloc = *alloc;
    ctx->device = cuda_device;
    ctx->sm_count = prop.multiProcessorCount;
    ctx->err = "";
    // phase-1 table of the E8 fast decoder: [parity][byte][copy] (hq_e8_decode.cuh)
    std::vector<uint32_t> lut(E8_LUT_WORDS);
    for (int par = 0; par < 2; ++par)
        for (int b = 0; b < 256; ++b)
            for (int c = 0; c < E8_LUT_COPIES; ++c) lut[(par * 256 + b) * E8_LUT_COPIES + c] = unary_lut_entry(b, par);
    ctx->e8_lut = (uint32_t*)ctx_alloc(ctx, E8_LUT_BYTES);
    if (!ctx->e8_lut) { delete ctx; return HQ_ERR_ALLOC; }
    if (cudaMemcpy(ctx->e8_lut, lut.data(), E8_LUT_BYTES, cudaMemcpyHostToDevice) != cudaSuccess) {
        ctx_free(ctx, ctx->e8_lut);
        delete ctx;
        return HQ_ERR_CUDA;
    }
    if (cudaStreamCreateWithFlags(&ctx->side, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&ctx->ev_join, cudaEventDisableTiming) != cudaSuccess) {
        ctx_free(ctx, ctx->e8_lut);
        delete ctx;
        return HQ_ERR_CUDA;
    }
    // set-up for hq_linear_static (the device is current): a failure here only disables that entry point
    (void)linear_static_setup(ctx);
    *out = ctx;
    return HQ_OK;
}

void hq_destroy(hq_ctx* ctx) {
    if (!ctx) return;
    if (ctx->side) cudaStreamDestroy(ctx->side);
    if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
    if (ctx->ev_join) cudaEventDestroy(ctx->ev_join);
    ctx_free(ctx, ctx->ws);
    ctx_free(ctx, ctx->e8_lut);
    ctx_free(ctx, ctx->e8_cnt);
    delete ctx;
}

const char* hq_last_error(const hq_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

hq_status hq_profile_enable(hq_ctx* ctx, int32_t on) {
    if (!ctx) return HQ_ERR_INVALID_ARG;
    ctx->prof = on != 0;
    return HQ_OK;
}

hq_status hq_profile_read(hq_ctx* ctx, double* total_ms, int64_t* launches) {
    if (!ctx || !total_ms || !launches) return HQ_ERR_INVALID_ARG;
    double ms = 0.0;
    int64_t n = 0;
    for (size_t i = 0; i + 1 < ctx->prof_ev.size(); i += 2) {
        HQ_CUDA_CHECK(ctx, cudaEventSynchronize(ctx->prof_ev[i + 1]));
        float t = 0.0f;
        HQ_CUDA_CHECK(ctx, cudaEventElapsedTime(&t, ctx->prof_ev[i], ctx->prof_ev[i + 1]));
        ms += t;
        ++n;
        cudaEventDestroy(ctx->prof_ev[i]);
        cudaEventDestroy(ctx->prof_ev[i + 1]);
    }
    ctx->prof_ev.clear();
    *total_ms = ms;
    *launches = n;
    return HQ_OK;
}

hq_status hq_measure_decode_ceiling(hq_ctx* ctx, const hq_weight* w, int32_t reps, void* stream, double* scalars_per_s) {
    if (!ctx) return HQ_ERR_INVALID_ARG;
    if (!w || !scalars_per_s || reps == 0) return fail(ctx, HQ_ERR_INVALID_ARG, "bad argument");
    if (w->ctx != ctx) return fail(ctx, HQ_ERR_INVALID_ARG, "the weight belongs to another context");
    if (!linear_uses_e8_fast(w) || w->m < 128) return fail(ctx, HQ_ERR_UNSUPPORTED, "needs an E8 / tile 128 / k <= 3 weight with a full row block");
    HQ_ENTER(ctx);
    return launch_decode_ceiling(ctx, w, reps, (cudaStream_t)stream, scalars_per_s);
}

double hq_alpha(int32_t lattice, double snr_db) {
    if (!valid_lattice(lattice)) return 0.0;
    return sqrt(pow(10.0, snr_db / 10.0) * second_moment(lattice));
}

hq_status hq_snr_for_bps(const hq_ctx* ctx, int32_t lattice, double target_bps, float* snr_db_out, int32_t* rice_k_out) {
    (void)ctx;   // a host table lookup
    if (!valid_lattice(lattice) || !snr_db_out) return HQ_ERR_INVALID_ARG;
    const float* b = HQ_CALIB_BPS[calib_index(lattice)];
    if (!(target_bps >= b[0]) || !(target_bps <= b[HQ_CALIB_N - 1])) return HQ_ERR_INVALID_ARG;
    int i = 0;
    while (i + 2 < HQ_CALIB_N && (double)b[i + 1] <= target_bps) ++i;   // b is increasing in SNR (checked by the generator)
    const double f = (double)b[i + 1] > (double)b[i] ? (target_bps - b[i]) / ((double)b[i + 1] - (double)b[i]) : 0.0;
    *snr_db_out = (float)(HQ_CALIB_SNR0 + HQ_CALIB_STEP * ((double)i + f));
    if (rice_k_out) {
        rice_k_out[0] = HQ_CALIB_K[calib_index(lattice)][i][0];
        rice_k_out[1] = HQ_CALIB_K[calib_index(lattice)][i][1];
    }
    return HQ_OK;
}

// ---------------------------------------------------------------------------------------------
hq_status hq_encode_weights(hq_ctx* ctx, const void* W_dev, int32_t dtype, int64_t m_out, int64_t n_in, int64_t ld,
                            const hq_codec_config* cfg, void* stream, hq_weight** out) {
    if (!ctx) return HQ_ERR_INVALID_ARG;
    if (!W_dev || !cfg || !out) return fail(ctx, HQ_ERR_INVALID_ARG, "null argument");
    *out = nullptr;
    if (!valid_lattice(cfg->lattice) || (dtype != HQ_F32 && dtype != HQ_BF16))
        return fail(ctx, HQ_ERR_INVALID_ARG, "bad lattice or dtype");
    if (!valid_tile(cfg->n_tile) || m_out <= 0 || n_in <= 0 || n_in % cfg->n_tile != 0 || ld < n_in)
        return fail(ctx, HQ_ERR_SHAPE, "n_tile must be 64/128/256 and divide n_in (the paper auto-shrinks, Table 4 L322; we reject)");
    for (int a = 0; a < 2; ++a)
        if (cfg->rice_k[a] < -1 || cfg->rice_k[a] > 7) return fail(ctx, HQ_ERR_INVALID_ARG, "rice_k must be -1 or 0..7");
    cudaStream_t st = (cudaStream_t)stream;
    HQ_CUDA_CHECK(ctx, cudaSetDevice(ctx->device));

    hq_weight* w = new (std::nothrow) hq_weight();
    if (!w) return HQ_ERR_ALLOC;
    memset((void*)w, 0, sizeof(*w));
    w->ctx = ctx;
    w->m = m_out; w->n_in = n_in; w->lattice = cfg->lattice; w->n = cfg->n_tile; w->snr_db = cfg->snr_db;
    w->seed = cfg->seed;
    w->alpha = hq_alpha(cfg->lattice, (double)cfg->snr_db);
    w->A = (float)(w->alpha * sqrt((double)w->n));
    w->n_kt = n_in / w->n; w->n_rb = (m_out + 127) / 128; w->G = w->n_rb * w->n_kt;

    int8_t* codes = nullptr;
    uint16_t *norms = nullptr, *ulen_tmp = nullptr;
    unsigned long long* counters = nullptr;  // [0] clamps, [1..16] auto-k totals, [17] ubits total, [18] err flag, [19] max group
    hq_status rc = HQ_OK;
    auto cleanup = [&]() {
        ctx_free(ctx, codes); ctx_free(ctx, norms); ctx_free(ctx, ulen_tmp); ctx_free(ctx, counters);
    };
    auto bail = [&](hq_status s) {
        cleanup();
        hq_weight_free(ctx, w);
        return s;
    };
    w->dsign = (int8_t*)ctx_alloc(ctx, (size_t)n_in);
    codes = (int8_t*)ctx_alloc(ctx, (size_t)(m_out * n_in));
    norms = (uint16_t*)ctx_alloc(ctx, (size_t)(m_out * w->n_kt) * 2);
    ulen_tmp = (uint16_t*)ctx_alloc(ctx, (size_t)w->G * 128 * 2);
    counters = (unsigned long long*)ctx_alloc(ctx, 32 * sizeof(unsigned long long));
    w->group_off = (uint32_t*)ctx_alloc(ctx, (size_t)(4 * w->G + 1) * 4);
    if (!w->dsign || !codes || !norms || !ulen_tmp || !counters || !w->group_off) return bail(HQ_ERR_ALLOC);

#define HQ_TRY(call)                                                                 \
    do {                                                                             \
        cudaError_t e__ = (call);                                                    \
        if (e__ != cudaSuccess) {                                                    \
            ctx->err = std::string(#call) + ": " + cudaGetErrorString(e__);          \
            return bail(HQ_ERR_CUDA);                                                \
        }                                                                            \
    } while (0)

    HQ_TRY(cudaMemsetAsync(counters, 0, 32 * sizeof(unsigned long long), st));
    launch_signs(w->seed, 1u, n_in, w->dsign, st);
    launch_quantize_weights(W_dev, dtype, m_out, n_in, ld, w->lattice, w->n, w->A, w->dsign, codes, norms, counters, st);
    HQ_TRY(cudaGetLastError());
    unsigned long long hc[32];
    HQ_TRY(cudaMemcpyAsync(hc, counters, sizeof(hc), cudaMemcpyDeviceToHost, st));
    HQ_TRY(cudaStreamSynchronize(st));
    w->clamp_count = (int64_t)hc[0];
    // Rice parameters (FORMAT §3): argmin of total bits, ties -> smaller; D4 ties k_t = max(k_s-1, 0)
    int k0 = cfg->rice_k[0], k1 = cfg->rice_k[1];
    if (k0 < 0 || (k1 < 0 && (w->lattice == HQ_D4 || w->lattice == HQ_A2))) {
        const unsigned long long* t0 = hc + 1;
        const unsigned long long* t1 = hc + 9;
        if (w->lattice == HQ_D4) {
            int best = 0;
            unsigned long long bv = ~0ull;
            for (int ks = 0; ks < 8; ++ks) {
                unsigned long long v = t0[ks] + t1[ks > 0 ? ks - 1 : 0];
                if (v < bv) { bv = v; best = ks; }
            }
            k0 = best; k1 = best > 0 ? best - 1 : 0;
        } else {
            int b0 = 0, b1 = 0;
            for (int kk = 1; kk < 8; ++kk) {
                if (t0[kk] < t0[b0]) b0 = kk;
                if (t1[kk] < t1[b1]) b1 = kk;
            }
            k0 = b0; k1 = (w->lattice == HQ_A2) ? b1 : b0;
        }
    }
    if (k1 < 0) k1 = k0;
    if (w->lattice == HQ_Z || w->lattice == HQ_E8) k1 = k0;
    w->k0 = k0; w->k1 = k1;
    w->rbits = rbits_of(w->lattice, w->n, k0, k1);

    int* err_flag = (int*)(counters + 18);
    uint32_t* maxg = (uint32_t*)(counters + 19);
    launch_tile_ulen(codes, m_out, n_in, w->lattice, w->n, k0, k1, ulen_tmp, err_flag, st);
    launch_group_offsets(ulen_tmp, 4 * w->G, (w->rbits + 31) / 32, w->group_off, counters + 17, maxg, st);
    HQ_TRY(cudaGetLastError());
    uint32_t total16 = 0;
    HQ_TRY(cudaMemcpyAsync(&total16, w->group_off + 4 * w->G, 4, cudaMemcpyDeviceToHost, st));
    HQ_TRY(cudaMemcpyAsync(hc, counters, sizeof(hc), cudaMemcpyDeviceToHost, st));
    HQ_TRY(cudaStreamSynchronize(st));
    if (*(int*)(hc + 18) != 0) {
        ctx->err = "a tile's U-section exceeds 8160 bits (FORMAT §5)";
        return bail(HQ_ERR_FORMAT);
    }
    w->max_group16 = *(uint32_t*)(hc + 19);
    w->min_ulen = 65535u - ((uint32_t*)(hc + 18))[4];
    w->max_ulen = ((uint32_t*)(hc + 18))[5];
    w->blob_bytes = (int64_t)total16 * 16;
    w->payload_bits = (int64_t)hc[17] + m_out * w->n_kt * (int64_t)w->rbits;
    w->blob = (uint8_t*)ctx_alloc(ctx, (size_t)w->blob_bytes + 4096);  // slack: decoders read a word ahead, the fused kernel prefetches whole lines
    if (!w->blob) return bail(HQ_ERR_ALLOC);
    HQ_TRY(cudaMemsetAsync(w->blob, 0, (size_t)w->blob_bytes + 4096, st));
    launch_pack_groups(codes, norms, ulen_tmp, m_out, n_in, w->lattice, w->n, k0, k1, w->group_off, w->blob, st);
    HQ_TRY(cudaGetLastError());
    HQ_TRY(cudaStreamSynchronize(st));
#undef HQ_TRY
    cleanup();
    *out = w;
    return rc;
}

void hq_weight_free(hq_ctx* ctx, hq_weight* w) {
    if (!w) return;
    if (!ctx) ctx = w->ctx;
    ctx_free(ctx, w->blob);
    ctx_free(ctx, w->group_off);
    ctx_free(ctx, w->dsign);
    delete w;
}

hq_status hq_weight_get_info(const hq_weight* w, hq_weight_info* out) {
    if (!w || !out) return HQ_ERR_INVALID_ARG;
    out->m_out = w->m; out->n_in = w->n_in; out->lattice = w->lattice; out->n_tile = w->n;
    out->rice_k[0] = w->k0; out->rice_k[1] = w->k1; out->snr_db = w->snr_db; out->alpha = w->alpha;
    out->seed = w->seed; out->payload_bits = w->payload_bits;
    out->norm_bits = 16 * w->m * w->n_kt; out->length_bits = 16 * w->m * w->n_kt;
    out->blob_bytes = w->blob_bytes; out->n_groups = 4 * w->G; out->clamp_count = w->clamp_count;
    return HQ_OK;
}

hq_status hq_weight_export(const hq_weight* w, const void** blob_dev, const uint32_t** group_off_dev) {
    if (!w || !blob_dev || !group_off_dev) return HQ_ERR_INVALID_ARG;
    *blob_dev = w->blob;
    *group_off_dev = w->group_off;
    return HQ_OK;
}

hq_status hq_weight_stats(const hq_weight* w, hq_stats* out) {
    if (!w || !out) return HQ_ERR_INVALID_ARG;
    const int64_t tiles = w->m * w->n_kt;
    out->payload_bits = w->payload_bits; out->norm_bits = 16 * tiles; out->length_bits = 16 * tiles;
    out->offset_bits = 32 * 4 * w->G;
    out->padding_bits = 8 * w->blob_bytes - out->payload_bits - out->norm_bits - out->length_bits;
    out->clamp_count = w->clamp_count; out->n_tiles = tiles;
    out->tile_bits_min = (int32_t)(w->rbits + w->min_ulen); out->tile_bits_max = (int32_t)(w->rbits + w->max_ulen);
    const double sc = (double)w->m * (double)w->n_in;
    out->bits_per_scalar_payload = (double)out->payload_bits / sc;
    out->bits_per_scalar_total = (double)(out->payload_bits + out->norm_bits + out->length_bits) / sc;
    return HQ_OK;
}

hq_status hq_weight_export_host(hq_ctx* ctx, const hq_weight* w, hq_weight_header* hd, void* blob_host,
                                uint32_t* sub_off_host, void* stream) {
    if (!ctx) return HQ_ERR_INVALID_ARG;
    if (!w || !hd || ((blob_host == nullptr) != (sub_off_host == nullptr))) return fail(ctx, HQ_ERR_INVALID_ARG, "null argument");
    if (w->ctx != ctx) return fail(ctx, HQ_ERR_INVALID_ARG, "the weight belongs to another context");
    HQ_ENTER(ctx);
    memset(hd, 0, sizeof(*hd));
    hd->magic = HQW_MAGIC; hd->version = HQW_VERSION;
    hd->m_out = w->m; hd->n_in = w->n_in; hd->lattice = w->lattice; hd->n_tile = w->n;
    hd->rice_k[0] = w->k0; hd->rice_k[1] = w->k1; hd->snr_db = w->snr_db; hd->seed = w->seed;
    hd->blob_bytes = w->blob_bytes; hd->n_groups = 4 * w->G;
    hd->payload_bits = w->payload_bits; hd->clamp_count = w->clamp_count;
    hd->ulen_min = (int32_t)w->min_ulen; hd->ulen_max = (int32_t)w->max_ulen;
    if (!blob_host) return HQ_OK;
    cudaStream_t st = (cudaStream_t)stream;
    HQ_CUDA_CHECK(ctx, cudaMemcpyAsync(blob_host, w->blob, (size_t)w->blob_bytes, cudaMemcpyDeviceToHost, st));
    HQ_CUDA_CHECK(ctx, cudaMemcpyAsync(sub_off_host, w->group_off, (size_t)(4 * w->G + 1) * 4, cudaMemcpyDeviceToHost, st));
    HQ_CUDA_CHECK(ctx, cudaStreamSynchronize(st));
    return HQ_OK;
}

hq_status hq_weight_import(hq_ctx* ctx, const hq_weight_header* hd, const void* blob_host, const uint32_t* sub_off_host,
                           void* stream, hq_weight** out) {
    if (!ctx) return HQ_ERR_INVALID_ARG;
    if (!hd || !blob_host || !sub_off_host || !out) return fail(ctx, HQ_ERR_INVALID_ARG, "null argument");
    *out = nullptr;
    if (hd->magic != HQW_MAGIC || hd->version != HQW_VERSION) return fail(ctx, HQ_ERR_FORMAT, "not an HQW1 v2 header");
    if (!valid_lattice(hd->lattice) || !valid_tile(hd->n_tile) || hd->m_out <= 0 || hd->n_in <= 0 || hd->n_in % hd->n_tile != 0)
        return fail(ctx, HQ_ERR_FORMAT, "bad lattice / tile / shape in the header");
    for (int a = 0; a < 2; ++a)
        if (hd->rice_k[a] < 0 || hd->rice_k[a] > 7) return fail(ctx, HQ_ERR_FORMAT, "bad rice_k in the header");
    const int64_t n_kt = hd->n_in / hd->n_tile, n_rb = (hd->m_out + 127) / 128, G = n_rb * n_kt;
    if (hd->n_groups != 4 * G || hd->blob_bytes <= 0 || hd->blob_bytes % 16 != 0) return fail(ctx, HQ_ERR_FORMAT, "group count / blob size do not match the shape");
    const int rbits = rbits_of(hd->lattice, hd->n_tile, hd->rice_k[0], hd->rice_k[1]);
    const int64_t rw_words = (rbits + 31) / 32;
    // layout checks (FORMAT §5): offsets increasing, inside the blob, and each sub-group exactly as long as its
    // ulen header implies; present rows' ulen in [n_tile, 8160], absent rows' 0.  A decoder never leaves a checked blob.
    const uint8_t* blob = (const uint8_t*)blob_host;
    uint32_t umin = 65535u, umax = 0u;
    int64_t usum = 0;
    if (sub_off_host[0] != 0 || (int64_t)sub_off_host[4 * G] * 16 != hd->blob_bytes) return fail(ctx, HQ_ERR_FORMAT, "sub_off does not span the blob");
    for (int64_t sg = 0; sg < 4 * G; ++sg) {
        const int64_t o0 = (int64_t)sub_off_host[sg] * 16, o1 = (int64_t)sub_off_host[sg + 1] * 16;
        if (o1 <= o0 || o1 > hd->blob_bytes || o1 - o0 < 128 + rw_words * 128) return fail(ctx, HQ_ERR_FORMAT, "sub_off is not increasing / a sub-group is truncated");
        const uint16_t* ul = (const uint16_t*)(blob + o0);
        const int64_t rb = (sg / 4) / n_kt, row0 = rb * 128 + (sg % 4) * 32;
        int64_t words = 0;
        for (int i = 0; i < 32; ++i) {
            const uint32_t L = ul[i];
            const bool present = row0 + i < hd->m_out;
            if (present ? (L < (uint32_t)hd->n_tile || L > 8160u) : (L != 0u)) return fail(ctx, HQ_ERR_FORMAT, "a tile's ulen is out of range");
            if (present) { umin = L < umin ? L : umin; umax = L > umax ? L : umax; usum += L; }
            words += (L + 31) / 32;
        }
        const int64_t need = (128 + rw_words * 128 + words * 4 + 15) / 16 * 16;
        if (need != o1 - o0) return fail(ctx, HQ_ERR_FORMAT, "a sub-group's size does not match its ulen header");
    }
    if (usum + hd->m_out * n_kt * (int64_t)rbits != hd->payload_bits) return fail(ctx, HQ_ERR_FORMAT, "payload_bits does not match the blob");
    HQ_ENTER(ctx);
    cudaStream_t st = (cudaStream_t)stream;
    hq_weight* w = new (std::nothrow) hq_weight();
    if (!w) return HQ_ERR_ALLOC;
    memset((void*)w, 0, sizeof(*w));
    w->ctx = ctx;
    w->m = hd->m_out; w->n_in = hd->n_in; w->lattice = hd->lattice; w->n = hd->n_tile; w->snr_db = hd->snr_db;
    w->seed = hd->seed; w->k0 = hd->rice_k[0]; w->k1 = hd->rice_k[1]; w->rbits = rbits;
    w->alpha = hq_alpha(hd->lattice, (double)hd->snr_db);
    w->A = (float)(w->alpha * sqrt((double)w->n));
    w->n_kt = n_kt; w->n_rb = n_rb; w->G = G;
    w->blob_bytes = hd->blob_bytes; w->payload_bits = hd->payload_bits; w->clamp_count = hd->clamp_count;
    w->min_ulen = umin; w->max_ulen = umax;
    w->dsign = (int8_t*)ctx_alloc(ctx, (size_t)w->n_in);
    w->group_off = (uint32_t*)ctx_alloc(ctx, (size_t)(4 * G + 1) * 4);
    w->blob = (uint8_t*)ctx_alloc(ctx, (size_t)w->blob_bytes + 4096);
    if (!w->dsign || !w->group_off || !w->blob) { hq_weight_free(ctx, w); return HQ_ERR_ALLOC; }
    cudaError_t e = cudaMemsetAsync(w->blob + w->blob_bytes, 0, 4096, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(w->blob, blob_host, (size_t)w->blob_bytes, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(w->group_off, sub_off_host, (size_t)(4 * G + 1) * 4, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) { launch_signs(w->seed, 1u, w->n_in, w->dsign, st); e = cudaGetLastError(); }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);   // the host buffers are the caller's again on return
    if (e != cudaSuccess) {
        ctx->err = std::string("hq_weight_import: ") + cudaGetErrorString(e);
        hq_weight_free(ctx, w);
        return HQ_ERR_CUDA;
    }
    *out = w;
    return HQ_OK;
}

hq_status hq_decode_int8(hq_ctx* ctx, const hq_weight* w, int8_t* codes_dev, uint16_t* norms_dev, void* stream) {
    if (!ctx) return HQ_ERR_INVALID_ARG;
    if (!w || !codes_dev) return fail(ctx, HQ_ERR_INVALID_ARG, "null argument");
    HQ_ENTER(ctx);
    launch_decode_int8(w, codes_dev, norms_dev, (cudaStream_t)stream);
    HQ_CUDA_CHECK(ctx, cudaGetLastError());
    return HQ_OK;
}

hq_status hq_act_quant(hq_ctx* ctx, const hq_weight* w, const void* x_dev, int32_t dtype, int64_t batch, int64_t ldx,
                       int8_t* q_dev, float* s_x_dev, float* u_dev_or_null, void* stream) {
    if (!ctx) return HQ_ERR_INVALID_ARG;
    if (!w || !x_dev || !q_dev || !s_x_dev) return fail(ctx, HQ_ERR_INVALID_ARG, "null argument");
    if (batch <= 0 || ldx < w->n_in) return fail(ctx, HQ_ERR_SHAPE, "bad batch / ldx");
    HQ_ENTER(ctx);
    launch_act_quant(x_dev, dtype, batch, w->n_in, ldx, w->lattice, w->n, w->dsign, q_dev, s_x_dev, u_dev_or_null,
                     (cudaStream_t)stream);
    HQ_CUDA_CHECK(ctx, cudaGetLastError());
    return HQ_OK;
}

hq_status hq_linear_workspace_bytes(const hq_weight* w, int64_t batch, size_t* bytes) {
    if (!w || !bytes || batch <= 0) return HQ_ERR_INVALID_ARG;
    *bytes = linear_workspace_bytes(w->ctx, w, batch);
    return HQ_OK;
}

hq_status hq_linear(hq_ctx* ctx, const hq_weight* w, const void* x_dev, int32_t dtype, int64_t batch, int64_t ldx,
                    void* y_bf16_dev, int64_t ldy, float* y_f32_dev_or_null, int32_t* acc_i32_dev_or_null, void* stream) {
    if (!ctx) return HQ_ERR_INVALID_ARG;
    if (!w || !x_dev || (!y_bf16_dev && !y_f32_dev_or_null)) return fail(ctx, HQ_ERR_INVALID_ARG, "null argument");
    if (batch <= 0 || ldx < w->n_in || (y_bf16_dev && ldy < w->m)) return fail(ctx, HQ_ERR_SHAPE, "bad batch / ldx / ldy");
    if (dtype != HQ_F32 && dtype != HQ_BF16) return fail(ctx, HQ_ERR_INVALID_ARG, "bad dtype");
    if (w->ctx != ctx) return fail(ctx, HQ_ERR_INVALID_ARG, "the weight belongs to another context");
    HQ_ENTER(ctx);
    cudaStream_t st = (cudaStream_t)stream;
    size_t need = linear_workspace_bytes(ctx, w, batch);
    if (need > ctx->ws_bytes) {
        // the old buffer may still be in use by work already enqueued
        if (ctx->ws) { HQ_CUDA_CHECK(ctx, cudaDeviceSynchronize()); ctx_free(ctx, ctx->ws); ctx->ws = nullptr; ctx->ws_bytes = 0; }
        ctx->ws = ctx_alloc(ctx, need);
        if (!ctx->ws) return HQ_ERR_ALLOC;
        ctx->ws_bytes = need;
    }
    return launch_linear(ctx, w, x_dev, dtype, batch, ldx, y_bf16_dev, ldy, y_f32_dev_or_null, acc_i32_dev_or_null,
                         (uint8_t*)ctx->ws, st);
}

hq_status hq_linear_cast(hq_ctx* ctx, const hq_weight* w, const void* x_dev, int32_t dtype, int64_t batch, int64_t ldx,
                         void* y_bf16_dev, int64_t ldy, float* y_f32_dev_or_null, void* acc_dev_or_null, int32_t cast,
                         void* stream) {
    if (!ctx) return HQ_ERR_INVALID_ARG;
    if (cast == HQ_CAST_INT8)
        return hq_linear(ctx, w, x_dev, dtype, batch, ldx, y_bf16_dev, ldy, y_f32_dev_or_null, (int32_t*)acc_dev_or_null, stream);
    if (cast != HQ_CAST_FP8_E4M3) return fail(ctx, HQ_ERR_INVALID_ARG, "bad cast");
    if (!w || !x_dev || (!y_bf16_dev && !y_f32_dev_or_null)) return fail(ctx, HQ_ERR_INVALID_ARG, "null argument");
    if (batch <= 0 || ldx < w->n_in || (y_bf16_dev && ldy < w->m)) return fail(ctx, HQ_ERR_SHAPE, "bad batch / ldx / ldy");
    if (dtype != HQ_F32 && dtype != HQ_BF16) return fail(ctx, HQ_ERR_INVALID_ARG, "bad dtype");
    if (w->ctx != ctx) return fail(ctx, HQ_ERR_INVALID_ARG, "the weight belongs to another context");
    if (w->lattice != HQ_E8 || (w->n != 128 && w->n != 256) || w->k0 > 3 || batch < 64)
        return fail(ctx, HQ_ERR_UNSUPPORTED, "the FP8 cast needs an E8 weight at tile 128 or 256, k <= 3 and batch >= 64");
    HQ_ENTER(ctx);
    const size_t need = (((size_t)((batch + 255) / 256) * (w->n_in / 128) * (256 * 128 + 256 * 4) + 255) & ~(size_t)255) +
                        (((size_t)w->n_rb * (w->n_in / 128) * (16384 + 512) + 255) & ~(size_t)255) + 256;
    if (need > ctx->ws_bytes) {
        if (ctx->ws) { HQ_CUDA_CHECK(ctx, cudaDeviceSynchronize()); ctx_free(ctx, ctx->ws); ctx->ws = nullptr; ctx->ws_bytes = 0; }
        ctx->ws = ctx_alloc(ctx, need);
        if (!ctx->ws) return HQ_ERR_ALLOC;
        ctx->ws_bytes = need;
    }
    return launch_linear_fp8(ctx, w, x_dev, dtype, batch, ldx, y_bf16_dev, ldy, y_f32_dev_or_null, (float*)acc_dev_or_null,
                             (uint8_t*)ctx->ws, (cudaStream_t)stream);
}

hq_status hq_linear_static(hq_ctx* ctx, const hq_weight* w, const void* x_dev, int32_t dtype, void* y_bf16_dev,
                           float* y_f32_dev_or_null, void* stream) {
    if (!ctx) return HQ_ERR_INVALID_ARG;
    if (!w || !x_dev || (!y_bf16_dev && !y_f32_dev_or_null)) return fail(ctx, HQ_ERR_INVALID_ARG, "null argument");
    if (dtype != HQ_F32 && dtype != HQ_BF16) return fail(ctx, HQ_ERR_INVALID_ARG, "bad dtype");
    if (w->ctx != ctx) return fail(ctx, HQ_ERR_INVALID_ARG, "the weight belongs to another context");
    HQ_ENTER(ctx);
    return launch_linear_static(ctx, w, x_dev, dtype, y_bf16_dev, y_f32_dev_or_null, (cudaStream_t)stream);
}

hq_status hq_linear_group(hq_ctx* ctx, const hq_weight* const* ws, int32_t n_w, const void* x_dev, int32_t dtype,
                          int64_t batch, int64_t ldx, void* const* ys_bf16_dev, const int64_t* ldys,
                          float* const* ys_f32_or_null, void* stream) {
    if (!ctx) return HQ_ERR_INVALID_ARG;
    if (!ws || !x_dev || !ys_bf16_dev || !ldys || n_w < 1 || n_w > 4) return fail(ctx, HQ_ERR_INVALID_ARG, "bad group arguments");
    for (int i = 0; i < n_w; ++i) {
        if (!ws[i] || !ys_bf16_dev[i]) return fail(ctx, HQ_ERR_INVALID_ARG, "null weight or output in group");
        if (ws[i]->n_in != ws[0]->n_in) return fail(ctx, HQ_ERR_SHAPE, "the weights of a group must share n_in");
        if (ldys[i] < ws[i]->m) return fail(ctx, HQ_ERR_SHAPE, "bad ldy");
        if (ws[i]->ctx != ctx) return fail(ctx, HQ_ERR_INVALID_ARG, "a weight belongs to another context");
    }
    HQ_ENTER(ctx);
    if (batch <= 0 || ldx < ws[0]->n_in) return fail(ctx, HQ_ERR_SHAPE, "bad batch / ldx");
    if (dtype != HQ_F32 && dtype != HQ_BF16) return fail(ctx, HQ_ERR_INVALID_ARG, "bad dtype");
    if (!linear_group_compatible(ws, n_w)) {   // one by one: same results, more launches
        for (int i = 0; i < n_w; ++i) {
            hq_status s = hq_linear(ctx, ws[i], x_dev, dtype, batch, ldx, ys_bf16_dev[i], ldys[i],
                                    ys_f32_or_null ? ys_f32_or_null[i] : nullptr, nullptr, stream);
            if (s != HQ_OK) return s;
        }
        return HQ_OK;
    }
    size_t need = linear_group_workspace_bytes(ctx, ws, n_w, batch);
    if (need > ctx->ws_bytes) {
        if (ctx->ws) { HQ_CUDA_CHECK(ctx, cudaDeviceSynchronize()); ctx_free(ctx, ctx->ws); ctx->ws = nullptr; ctx->ws_bytes = 0; }
        ctx->ws = ctx_alloc(ctx, need);
        if (!ctx->ws) return HQ_ERR_ALLOC;
        ctx->ws_bytes = need;
    }
    return launch_linear_group(ctx, ws, n_w, x_dev, dtype, batch, ldx, ys_bf16_dev, ldys, ys_f32_or_null, nullptr,
                               (uint8_t*)ctx->ws, (cudaStream_t)stream);
}

hq_status hq_linear_group_fold(hq_ctx* ctx, const hq_weight* const* ws, int32_t n_w, const void* x_dev,
                               const hq_fold* fold, void* const* ys_bf16_dev, float* const* ys_f32_or_null, void* stream) {
    if (!ctx) return HQ_ERR_INVALID_ARG;
    if (!ws || !x_dev || !fold || !ys_bf16_dev || n_w < 1 || n_w > 4) return fail(ctx, HQ_ERR_INVALID_ARG, "bad group arguments");
    if (fold->mode < HQ_FOLD_NONE || fold->mode > HQ_FOLD_SILU_MUL) return fail(ctx, HQ_ERR_INVALID_ARG, "bad fold mode");
    if (fold->mode != HQ_FOLD_NONE && !fold->aux_dev) return fail(ctx, HQ_ERR_INVALID_ARG, "the fold needs aux_dev");
    if (((uintptr_t)x_dev & 7) || ((uintptr_t)fold->aux_dev & 7)) return fail(ctx, HQ_ERR_INVALID_ARG, "x_dev / aux_dev must be 8-byte aligned");
    int64_t ldys[4];
    for (int i = 0; i < n_w; ++i) {
        if (!ws[i] || !ys_bf16_dev[i]) return fail(ctx, HQ_ERR_INVALID_ARG, "null weight or output in group");
        if (ws[i]->n_in != ws[0]->n_in) return fail(ctx, HQ_ERR_SHAPE, "the weights of a group must share n_in");
        if (ws[i]->ctx != ctx) return fail(ctx, HQ_ERR_INVALID_ARG, "a weight belongs to another context");
        ldys[i] = ws[i]->m;
    }
    HQ_ENTER(ctx);
    if (!linear_group_compatible(ws, n_w)) return fail(ctx, HQ_ERR_UNSUPPORTED, "the folds need E8 / tile 128 / k <= 3 weights that share a launch");
    size_t need = linear_group_workspace_bytes(ctx, ws, n_w, 1);
    if (need > ctx->ws_bytes) {
        if (ctx->ws) { HQ_CUDA_CHECK(ctx, cudaDeviceSynchronize()); ctx_free(ctx, ctx->ws); ctx->ws = nullptr; ctx->ws_bytes = 0; }
        ctx->ws = ctx_alloc(ctx, need);
        if (!ctx->ws) return HQ_ERR_ALLOC;
        ctx->ws_bytes = need;
    }
    return launch_linear_group(ctx, ws, n_w, x_dev, HQ_BF16, 1, ws[0]->n_in, ys_bf16_dev, ldys, ys_f32_or_null, nullptr,
                               (uint8_t*)ctx->ws, (cudaStream_t)stream, fold);
}

static size_t a256(size_t v) { return (v + 255) & ~(size_t)255; }
hq_status hq_layer_scratch_view(const hq_layer* L, hq_layer_scratch* out) {
    if (!L || !out || !L->wq || !L->wk || !L->wgate || !L->wo) return HQ_ERR_INVALID_ARG;
    size_t o = 0;
    out->q = o; o += a256((size_t)L->wq->m * 2);
    out->k = o; o += a256((size_t)L->wk->m * 2);
    out->v = o; o += a256((size_t)L->wk->m * 2);
    out->a = o; o += a256((size_t)L->wq->m * 2);
    out->h2 = o; o += a256((size_t)L->wo->m * 2);
    out->gate = o; o += a256((size_t)L->wgate->m * 2);
    out->up = o; o += a256((size_t)L->wgate->m * 2);
    out->total = o;
    return HQ_OK;
}

hq_status hq_layer_decode(hq_ctx* ctx, const hq_layer* L, const void* h_in_dev, void* h_out_dev, void* scratch_dev,
                          size_t scratch_bytes, void* stream) {
    if (!ctx) return HQ_ERR_INVALID_ARG;
    if (!L || !h_in_dev || !h_out_dev || !scratch_dev) return fail(ctx, HQ_ERR_INVALID_ARG, "null argument");
    if (!L->wq || !L->wk || !L->wv || !L->wo || !L->wgate || !L->wup || !L->wdown || !L->g_attn_dev || !L->g_mlp_dev || !L->kv)
        return fail(ctx, HQ_ERR_INVALID_ARG, "incomplete layer");
    const int64_t hidden = L->wq->n_in, d = L->kv->cfg.head_dim, Hkv = L->kv->cfg.kv_heads, ffn = L->wgate->m;
    if (L->q_heads <= 0 || L->wq->m != (int64_t)L->q_heads * d || L->wk->m != Hkv * d || L->wv->m != Hkv * d ||
        L->wk->n_in != hidden || L->wv->n_in != hidden || L->wo->n_in != L->wq->m || L->wo->m != hidden ||
        L->wgate->n_in != hidden || L->wup->n_in != hidden || L->wup->m != ffn || L->wdown->n_in != ffn || L->wdown->m != hidden)
        return fail(ctx, HQ_ERR_SHAPE, "the layer's weight shapes do not fit together");
    hq_layer_scratch sv;
    hq_layer_scratch_view(L, &sv);
    if (scratch_bytes < sv.total || ((uintptr_t)scratch_dev & 255)) return fail(ctx, HQ_ERR_INVALID_ARG, "scratch too small or not 256-byte aligned");
    uint8_t* sc = (uint8_t*)scratch_dev;
    void *q = sc + sv.q, *k = sc + sv.k, *v = sc + sv.v, *a = sc + sv.a, *h2 = sc + sv.h2, *gate = sc + sv.gate, *up = sc + sv.up;
    hq_status s;
    {   // q, k, v = W RMSNorm(h)
        const hq_weight* ws[3] = {L->wq, L->wk, L->wv};
        void* ys[3] = {q, k, v};
        hq_fold f = {HQ_FOLD_RMSNORM, L->eps, L->g_attn_dev, nullptr};
        if ((s = hq_linear_group_fold(ctx, ws, 3, h_in_dev, &f, ys, nullptr, stream)) != HQ_OK) return s;
    }
    if ((s = hq_kv_append(ctx, L->kv, k, v, 1, stream)) != HQ_OK) return s;
    if ((s = hq_attend(ctx, L->kv, q, L->q_heads, a, nullptr, stream)) != HQ_OK) return s;
    {   // h2 = h + W_o a
        const hq_weight* ws[1] = {L->wo};
        void* ys[1] = {h2};
        const void* res[1] = {h_in_dev};
        hq_fold f = {HQ_FOLD_NONE, 0.0f, nullptr, res};
        if ((s = hq_linear_group_fold(ctx, ws, 1, a, &f, ys, nullptr, stream)) != HQ_OK) return s;
    }
    {   // gate, up = W RMSNorm(h2)
        const hq_weight* ws[2] = {L->wgate, L->wup};
        void* ys[2] = {gate, up};
        hq_fold f = {HQ_FOLD_RMSNORM, L->eps, L->g_mlp_dev, nullptr};
        if ((s = hq_linear_group_fold(ctx, ws, 2, h2, &f, ys, nullptr, stream)) != HQ_OK) return s;
    }
    {   // h_out = h2 + W_down (silu(gate) * up)
        const hq_weight* ws[1] = {L->wdown};
        void* ys[1] = {h_out_dev};
        const void* res[1] = {h2};
        hq_fold f = {HQ_FOLD_SILU_MUL, 0.0f, up, res};
        if ((s = hq_linear_group_fold(ctx, ws, 1, gate, &f, ys, nullptr, stream)) != HQ_OK) return s;
    }
    return HQ_OK;
}

// ---------------------------------------------------------------------------------------------
hq_status hq_kv_create(hq_ctx* ctx, const hq_kv_config* cfg, hq_kv** out) {
    if (!ctx) return HQ_ERR_INVALID_ARG;
    if (!cfg || !out) return fail(ctx, HQ_ERR_INVALID_ARG, "null argument");
    *out = nullptr;
    if (!valid_lattice(cfg->codec.lattice)) return fail(ctx, HQ_ERR_INVALID_ARG, "bad lattice");
    if (!valid_tile(cfg->head_dim) || cfg->codec.n_tile != cfg->head_dim || cfg->kv_heads <= 0 || cfg->max_tokens <= 0)
        return fail(ctx, HQ_ERR_SHAPE, "head_dim must be 64/128/256 and equal codec.n_tile");
    if (cfg->rotation != HQ_ROT_NONE && cfg->rotation != HQ_ROT_SIGNS && cfg->rotation != HQ_ROT_QJL) return fail(ctx, HQ_ERR_INVALID_ARG, "bad rotation");
    if ((cfg->rotation == HQ_ROT_QJL) != (cfg->qjl_dev != nullptr)) return fail(ctx, HQ_ERR_INVALID_ARG, "rotation qjl needs qjl_dev, the other rotations must not pass one");
    if (cfg->una_capacity_bits < 0) return fail(ctx, HQ_ERR_INVALID_ARG, "una_capacity_bits must be >= 0");
    HQ_ENTER(ctx);
    if (cfg->codec.rice_k[0] < 0 || cfg->codec.rice_k[0] > 7 || cfg->codec.rice_k[1] > 7)
        return fail(ctx, HQ_ERR_INVALID_ARG, "KV needs explicit rice_k");
    if (cfg->window < 0 || cfg->window > cfg->head_dim) return fail(ctx, HQ_ERR_SHAPE, "window must be in [0, head_dim]");
    hq_kv* kv = new (std::nothrow) hq_kv();
    if (!kv) return HQ_ERR_ALLOC;
    memset((void*)kv, 0, sizeof(*kv));
    kv->ctx = ctx;
    kv->cfg = *cfg;
    int H = cfg->kv_heads, d = cfg->head_dim, lat = cfg->codec.lattice;
    kv->k0 = cfg->codec.rice_k[0];
    kv->k1 = (lat == HQ_Z || lat == HQ_E8 || cfg->codec.rice_k[1] < 0) ? kv->k0 : cfg->codec.rice_k[1];
    kv->rbits = rbits_of(lat, d, kv->k0, kv->k1);
    kv->alpha = hq_alpha(lat, (double)cfg->codec.snr_db);
    kv->A = (float)(kv->alpha * sqrt((double)d));
    int64_t mt = cfg->max_tokens;
    if ((double)mt * (kv->rbits > 0 ? kv->rbits : 1) > 4.0e9) { delete kv; return fail(ctx, HQ_ERR_SHAPE, "max_tokens too large for 32-bit bit offsets"); }
    kv->n_blk = (mt + 127) / 128;
    kv->rem_words = (mt * kv->rbits + 31) / 32 + 4;
    // U-stream capacity per (role, head): the caller's figure, else an estimate with margin.  On a vector normalized to
    // radius alpha sqrt(d), E|zz| ~ E|c| <= alpha (0.8 alpha if Gaussian), so a class-a symbol costs about
    // 1 + (0.8 alpha + 0.5) / 2^k_a unary bits; x 1.3, at least 4 per scalar.  Overflow is detected, never written.
    int64_t una_bits = cfg->una_capacity_bits;
    if (una_bits == 0) {
        const int kmin = kv->k0 < kv->k1 ? kv->k0 : kv->k1;
        double per = 1.3 * (1.0 + (0.8 * kv->alpha + 0.5) / (double)(1 << kmin));
        if (per < 4.0) per = 4.0;
        una_bits = (int64_t)((double)mt * d * per) + 4096;
    }
    if (una_bits > 0xffff0000ll) una_bits = 0xffff0000ll;
    kv->una_words = una_bits / 32 + 4;
    size_t n_rh = (size_t)2 * H;
    kv->rem = (uint32_t*)ctx_alloc(ctx, n_rh * kv->rem_words * 4);
    kv->una = (uint32_t*)ctx_alloc(ctx, n_rh * kv->una_words * 4);
    kv->ulen = (uint16_t*)ctx_alloc(ctx, n_rh * mt * 2 + 512);
    kv->norm = (uint16_t*)ctx_alloc(ctx, n_rh * mt * 2 + 512);
    kv->blk_off = (uint32_t*)ctx_alloc(ctx, n_rh * (kv->n_blk + 1) * 4);
    kv->upos = (uint32_t*)ctx_alloc(ctx, n_rh * 4 + 64);
    kv->ring = (__nv_bfloat16*)ctx_alloc(ctx, (size_t)2 * (cfg->window > 0 ? cfg->window : 1) * H * d * 2);
    kv->dsign = (int8_t*)ctx_alloc(ctx, d);
    kv->ssign = (int8_t*)ctx_alloc(ctx, d);
    kv->counters = (unsigned long long*)ctx_alloc(ctx, 64);
    if (cfg->rotation == HQ_ROT_QJL) {
        kv->qjl = (float*)ctx_alloc(ctx, (size_t)2 * d * d * sizeof(float));
        if (!kv->qjl) { hq_kv_free(ctx, kv); return HQ_ERR_ALLOC; }
    }
    kv->cfg.qjl_dev = nullptr;   // the cache keeps its own copy
    if (cfg->device_position) {
        kv->pos_dev = (uint32_t*)ctx_alloc(ctx, 256);
        if (!kv->pos_dev) { hq_kv_free(ctx, kv); return HQ_ERR_ALLOC; }
        cudaMemset(kv->pos_dev, 0, 256);
    }
    kv->att_ws_bytes = attend_workspace_bytes(ctx, kv);
    kv->att_ws = (float*)ctx_alloc(ctx, kv->att_ws_bytes);
    if (cudaHostAlloc((void**)&kv->flag_host, 64, cudaHostAllocMapped) != cudaSuccess ||
        cudaHostGetDevicePointer((void**)&kv->flag_dev, kv->flag_host, 0) != cudaSuccess) {
        hq_kv_free(ctx, kv);
        return fail(ctx, HQ_ERR_CUDA, "cudaHostAlloc for the cache's error flag failed");
    }
    *kv->flag_host = 0;
    if (!kv->rem || !kv->una || !kv->ulen || !kv->norm || !kv->blk_off || !kv->upos || !kv->ring || !kv->dsign ||
        !kv->ssign || !kv->counters || !kv->att_ws) {
        hq_kv_free(ctx, kv);
        return HQ_ERR_ALLOC;
    }
    cudaMemset(kv->rem, 0, n_rh * kv->rem_words * 4);
    cudaMemset(kv->una, 0, n_rh * kv->una_words * 4);
    cudaMemset(kv->ulen, 0, n_rh * mt * 2 + 512);
    cudaMemset(kv->norm, 0, n_rh * mt * 2 + 512);
    cudaMemset(kv->blk_off, 0, n_rh * (kv->n_blk + 1) * 4);
    cudaMemset(kv->upos, 0, n_rh * 4 + 64);
    cudaMemset(kv->counters, 0, 64);
    launch_signs(cfg->codec.seed, 1u, d, kv->dsign, 0);
    launch_signs(cfg->codec.seed, 2u, d, kv->ssign, 0);
    if (kv->qjl) {
        cudaMemcpyAsync(kv->qjl, cfg->qjl_dev, (size_t)d * d * sizeof(float), cudaMemcpyDeviceToDevice, 0);
        launch_transpose_f32(kv->qjl, kv->qjl + (size_t)d * d, d, 0);
    }
    cudaError_t e = cudaDeviceSynchronize();
    if (e != cudaSuccess) {
        ctx->err = cudaGetErrorString(e);
        hq_kv_free(ctx, kv);
        return HQ_ERR_CUDA;
    }
    *out = kv;
    return HQ_OK;
}

void hq_kv_free(hq_ctx* ctx, hq_kv* kv) {
    if (!kv) return;
    if (!ctx) ctx = kv->ctx;
    ctx_free(ctx, kv->rem); ctx_free(ctx, kv->una); ctx_free(ctx, kv->ulen); ctx_free(ctx, kv->norm);
    ctx_free(ctx, kv->blk_off); ctx_free(ctx, kv->upos); ctx_free(ctx, kv->ring); ctx_free(ctx, kv->dsign);
    ctx_free(ctx, kv->ssign); ctx_free(ctx, kv->qjl); ctx_free(ctx, kv->pos_dev); ctx_free(ctx, kv->counters); ctx_free(ctx, kv->scratch_codes); ctx_free(ctx, kv->att_ws);
    if (kv->flag_host) { cudaDeviceSynchronize(); cudaFreeHost(kv->flag_host); }
    delete kv;
}

hq_status hq_kv_append(hq_ctx* ctx, hq_kv* kv, const void* k_dev, const void* v_dev, int64_t n_tok, void* stream) {
    if (!ctx) return HQ_ERR_INVALID_ARG;
    if (!kv || !k_dev || !v_dev) return fail(ctx, HQ_ERR_INVALID_ARG, "null argument");
    if (kv->ctx != ctx) return fail(ctx, HQ_ERR_INVALID_ARG, "the cache belongs to another context");
    if (kv->pos_dev && n_tok > 1) {   // replays may have advanced the device's count past the host's
        HQ_ENTER(ctx);
        if (hq_status rs = kv_refresh_position(ctx, kv)) return rs;
    }
    if (n_tok <= 0 || kv->n_tokens + n_tok > kv->cfg.max_tokens) return fail(ctx, HQ_ERR_SHAPE, "n_tok out of range");
    if (hq_status fs = kv_flag_status(ctx, kv)) return fs;
    HQ_ENTER(ctx);
    cudaStream_t st = (cudaStream_t)stream;
    int H = kv->cfg.kv_heads, d = kv->cfg.head_dim;
    if (n_tok == 1) {   // the decode step: one fused launch
        launch_kv_append1(kv, k_dev, v_dev, st);
        HQ_CUDA_CHECK(ctx, cudaGetLastError());
        kv->n_tokens += 1;
        return HQ_OK;
    }
    const int64_t CHUNK = 4096;
    int64_t chunk = n_tok < CHUNK ? n_tok : CHUNK;
    if (chunk > kv->scratch_tokens) {
        if (kv->scratch_codes) { HQ_CUDA_CHECK(ctx, cudaDeviceSynchronize()); ctx_free(ctx, kv->scratch_codes); kv->scratch_codes = nullptr; }
        int64_t cap = chunk < 64 ? 64 : chunk;
        kv->scratch_codes = (int8_t*)ctx_alloc(ctx, (size_t)2 * cap * H * (d + 4));
        if (!kv->scratch_codes) { kv->scratch_tokens = 0; return HQ_ERR_ALLOC; }
        kv->scratch_tokens = cap;
    }
    int* err_flag = kv->flag_dev;
    for (int64_t c0 = 0; c0 < n_tok; c0 += chunk) {
        int64_t nt = n_tok - c0 < chunk ? n_tok - c0 : chunk;
        int64_t token0 = kv->n_tokens + c0;
        for (int role = 0; role < 2; ++role) {
            const __nv_bfloat16* src = (const __nv_bfloat16*)(role ? v_dev : k_dev) + c0 * H * d;
            int8_t* codes = kv->scratch_codes + (size_t)role * kv->scratch_tokens * H * (d + 4);
            uint16_t* norm_r = kv->norm + (int64_t)role * H * kv->cfg.max_tokens;
            launch_quantize_kv(src, nt, H, d, token0, role, kv->cfg.codec.lattice, kv->A, kv->cfg.rotation,
                               kv->cfg.dither, kv->cfg.codec.seed, kv->dsign, kv->ssign, codes, norm_r,
                               kv->cfg.max_tokens, kv->counters, st, kv->qjl ? kv->qjl + (size_t)d * d : nullptr);
            launch_kv_pack(codes, nt, H, d, token0, role, kv->cfg.codec.lattice, kv->k0, kv->k1, kv->rbits,
                           kv->cfg.max_tokens, kv->rem_words, kv->una_words, kv->n_blk, kv->rem, kv->una, kv->ulen,
                           kv->blk_off, kv->upos, err_flag, st);
        }
    }
    launch_kv_ring(k_dev, v_dev, n_tok, H, d, kv->n_tokens, kv->cfg.window, kv->ring, st);
    HQ_CUDA_CHECK(ctx, cudaGetLastError());
    kv->n_tokens += n_tok;
    if (kv->pos_dev) {
        launch_set_u32(kv->pos_dev, (uint32_t)kv->n_tokens, st);
        HQ_CUDA_CHECK(ctx, cudaGetLastError());
    }
    return HQ_OK;
}

hq_status hq_attend(hq_ctx* ctx, const hq_kv* kv, const void* q_dev, int32_t q_heads, void* out_bf16_dev,
                    float* out_f32_dev_or_null, void* stream) {
    if (!ctx) return HQ_ERR_INVALID_ARG;
    if (!kv || !q_dev || (!out_bf16_dev && !out_f32_dev_or_null)) return fail(ctx, HQ_ERR_INVALID_ARG, "null argument");
    if (q_heads <= 0 || q_heads % kv->cfg.kv_heads != 0 || q_heads / kv->cfg.kv_heads > 8 || q_heads > 64)
        return fail(ctx, HQ_ERR_SHAPE, "q_heads must be a multiple of kv_heads, group size <= 8, q_heads <= 64");
    if (kv->n_tokens <= 0 && !kv->pos_dev) return fail(ctx, HQ_ERR_SHAPE, "empty cache");
    if (kv->ctx != ctx) return fail(ctx, HQ_ERR_INVALID_ARG, "the cache belongs to another context");
    if (hq_status fs = kv_flag_status(ctx, kv)) return fs;
    HQ_ENTER(ctx);
    return launch_attend(ctx, kv, q_dev, q_heads, out_bf16_dev, out_f32_dev_or_null, (cudaStream_t)stream);
}

hq_status hq_kv_sync_position(hq_ctx* ctx, hq_kv* kv, int64_t* n_tokens_out) {
    if (!ctx) return HQ_ERR_INVALID_ARG;
    if (!kv) return fail(ctx, HQ_ERR_INVALID_ARG, "null argument");
    if (kv->ctx != ctx) return fail(ctx, HQ_ERR_INVALID_ARG, "the cache belongs to another context");
    HQ_ENTER(ctx);
    if (hq_status rs = kv_refresh_position(ctx, kv)) return rs;
    if (n_tokens_out) *n_tokens_out = kv->n_tokens;
    return kv_flag_status(ctx, kv);
}

hq_status hq_kv_export(hq_ctx* ctx, const hq_kv* kv, hq_kv_view* out) {
    if (!ctx) return HQ_ERR_INVALID_ARG;
    if (!kv || !out) return fail(ctx, HQ_ERR_INVALID_ARG, "null argument");
    HQ_ENTER(ctx);
    if (hq_status rs = kv_refresh_position(ctx, const_cast<hq_kv*>(kv))) return rs;
    HQ_CUDA_CHECK(ctx, cudaDeviceSynchronize());
    unsigned long long hc[8];
    HQ_CUDA_CHECK(ctx, cudaMemcpy(hc, kv->counters, sizeof(hc), cudaMemcpyDeviceToHost));
    if (hq_status fs = kv_flag_status(ctx, kv)) return fs;
    out->n_tokens = kv->n_tokens; out->rbits = kv->rbits;
    out->rem_dev = kv->rem; out->una_dev = kv->una; out->ulen_dev = kv->ulen; out->norm_dev = kv->norm;
    out->blk_off_dev = kv->blk_off; out->upos_dev = kv->upos;
    out->rem_words = kv->rem_words; out->una_words = kv->una_words;
    out->clamp_count = (int64_t)hc[0];
    return HQ_OK;
}

hq_status hq_kv_decode_int8(hq_ctx* ctx, const hq_kv* kv, int32_t role, int64_t t0, int64_t n, int8_t* codes_dev,
                            void* stream) {
    if (!ctx) return HQ_ERR_INVALID_ARG;
    if (!kv || !codes_dev || role < 0 || role > 1) return fail(ctx, HQ_ERR_INVALID_ARG, "bad argument");
    if (kv->pos_dev) {
        HQ_ENTER(ctx);
        if (hq_status rs = kv_refresh_position(ctx, const_cast<hq_kv*>(kv))) return rs;
    }
    if (t0 < 0 || n <= 0 || t0 + n > kv->n_tokens) return fail(ctx, HQ_ERR_SHAPE, "token range out of bounds");
    if (hq_status fs = kv_flag_status(ctx, kv)) return fs;
    HQ_ENTER(ctx);
    launch_kv_decode_int8(kv, role, t0, n, codes_dev, (cudaStream_t)stream);
    HQ_CUDA_CHECK(ctx, cudaGetLastError());
    return HQ_OK;
}

}  // extern "C"
