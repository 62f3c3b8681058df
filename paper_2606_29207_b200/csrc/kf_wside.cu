// kf_wside.cu -- C ABI of the W-node stages (kf_wside_*, kf_w_*) and of the M-microbatch inter-layer kernel pipeline
// (kf_pipeline_step).  Argument checking, tensor-map encoding, launches, stream/event plumbing; the
// arithmetic is in kf_wgemm.cu (tcgen05 GEMM) and in the attend kernels.
#include <stdio.h>
#include <string.h>

#include <new>

#include "kf_ctx.h"
#include "kf_wside.cuh"

using namespace kf;

struct kf_wside {
    kf_wside_config cfg;
    unsigned char *weights;
    // workspace slices
    __half *o16, *y, *h;      // [B][Hq*d], [B][hidden], [B][ffn]
    float *partial;
    CUtensorMap *maps;        // [L][5] weight maps (host copies, passed to kernels by value)
    // activation maps already encoded, direct-mapped by address: a decode loop presents the same few buffers (x, o16, y,
    // h per microbatch) at every layer, and cuTensorMapEncodeTiled is a driver call on the launch path.  A map is a pure
    // function of its key (address, rows, cols, box rows), so an entry can never go stale.
    struct XMap {
        const void *base;
        int rows, cols, box;
        CUtensorMap map;
    };
    static constexpr int kXMaps = 32;
    XMap xmaps[kXMaps];
    cudaEvent_t ev[64];       // cross-stream dependencies of kf_pipeline_step
    int n_ev;
    int n_ctas;               // persistent GEMM grid (<= SM count; kf_wside_set_sms)
    int sm_count;
    int64_t launches;
    char cuda_err[256];
};

namespace {

constexpr int kMatQ = 0, kMatKV = 1, kMatO = 2, kMatGU = 3, kMatD = 4;

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encoder() {
    static EncodeTiledFn fn = [] {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
            q != cudaDriverEntryPointSuccess) {
            cudaGetLastError();
            p = nullptr;
        }
        return (EncodeTiledFn)p;
    }();
    return fn;
}

bool valid(const kf_wside_config *c) {
    if (!c) return false;
    if (c->head_dim != 128 || c->n_q_heads < 1 || c->n_kv_heads < 1 || c->n_q_heads % c->n_kv_heads) return false;
    if (c->hidden < 128 || c->hidden % 128 || c->ffn < 128 || c->ffn % 128) return false;
    if (c->n_layers < 1 || c->max_batch < 1 || c->max_batch > kWgMaxBatch) return false;
    return true;
}
size_t rows_of(const kf_wside_config *c, int m) {
    const size_t qd = (size_t)c->n_q_heads * 128, kvd = (size_t)c->n_kv_heads * 128;
    switch (m) {
        case kMatQ: return qd;
        case kMatKV: return 2 * kvd;
        case kMatO: return c->hidden;
        case kMatGU: return 2 * (size_t)c->ffn;
        default: return c->hidden;
    }
}
size_t cols_of(const kf_wside_config *c, int m) {
    switch (m) {
        case kMatO: return (size_t)c->n_q_heads * 128;
        case kMatD: return c->ffn;
        default: return c->hidden;
    }
}
size_t layer_bytes(const kf_wside_config *c) {
    size_t b = 0;
    for (int m = 0; m < 5; ++m) b += rows_of(c, m) * cols_of(c, m) * 2;
    return b;
}
size_t mat_offset(const kf_wside_config *c, int layer, int m) {
    size_t b = (size_t)layer * layer_bytes(c);
    for (int i = 0; i < m; ++i) b += rows_of(c, i) * cols_of(c, i) * 2;
    return b;
}
inline size_t up(size_t x) { return (x + 255) / 256 * 256; }
int nb_of(int batch) { return batch <= 16 ? 16 : batch <= 32 ? 32 : batch <= 64 ? 64 : 128; }
size_t partial_floats(const kf_wside_config *) {
    // every CTA of the persistent grid owns two slots of one (dual) accumulator tile [2][NB = 128][128] fp32
    return (size_t)kWgMaxCtas * 2 * 2 * kWgMaxBatch * kWgTileN;
}

int fail(kf_wside *w, cudaError_t e) {
    snprintf(w->cuda_err, sizeof(w->cuda_err), "%s: %s", cudaGetErrorName(e), cudaGetErrorString(e));
    return KF_ECUDA;
}

int encode(kf_wside *w, CUtensorMap *map, const void *base, size_t rows, size_t cols, int box_rows) {
    EncodeTiledFn enc = encoder();
    if (!enc) {
        snprintf(w->cuda_err, sizeof(w->cuda_err), "cuTensorMapEncodeTiled entry point unavailable");
        return KF_ECUDA;
    }
    const cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
    const cuuint64_t strides[1] = {(cuuint64_t)cols * 2};
    const cuuint32_t box[2] = {(cuuint32_t)kWgBK, (cuuint32_t)box_rows};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, const_cast<void *>(base), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(w->cuda_err, sizeof(w->cuda_err), "cuTensorMapEncodeTiled failed: CUresult %d", (int)r);
        return KF_ECUDA;
    }
    return KF_OK;
}

// out segments [0, e0) -> o0, [e0, e1) -> o1: one GEMM x [B][K] . W(m)^T
int gemm(kf_wside *w, int layer, int m, const void *x, int batch, __half *o0, int ld0, int e0, __half *o1, int ld1,
         cudaStream_t s, bool pdl = true) {
    const kf_wside_config *c = &w->cfg;
    const bool dual = m == kMatGU;
    const int K = (int)cols_of(c, m);
    const int N = dual ? c->ffn : (int)rows_of(c, m);
    const int nb = nb_of(batch);
    kf_wside::XMap &xm = w->xmaps[((uintptr_t)x >> 8) % kf_wside::kXMaps];
    int rc = KF_OK;
    if (xm.base != x || xm.rows != batch || xm.cols != K || xm.box != nb) {
        xm.base = nullptr;
        rc = encode(w, &xm.map, x, (size_t)batch, (size_t)K, nb);  // rows >= batch of the box are zero-filled by TMA
        if (rc != KF_OK) return rc;
        xm.base = x;
        xm.rows = batch;
        xm.cols = K;
        xm.box = nb;
    }
    const CUtensorMap &tmX = xm.map;
    WGemmArgs a;
    memset(&a, 0, sizeof(a));
    a.K = K;
    a.N = N;
    a.B = batch;
    a.nkb = K / kWgBK;
    a.n_ctas = w->n_ctas;
    a.seg_end[0] = e0;
    a.seg_end[1] = N;
    a.seg_end[2] = N;
    a.out[0] = o0;
    a.ld[0] = ld0;
    a.out[1] = o1 ? o1 : o0;
    a.ld[1] = o1 ? ld1 : ld0;
    a.out[2] = a.out[1];
    a.ld[2] = a.ld[1];
    a.partial = w->partial;
    a.up_row_offset = dual ? c->ffn : 0;
    rc = launch_wgemm(w->maps[layer * 5 + m], tmX, a, nb, dual, pdl, s);
    if (rc < 0) {
        if (rc == KF_ECUDA) fail(w, cudaGetLastError());  // a launch or its set-up was refused: keep the runtime's text
        return rc;
    }
    w->launches += rc;
    const cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(w, e);
    }
    return KF_OK;
}

bool bad_call(const kf_wside *w, int layer, int batch) {
    return !w || layer < 0 || layer >= w->cfg.n_layers || batch < 1 || batch > w->cfg.max_batch;
}

}  // namespace

extern "C" {

size_t kf_wside_weight_bytes(const kf_wside_config *cfg) { return valid(cfg) ? layer_bytes(cfg) * cfg->n_layers : 0; }

size_t kf_wside_weight_offset(const kf_wside_config *cfg, int32_t layer, int32_t which) {
    if (!valid(cfg) || layer < 0 || layer >= cfg->n_layers || which < KF_W_Q || which > KF_W_DOWN) return (size_t)-1;
    // KF_W_Q, KF_W_KV, KF_W_O, KF_W_GATE, KF_W_UP, KF_W_DOWN
    switch (which) {
        case KF_W_Q: return mat_offset(cfg, layer, kMatQ);
        case KF_W_KV: return mat_offset(cfg, layer, kMatKV);
        case KF_W_O: return mat_offset(cfg, layer, kMatO);
        case KF_W_GATE: return mat_offset(cfg, layer, kMatGU);
        case KF_W_UP: return mat_offset(cfg, layer, kMatGU) + (size_t)cfg->ffn * cfg->hidden * 2;
        default: return mat_offset(cfg, layer, kMatD);
    }
}

size_t kf_wside_workspace_bytes(const kf_wside_config *c) {
    if (!valid(c)) return 0;
    const size_t B = c->max_batch;
    return up(B * c->n_q_heads * 128 * 2) + up(B * c->hidden * 2) + up(B * (size_t)c->ffn * 2) + up(partial_floats(c) * 4);
}

int kf_wside_create(kf_wside **out, const kf_wside_config *cfg, void *weights, void *workspace, size_t workspace_bytes) {
    if (!out) return KF_EINVAL;
    *out = nullptr;
    if (!valid(cfg) || !weights || !workspace || ((uintptr_t)weights & 1023) || ((uintptr_t)workspace & 255) ||
        workspace_bytes < kf_wside_workspace_bytes(cfg))
        return KF_EINVAL;
    kf_wside *w = new (std::nothrow) kf_wside();
    if (!w) return KF_EINVAL;
    memset(w, 0, sizeof(*w));
    w->cfg = *cfg;
    w->weights = (unsigned char *)weights;
    *out = w;  // returned even on KF_ECUDA so that kf_wside_last_error() can be read; the caller destroys it
    unsigned char *ws = (unsigned char *)workspace;
    const size_t B = cfg->max_batch;
    w->o16 = (__half *)ws;
    ws += up(B * cfg->n_q_heads * 128 * 2);
    w->y = (__half *)ws;
    ws += up(B * cfg->hidden * 2);
    w->h = (__half *)ws;
    ws += up(B * (size_t)cfg->ffn * 2);
    w->partial = (float *)ws;
    cudaError_t e = cudaSuccess;
    w->maps = new (std::nothrow) CUtensorMap[(size_t)cfg->n_layers * 5];
    if (!w->maps) return KF_EINVAL;
    for (int l = 0; l < cfg->n_layers; ++l)
        for (int m = 0; m < 5; ++m) {
            const int rc = encode(w, &w->maps[l * 5 + m], w->weights + mat_offset(cfg, l, m), rows_of(cfg, m),
                                  cols_of(cfg, m), kWgTileN);
            if (rc != KF_OK) return rc;
        }
    int dev_id = 0;
    cudaDeviceProp prop;
    e = cudaGetDevice(&dev_id);
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, dev_id);
    if (e != cudaSuccess) return fail(w, e);
    w->sm_count = prop.multiProcessorCount < kWgMaxCtas ? prop.multiProcessorCount : kWgMaxCtas;
    w->n_ctas = w->sm_count;
    w->n_ev = 64;
    for (int i = 0; i < w->n_ev; ++i) {
        e = cudaEventCreateWithFlags(&w->ev[i], cudaEventDisableTiming);
        if (e != cudaSuccess) {
            w->n_ev = i;
            return fail(w, e);
        }
    }
    return KF_OK;
}

int kf_wside_destroy(kf_wside *w) {
    if (!w) return KF_EINVAL;
    for (int i = 0; i < w->n_ev; ++i) cudaEventDestroy(w->ev[i]);
    delete[] w->maps;
    delete w;
    return KF_OK;
}

int kf_wside_set_sms(kf_wside *w, int32_t n_sms) {
    if (!w || n_sms < 0) return KF_EINVAL;
    w->n_ctas = n_sms == 0 || n_sms > w->sm_count ? w->sm_count : n_sms;
    return KF_OK;
}

const char *kf_wside_last_error(const kf_wside *w) { return w ? w->cuda_err : ""; }
int64_t kf_wside_launch_count(const kf_wside *w) { return w ? w->launches : 0; }

int kf_w_project_q(kf_wside *w, int32_t layer, const void *x, int32_t batch, void *q, kf_stream stream) {
    if (bad_call(w, layer, batch) || !x || !q || ((uintptr_t)x & 15) || ((uintptr_t)q & 15)) return KF_EINVAL;
    const int qd = w->cfg.n_q_heads * 128;
    return gemm(w, layer, kMatQ, x, batch, (__half *)q, qd, qd, nullptr, 0, (cudaStream_t)stream);
}

int kf_w_project_kv(kf_wside *w, int32_t layer, const void *x, int32_t batch, void *k_new, void *v_new, kf_stream stream) {
    if (bad_call(w, layer, batch) || !x || !k_new || !v_new || (((uintptr_t)x | (uintptr_t)k_new | (uintptr_t)v_new) & 15))
        return KF_EINVAL;
    const int kvd = w->cfg.n_kv_heads * 128;
    return gemm(w, layer, kMatKV, x, batch, (__half *)k_new, kvd, kvd, (__half *)v_new, kvd, (cudaStream_t)stream);
}

int kf_w_post_attention(kf_wside *w, int32_t layer, const float *o, int32_t batch, void *x_next, kf_stream stream) {
    if (bad_call(w, layer, batch) || !o || !x_next || (((uintptr_t)o | (uintptr_t)x_next) & 15)) return KF_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    const kf_wside_config *c = &w->cfg;
    const int qd = c->n_q_heads * 128;
    launch_cast_o(o, w->o16, (size_t)batch * qd, s);
    w->launches += 1;
    // every GEMM is a programmatic dependent launch (kf_wgemm.cu): before its griddepcontrol.wait it touches no global
    // memory, so this is safe behind any kernel; the cast kernel has no such wait and is launched normally
    int rc = gemm(w, layer, kMatO, w->o16, batch, w->y, c->hidden, c->hidden, nullptr, 0, s, true);
    if (rc == KF_OK) rc = gemm(w, layer, kMatGU, w->y, batch, w->h, c->ffn, c->ffn, nullptr, 0, s, true);
    if (rc == KF_OK) rc = gemm(w, layer, kMatD, w->h, batch, (__half *)x_next, c->hidden, c->hidden, nullptr, 0, s, true);
    return rc;
}

// ---- M-microbatch inter-layer kernel pipeline (Fig. 7) -------------------------------------------
int kf_pipeline_step(kf_wside *w, kf_ctx *const *ctxs, int32_t n_micro, int32_t n_layers, const int32_t *layers,
                     void *const *x, void *const *q, void *const *k_new, void *const *v_new, float *const *o,
                     float *const *lse, int32_t pipelined, kf_stream w_stream, kf_stream a_stream) {
    if (!w || !ctxs || n_micro < 1 || n_micro > 8 || n_layers < 1 || !layers || !x || !q || !k_new || !v_new || !o || !lse ||
        !w_stream || !a_stream)
        return KF_EINVAL;
    if (pipelined && w_stream == a_stream) return KF_EINVAL;
    for (int m = 0; m < n_micro; ++m)
        if (!ctxs[m] || !x[m] || !q[m] || !k_new[m] || !v_new[m] || !o[m] || !lse[m] || ctxs[m]->cfg.max_requests > w->cfg.max_batch ||
            ctxs[m]->cfg.n_q_heads != w->cfg.n_q_heads || ctxs[m]->cfg.n_kv_heads != w->cfg.n_kv_heads)
            return KF_EINVAL;
    for (int l = 0; l < n_layers; ++l)
        if (layers[l] < 0 || layers[l] >= w->cfg.n_layers) return KF_EINVAL;
    cudaStream_t ws = (cudaStream_t)w_stream, as = pipelined ? (cudaStream_t)a_stream : ws;
    int rc = KF_OK;
    // cross-stream dependencies: one "projection done" and one "attention done" event per microbatch, re-recorded every
    // layer (a wait refers to the record that precedes it in host order, so re-recording later is safe)
    auto record = [&](int idx, cudaStream_t on) {
        if (rc != KF_OK || ws == as) return;
        const cudaError_t ce = cudaEventRecord(w->ev[idx], on);
        if (ce != cudaSuccess) rc = fail(w, ce);
    };
    auto wait = [&](int idx, cudaStream_t on) {
        if (rc != KF_OK || ws == as) return;
        const cudaError_t ce = cudaStreamWaitEvent(on, w->ev[idx], 0);
        if (ce != cudaSuccess) rc = fail(w, ce);
    };
    auto B = [&](int m) { return ctxs[m]->cfg.max_requests; };
    auto proj = [&](int m, int l) {
        if (rc != KF_OK) return;
        rc = kf_w_project_q(w, layers[l], x[m], B(m), q[m], (kf_stream)ws);  // Q first
        if (rc == KF_OK) rc = kf_w_project_kv(w, layers[l], x[m], B(m), k_new[m], v_new[m], (kf_stream)ws);
        record(2 * m, ws);
    };
    auto attend = [&](int m, int l) {
        wait(2 * m, as);
        if (rc != KF_OK) return;
        const int lp = layers[l] % ctxs[m]->cfg.n_layers;
        // the last layer's attend also performs the step commit a5 of its microbatch; with the TMA kernel the append
        // a2 rides in the attend launch as well
        const bool fused = ctxs[m]->impl == KF_IMPL_TMA;
        if (!fused) rc = kf_kv_append(ctxs[m], lp, k_new[m], v_new[m], (kf_stream)as);
        if (rc == KF_OK)
            rc = kf_attend_impl(ctxs[m], lp, q[m], o[m], lse[m], nullptr, nullptr, l == n_layers - 1 ? 1 : 0,
                                fused ? k_new[m] : nullptr, fused ? v_new[m] : nullptr, (kf_stream)as);
        record(2 * m + 1, as);
    };
    auto post = [&](int m, int l) {
        wait(2 * m + 1, ws);
        if (rc != KF_OK) return;
        rc = kf_w_post_attention(w, layers[l], o[m], B(m), x[m], (kf_stream)ws);
    };
    // fork: the A stream joins the step after everything enqueued on the W stream so far (this also makes the whole
    // step capturable into one CUDA graph from the W stream); joined again at the end
    record(2 * n_micro, ws);
    wait(2 * n_micro, as);
    // a1 on the A side: one token boundary per microbatch and step
    for (int m = 0; m < n_micro && rc == KF_OK; ++m) rc = kf_token_boundary(ctxs[m], (kf_stream)as);
    if (!pipelined) {
        // serial: every microbatch runs proj -> attention -> post, one after the other: T_p + T_A + T_f each
        for (int l = 0; l < n_layers; ++l)
            for (int m = 0; m < n_micro; ++m) {
                proj(m, l);
                attend(m, l);
                post(m, l);
            }
        return rc;
    }
    // pipelined (Fig. 7): W stream = proj(mu_0, 0), proj(mu_1, 0), post(mu_0, 0), proj(mu_0, 1), post(mu_1, 0), ...
    //                     A stream = attend(mu_0, 0), attend(mu_1, 0), attend(mu_0, 1), ...
    // attend(m, l) waits for proj(m, l); post(m, l) waits for attend(m, l); proj(m, l+1) follows post(m, l) on the W
    // stream.  While the A side attends one microbatch, the W side does post + projection of its neighbour.
    for (int m = 0; m < n_micro; ++m) {
        proj(m, 0);
        attend(m, 0);
    }
    for (int l = 0; l < n_layers; ++l)
        for (int m = 0; m < n_micro; ++m) {
            post(m, l);
            if (l + 1 < n_layers) {
                proj(m, l + 1);
                attend(m, l + 1);
            }
        }
    record(2 * n_micro + 1, as);  // join
    wait(2 * n_micro + 1, ws);
    return rc;
}

}  // extern "C"
