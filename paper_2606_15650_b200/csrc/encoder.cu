// encoder.cu -- parameter upload and the A1-A8 forward pass (BJ north_star ¶1; S8c O1/O2).
//
// Activation layout in HBM (per chunk of whole sequences, carved from the context workspace):
//   dtype 1 (BF16):  x  FP32 [t,H]  residual stream        xb BF16 [t,H]  GEMM operand copy of x
//                    y  FP32 [t,H]  GEMM(+bias+residual)    qkv BF16 [t,3H]   ctx BF16 [t,H]   f BF16 [t,F]
//   dtype 0 (FP32):  the same tensors, all FP32 (xb unused)
// The residual stream, LayerNorm statistics, softmax and the classifier head stay FP32 in both modes
// (S7 H2: that is what keeps BF16 logits within 3e-2 and label agreement high).
#include "common.cuh"
#include "encoder_kernels.cuh"

#include <new>
#include <vector>
#include <stdlib.h>
#include <math.h>
#include <algorithm>

struct LayerW {
    void *W_qkv, *W_o, *W_1, *W_2;                     // BF16 or FP32 matrices
    float *b_qkv, *b_o, *g_1, *b_1, *b_1f, *b_2f, *g_2, *b_2;
    // LayerNorm fold (BF16, arch 0, H = 768 / 1024): Wf_qkv = bf16(W_qkv * gamma_2 of the previous layer), s[n] = sum_k Wf[n,k],
    // c[n] = b[n] + sum_k beta_2[k] W[n,k] (layer 0 reads the normalised embedding: no fold)
    void* Wf_qkv = nullptr;
    float *s_qkv = nullptr, *c_qkv = nullptr;
};
struct anon_weights {
    anon_ctx* ctx = nullptr;
    anon_model_desc d;
    uint8_t* store = nullptr;
    void *E_w = nullptr, *E_p = nullptr;
    float *E_t = nullptr, *g_e = nullptr, *b_e = nullptr, *W_c = nullptr, *b_c = nullptr;
    // arch 1 (NEXT-3): LayerW reuses g_1 = g_a, g_2 = g_m, W_1 = W_i [2F, H]; every bias / beta / E_p / E_t points at `zeros`
    float* g_f = nullptr;
    void* zeros = nullptr;
    float2 *rope_g = nullptr, *rope_l = nullptr;       // (cos, sin) of pos * theta^(-2i/64), [max_pos][32]
    float2 *rope_gt = nullptr, *rope_lt = nullptr;     // the same, pair-major [32][512], for the QKV GEMM's RoPE epilogue
    // W_i stored with its rows interleaved per 256-row tile (128 a-rows, then their 128 gate rows) so that the FFN1 GEMM's
    // GeGLU epilogue (gemm_tcgen05.cu EPI 4) finds a and gate in the same accumulator tile
    bool geglu_fused = false;
    bool folded = false;                               // the fold's tensors were prepared (see LayerW)
    std::vector<LayerW> layers;
};

namespace {

__global__ void f32_to_bf16_kernel(const float* __restrict__ src, __nv_bfloat16* __restrict__ dst, size_t n) {
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (; i < n; i += stride) dst[i] = __float2bfloat16_rn(src[i]);
}

int check_desc(const anon_model_desc* d) {
    if (!d) return ANON_ERR_INVALID_ARG;
    if (d->layers < 0 || d->hidden <= 0 || d->heads <= 0 || d->ffn <= 0 || d->vocab <= 0 || d->num_labels <= 0 ||
        d->max_pos <= 0 || (d->dtype != 0 && d->dtype != 1))
        return ANON_ERR_INVALID_ARG;
    if (d->hidden != d->heads * 64 || d->hidden % 128 != 0 || d->hidden > 1024 || d->ffn % 64 != 0 ||
        (d->num_labels & 1) == 0 || d->num_labels > 64 || d->max_pos > 512)
        return ANON_ERR_UNSUPPORTED;
    if (d->arch != 0 && d->arch != 1) return ANON_ERR_INVALID_ARG;
    if (d->arch == 1) {
        if (d->local_window < 0 || (d->local_window & 1) || d->global_every < 1 || !(d->rope_theta_global > 0.f) ||
            !(d->rope_theta_local > 0.f))
            return ANON_ERR_INVALID_ARG;
        const bool has_local = d->global_every > 1 && d->layers > 1;
        if (d->dtype == 1 && has_local && d->local_window != 128) return ANON_ERR_UNSUPPORTED;
    }
    return ANON_OK;
}

size_t desc_floats(const anon_model_desc& d) {
    const size_t H = d.hidden, F = d.ffn, V = d.vocab, NL = d.num_labels, P = d.max_pos, L = d.layers;
    if (d.arch == 1) return V * H + H + L * (H + 3 * H * H + H * H + H + 2 * F * H + H * F) + H + NL * H + NL;
    const size_t per_layer = 3 * H * H + 3 * H + H * H + H + 2 * H + F * H + F + H * F + H + 2 * H;
    return V * H + P * H + 3 * H + L * per_layer + NL * H + NL;
}

size_t per_token_bytes(const anon_model_desc& d) {
    const size_t H = d.hidden, F = d.ffn;
    if (d.arch == 1)      // x, y, h FP32; xb; qkv; ctx; u [2F]; f [F]; position id
        return d.dtype == 1 ? 12 * H + 2 * H + 6 * H + 2 * H + 4 * F + 2 * F + 4 : 12 * H + 12 * H + 4 * H + 8 * F + 4 * F + 4;
    if (d.dtype == 1) return 4 * H + 2 * H + 4 * H + 6 * H + 2 * H + 2 * F + 8 + 64;     // + row statistics (fold: 2 x H/256 partial pairs)
    return 4 * H + 4 * H + 12 * H + 4 * H + 4 * F;
}

}  // namespace

extern "C" size_t anon_workspace_bytes(const anon_model_desc* d, int64_t max_tokens, int32_t max_seqs) {
    if (!d || max_tokens < 0 || max_seqs < 0) return 0;
    const size_t per_tok = per_token_bytes(*d) + 64;                 // + decode / gather / scan scratch per item
    return (size_t)max_tokens * per_tok + (size_t)max_seqs * 64 + ((size_t)8 << 20);
}

extern "C" int anon_weights_load(anon_ctx* ctx, const anon_model_desc* desc, const float* blob, size_t n_floats,
                                 anon_weights** out)
{
    if (!ctx || !blob || !out) return ANON_ERR_INVALID_ARG;
    int rc = check_desc(desc);
    if (rc) return rc;
    if (n_floats != desc_floats(*desc)) return ANON_ERR_INVALID_ARG;
    CU_TRY(ctx, cudaSetDevice(ctx->device));
    anon_weights* w = new (std::nothrow) anon_weights();
    if (!w) return ANON_ERR_OOM;
    w->ctx = ctx; w->d = *desc;
    const anon_model_desc& d = *desc;
    const size_t H = d.hidden, F = d.ffn, V = d.vocab, NL = d.num_labels, P = d.max_pos;
    const bool bf = d.dtype == 1;
    const size_t msz = bf ? 2 : 4;
    struct Item { void** dst; size_t n; bool matrix; bool geglu_rows = false; const float* host = nullptr; };
    std::vector<Item> items;
    w->layers.resize(d.layers);
    size_t zero_bytes = 0;
    if (d.arch == 1) {
        w->geglu_fused = bf && F % 128 == 0;
        items.push_back({&w->E_w, V * H, true});
        items.push_back({(void**)&w->g_e, H, false});
        for (int l = 0; l < d.layers; l++) {
            LayerW& L = w->layers[l];
            items.push_back({(void**)&L.g_1, H, false});    items.push_back({&L.W_qkv, 3 * H * H, true});
            items.push_back({&L.W_o, H * H, true});         items.push_back({(void**)&L.g_2, H, false});
            items.push_back({&L.W_1, 2 * F * H, true, w->geglu_fused});     items.push_back({&L.W_2, H * F, true});
        }
        items.push_back({(void**)&w->g_f, H, false});
        zero_bytes = std::max(P * H * msz, 4 * std::max(3 * H, 2 * F));
        if (F % 8) { delete w; return ANON_ERR_UNSUPPORTED; }
    } else {
    items.push_back({&w->E_w, V * H, true});
    items.push_back({&w->E_p, P * H, true});
    items.push_back({(void**)&w->E_t, H, false});
    items.push_back({(void**)&w->g_e, H, false});
    items.push_back({(void**)&w->b_e, H, false});
    for (int l = 0; l < d.layers; l++) {
        LayerW& L = w->layers[l];
        items.push_back({&L.W_qkv, 3 * H * H, true});   items.push_back({(void**)&L.b_qkv, 3 * H, false});
        items.push_back({&L.W_o, H * H, true});         items.push_back({(void**)&L.b_o, H, false});
        items.push_back({(void**)&L.g_1, H, false});    items.push_back({(void**)&L.b_1, H, false});
        items.push_back({&L.W_1, F * H, true});         items.push_back({(void**)&L.b_1f, F, false});
        items.push_back({&L.W_2, H * F, true});         items.push_back({(void**)&L.b_2f, H, false});
        items.push_back({(void**)&L.g_2, H, false});    items.push_back({(void**)&L.b_2, H, false});
    }
    }
    items.push_back({(void**)&w->W_c, NL * H, false});   // head stays FP32 (values are BF16-representable)
    items.push_back({(void**)&w->b_c, NL, false});
    // ---- LayerNorm fold: extra tensors computed here from the blob (host, double accumulation) ----
    std::vector<std::vector<float>> fold_host;
    if (d.arch == 0 && bf && (H == 768 || H == 1024) && F % 256 == 0) {
        w->folded = true;
        // blob offsets of layer l's tensors (fixed order W_qkv, b_qkv, W_o, b_o, g_1, b_1, W_1, b_1f, W_2, b_2f, g_2, b_2)
        const size_t per_layer = 3 * H * H + 3 * H + H * H + H + 2 * H + F * H + F + H * F + H + 2 * H;
        const size_t base0 = V * H + P * H + 3 * H;
        auto bf16_rne = [](float f) { uint32_t u; memcpy(&u, &f, 4); u += 0x7FFFu + ((u >> 16) & 1u); u &= 0xFFFF0000u; float r; memcpy(&r, &u, 4); return r; };
        auto fold = [&](const float* Wm, const float* bias, const float* gam, const float* bet, size_t N_, void** dW, float** ds, float** dc) {
            const size_t i0 = fold_host.size();
            fold_host.emplace_back(N_ * H); fold_host.emplace_back(N_); fold_host.emplace_back(N_);
            std::vector<float>& Wf2 = fold_host[i0]; std::vector<float>& sv2 = fold_host[i0 + 1]; std::vector<float>& cv = fold_host[i0 + 2];
            for (size_t n = 0; n < N_; n++) {
                double ss = 0.0, cc = bias[n];
                for (size_t k = 0; k < H; k++) {
                    const float v = bf16_rne(Wm[n * H + k] * gam[k]);
                    Wf2[n * H + k] = v; ss += v; cc += (double)bet[k] * Wm[n * H + k];
                }
                sv2[n] = (float)ss; cv[n] = (float)cc;
            }
            items.push_back({dW, N_ * H, true, false, Wf2.data()});
            items.push_back({(void**)ds, N_, false, false, sv2.data()});
            items.push_back({(void**)dc, N_, false, false, cv.data()});
        };
        fold_host.reserve((size_t)d.layers * 6 + 8);     // the vectors must not move: items keep pointers into them
        for (int l = 0; l < d.layers; l++) {
            const float* Lb = blob + base0 + (size_t)l * per_layer;
            const float* Wqkv = Lb;                   const float* bqkv = Wqkv + 3 * H * H;
            const float* Wo = bqkv + 3 * H;           const float* bo = Wo + H * H;
            const float* g1 = bo + H;                 const float* b1 = g1 + H;
            const float* W1 = b1 + H;                 const float* b1f = W1 + F * H;
            LayerW& L = w->layers[l];
            (void)W1; (void)b1f; (void)g1; (void)b1;
            if (l > 0) {
                const float* Pb = blob + base0 + (size_t)(l - 1) * per_layer;
                const float* g2 = Pb + per_layer - 2 * H;  const float* b2 = g2 + H;
                fold(Wqkv, bqkv, g2, b2, 3 * H, &L.Wf_qkv, &L.s_qkv, &L.c_qkv);
            }
        }
    }
    size_t total = 0, max_matrix = 0;
    for (auto& it : items) {
        total = (total + 255) / 256 * 256 + it.n * (it.matrix ? msz : 4);
        if (it.matrix && bf && it.n > max_matrix) max_matrix = it.n;
    }
    float* stage = nullptr;
    const size_t zero_off = (total + 255) / 256 * 256;
    const size_t rope_off = (zero_off + zero_bytes + 255) / 256 * 256, rope_bytes = d.arch == 1 ? P * 32 * sizeof(float2) : 0;
    const size_t ropet_off = (rope_off + 2 * rope_bytes + 255) / 256 * 256, ropet_bytes = d.arch == 1 ? 32 * 512 * sizeof(float2) : 0;
    total = ropet_off + 2 * ropet_bytes;
    cudaError_t e = cudaMalloc(&w->store, total + 256);
    if (e == cudaSuccess && max_matrix) e = cudaMalloc(&stage, max_matrix * 4);
    if (e != cudaSuccess) { cudaFree(w->store); delete w; cuda_fail(ctx, e, "cudaMalloc(weights)"); return ANON_ERR_OOM; }
    size_t off = 0;
    const float* src = blob;
    for (auto& it : items) {
        off = (off + 255) / 256 * 256;
        void* dst = w->store + off;
        *it.dst = dst;
        std::vector<float> perm;
        const float* from = it.host ? it.host : src;
        if (it.geglu_rows) {                         // tile k: a-rows [128k, 128k + 128), then gate rows F + [128k, 128k + 128)
            perm.resize(it.n);
            for (size_t k = 0; k < F / 128; k++)
                for (size_t r = 0; r < 128; r++) {
                    memcpy(&perm[((2 * k) * 128 + r) * H], src + (k * 128 + r) * H, H * 4);
                    memcpy(&perm[((2 * k + 1) * 128 + r) * H], src + (F + k * 128 + r) * H, H * 4);
                }
            from = perm.data();
        }
        if (it.matrix && bf) {
            e = cudaMemcpyAsync(stage, from, it.n * 4, cudaMemcpyHostToDevice, ctx->stream);
            if (e == cudaSuccess) {
                f32_to_bf16_kernel<<<1024, 256, 0, ctx->stream>>>(stage, (__nv_bfloat16*)dst, it.n);
                e = cudaStreamSynchronize(ctx->stream);      // stage is reused by the next matrix
            }
        } else {
            e = cudaMemcpyAsync(dst, from, it.n * 4, cudaMemcpyHostToDevice, ctx->stream);
        }
        if (e != cudaSuccess) break;
        off += it.n * (it.matrix ? msz : 4);
        if (!it.host) src += it.n;
    }
    if (e == cudaSuccess && zero_bytes) {
        e = cudaMemsetAsync(w->store + zero_off, 0, zero_bytes, ctx->stream);
        w->zeros = w->store + zero_off;
        w->E_p = w->zeros; w->E_t = (float*)w->zeros; w->b_e = (float*)w->zeros;
        for (auto& L : w->layers) L.b_qkv = L.b_o = L.b_1 = L.b_1f = L.b_2f = L.b_2 = (float*)w->zeros;
    }
    if (e == cudaSuccess && rope_bytes) {
        std::vector<float2> tab(2 * P * 32);
        for (int which = 0; which < 2; which++) {
            const double theta = which ? d.rope_theta_local : d.rope_theta_global;
            for (size_t p = 0; p < P; p++)
                for (int i = 0; i < 32; i++) {
                    const double ang = (double)p * pow(theta, -2.0 * i / 64.0);
                    tab[(which * P + p) * 32 + i] = make_float2((float)cos(ang), (float)sin(ang));
                }
        }
        w->rope_g = (float2*)(w->store + rope_off);
        w->rope_l = w->rope_g + P * 32;
        e = cudaMemcpyAsync(w->rope_g, tab.data(), 2 * rope_bytes, cudaMemcpyHostToDevice, ctx->stream);
        std::vector<float2> tabt(2 * 32 * 512, make_float2(1.f, 0.f));
        for (int which = 0; which < 2; which++)
            for (size_t p = 0; p < P; p++)
                for (int i = 0; i < 32; i++) tabt[(which * 32 + i) * 512 + p] = tab[(which * P + p) * 32 + i];
        w->rope_gt = (float2*)(w->store + ropet_off);
        w->rope_lt = w->rope_gt + 32 * 512;
        if (e == cudaSuccess) e = cudaMemcpyAsync(w->rope_gt, tabt.data(), 2 * ropet_bytes, cudaMemcpyHostToDevice, ctx->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);          // the tables die at the end of this block
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    cudaFree(stage);
    if (e != cudaSuccess) { cudaFree(w->store); delete w; return cuda_fail(ctx, e, "weights upload"); }
    *out = w;
    return ANON_OK;
}

extern "C" void anon_weights_free(anon_weights* w) {
    if (!w) return;
    cudaFree(w->store);
    delete w;
}

const anon_model_desc* weights_desc(const anon_weights* w) { return &w->d; }

// K4 launcher: compile-time row length for the BF16 shapes (H = 768, 1024), generic kernel otherwise
static void launch_layer_norm(cudaStream_t st, unsigned grid, const float* y, int nt, int H, const float* g, const float* b,
                              float eps, float* x, __nv_bfloat16* xb, float2* stats = nullptr)
{
    if (xb && H == 768) enc::layer_norm_fixed_kernel<6><<<grid, enc::kRowWarps * 32, 0, st>>>(y, nt, g, b, eps, x, xb, stats);
    else if (xb && H == 1024) enc::layer_norm_fixed_kernel<8><<<grid, enc::kRowWarps * 32, 0, st>>>(y, nt, g, b, eps, x, xb, stats);
    else enc::layer_norm_kernel<<<grid, enc::kRowWarps * 32, 0, st>>>(y, nullptr, nt, H, g, b, eps, x, xb);
}

template <int EPI>
static int sgemm(anon_ctx* ctx, const float* A, const float* W, const float* bias, const float* res, float* C, int M, int N, int K) {
    if (M == 0) return ANON_OK;
    dim3 grid((N + 63) / 64, (M + 63) / 64);
    enc::sgemm_tn_kernel<EPI><<<grid, 256, 0, ctx->stream>>>(A, W, bias, res, C, M, N, K);
    CU_LAUNCH_CHECK(ctx, "sgemm_tn_kernel");
    return ANON_OK;
}

// ---- NEXT-3: one chunk of the ModernBERT-shaped forward (reading D20; oracle/encoder_modern.py) ---------------------
// x is the FP32 residual stream (never normalised in place): h / xb = LN(x) feed the GEMMs, the residual GEMM epilogue
// writes x + (...) into the other buffer of the x / y pair.
static int modern_chunk(anon_ctx* ctx, WsCursor c, const anon_weights* w, const int32_t* d_ids, const int32_t* d_cu, const int32_t* h_cu,
                        int B, int s0, int s1, float* d_logits, int32_t* d_labels)
{
    const anon_model_desc& d = w->d;
    const int H = d.hidden, F = d.ffn, NL = d.num_labels;
    const bool bf = d.dtype == 1;
    const int tok0 = h_cu[s0], nt = h_cu[s1] - tok0, nb = s1 - s0;
    cudaStream_t st = ctx->stream;
    const size_t es = bf ? 2 : 4;
    float* x = (float*)c.take((size_t)nt * H * 4);
    float* y = (float*)c.take((size_t)nt * H * 4);
    float* h = (float*)c.take((size_t)nt * H * 4);
    __nv_bfloat16* xb = bf ? (__nv_bfloat16*)c.take((size_t)nt * H * 2) : nullptr;
    void* qkv = c.take((size_t)nt * 3 * H * es);
    void* cx = c.take((size_t)nt * H * es);
    void* u = c.take((size_t)nt * 2 * F * es);
    void* f = c.take((size_t)nt * F * es);
    int* pos = (int*)c.take((size_t)nt * 4);
    if (!x || !y || !h || (bf && !xb) || !qkv || !cx || !u || !f || !pos) return ANON_ERR_OOM;
    const bool has_local = d.global_every > 1 && d.layers > 1;
    AttnPlan plan_g, plan_l;
    int rc = attention_plan(ctx, c, h_cu + s0, nb, d.dtype, &plan_g, 0);
    if (rc) return rc;
    plan_l = plan_g;
    if (has_local) { rc = attention_plan(ctx, c, h_cu + s0, nb, d.dtype, &plan_l, d.local_window); if (rc) return rc; }
    double fl_g = 0, fl_l = 0;                       // 4 n k d per (sequence, head), k = keys a query sees
    for (int s = s0; s < s1; s++) {
        const double n = h_cu[s + 1] - h_cu[s];
        fl_g += 4.0 * n * n * H;
        fl_l += 4.0 * n * std::min(n, (double)d.local_window + 1.0) * H;
    }
    const unsigned row_grid = (unsigned)((nt + enc::kRowWarps - 1) / enc::kRowWarps);
    const bool fixed_ln = bf && (H == 768 || H == 1024);
    const float* zf = (const float*)w->zeros;
    auto norm = [&](const float* in, const float* g, float* out32) {      // (out32, xb) = LN(in; g)
        ProfScope ps(ctx, PROF_ROW, (double)nt * H * (4 + (out32 ? 4 : 0) + (bf ? 2 : 0)));
        launch_layer_norm(st, row_grid, in, nt, H, g, zf, d.ln_eps, out32, xb);
    };
    auto gemm = [&](int cls, const void* A, const void* W, const float* res, void* C, int N, int K, int epi) -> int {
        ProfScope ps(ctx, cls, 2.0 * nt * N * K);
        if (bf) return gemm_bf16_impl(ctx, (const __nv_bfloat16*)A, (const __nv_bfloat16*)W, zf, res, C, nt, N, K, epi);
        return epi == 2 ? sgemm<2>(ctx, (const float*)A, (const float*)W, zf, res, (float*)C, nt, N, K)
                        : sgemm<0>(ctx, (const float*)A, (const float*)W, zf, res, (float*)C, nt, N, K);
    };
    { ProfScope ps(ctx, PROF_ROW, (double)nt * (4 + H * es + H * 4 + 4), 2);
    if (bf)
        enc::embed_ln_kernel<__nv_bfloat16><<<row_grid, enc::kRowWarps * 32, 0, st>>>(
            d_ids, d_cu, B, tok0, nt, (const __nv_bfloat16*)w->E_w, (const __nv_bfloat16*)w->E_p, w->E_t, w->g_e, w->b_e, d.ln_eps, H,
            d.vocab, d.max_pos, x, xb, ctx->d_status);
    else
        enc::embed_ln_kernel<float><<<row_grid, enc::kRowWarps * 32, 0, st>>>(
            d_ids, d_cu, B, tok0, nt, (const float*)w->E_w, (const float*)w->E_p, w->E_t, w->g_e, w->b_e, d.ln_eps, H, d.vocab,
            d.max_pos, x, nullptr, ctx->d_status);
    enc::token_pos_kernel<<<(unsigned)((nt + 255) / 256), 256, 0, st>>>(d_cu + s0, nb, tok0, nt, pos); }
    CU_LAUNCH_CHECK(ctx, "embed_ln_kernel");
    const void* gin = bf ? (const void*)xb : (const void*)h;             // the GEMM operand copy of LN(x)
    const long long rope_threads = (long long)nt * 2 * (H / 64) * (bf ? 4 : 8);
    for (int l = 0; l < d.layers; l++) {
        const LayerW& L = w->layers[l];
        const bool glob = !has_local || l % d.global_every == 0;
        norm(x, L.g_1, fixed_ln ? nullptr : h);
        CU_LAUNCH_CHECK(ctx, "layer_norm_kernel");
        if (bf && H % 64 == 0 && 3 * H > 128) {          // RoPE in the QKV GEMM's epilogue
            ProfScope ps(ctx, PROF_GEMM, 2.0 * nt * 3 * H * H);
            rc = gemm_bf16_rope_impl(ctx, xb, (const __nv_bfloat16*)L.W_qkv, pos, glob ? w->rope_gt : w->rope_lt, qkv, nt, 3 * H, H);
            if (rc) return rc;
        } else {
        if ((rc = gemm(PROF_GEMM, gin, L.W_qkv, nullptr, qkv, 3 * H, H, 0))) return rc;
        { ProfScope ps(ctx, PROF_ROW, (double)nt * 2 * H * es * 2);
        const float2* tab = glob ? w->rope_g : w->rope_l;
        if (bf) enc::rope_kernel<__nv_bfloat16><<<(unsigned)((rope_threads + 255) / 256), 256, 0, st>>>((__nv_bfloat16*)qkv, pos, nt, H, tab);
        else enc::rope_kernel<float><<<(unsigned)((rope_threads + 255) / 256), 256, 0, st>>>((float*)qkv, pos, nt, H, tab); }
        CU_LAUNCH_CHECK(ctx, "rope_kernel");
        }
        { ProfScope ps(ctx, PROF_ATTN, glob ? fl_g : fl_l);
        rc = attention_run(ctx, glob ? plan_g : plan_l, qkv, d_cu + s0, tok0, nb, H, d.heads, d.dtype, cx); }
        if (rc) return rc;
        if ((rc = gemm(PROF_GEMM_OUT, cx, L.W_o, x, y, H, H, 2))) return rc;
        std::swap(x, y);
        norm(x, L.g_2, fixed_ln ? nullptr : h);
        CU_LAUNCH_CHECK(ctx, "layer_norm_kernel");
        if (w->geglu_fused) {
            if ((rc = gemm(PROF_GEMM_FFN1, gin, L.W_1, nullptr, f, 2 * F, H, 4))) return rc;
        } else {
        if ((rc = gemm(PROF_GEMM_FFN1, gin, L.W_1, nullptr, u, 2 * F, H, 0))) return rc;
        { ProfScope ps(ctx, PROF_ROW, (double)nt * 3 * F * es);
        const long long vecs = (long long)nt * F / (bf ? 8 : 4);
        if (bf) enc::geglu_kernel<__nv_bfloat16><<<(unsigned)((vecs + 255) / 256), 256, 0, st>>>((const __nv_bfloat16*)u, (__nv_bfloat16*)f, nt, F);
        else enc::geglu_kernel<float><<<(unsigned)((vecs + 255) / 256), 256, 0, st>>>((const float*)u, (float*)f, nt, F); }
        CU_LAUNCH_CHECK(ctx, "geglu_kernel");
        }
        if ((rc = gemm(PROF_GEMM_FFN2, f, L.W_2, x, y, H, F, 2))) return rc;
        std::swap(x, y);
    }
    norm(x, w->g_f, y);                                                  // final norm: FP32 rows for the head
    CU_LAUNCH_CHECK(ctx, "layer_norm_kernel");
    { ProfScope ps(ctx, PROF_ROW, (double)nt * (H * 4 + (d_logits ? NL * 4 : 0) + (d_labels ? 4 : 0)));
    enc::launch_head_argmax(st, y, nt, H, w->W_c, w->b_c, NL, d_logits ? d_logits + (size_t)tok0 * NL : nullptr,
                            d_labels ? d_labels + tok0 : nullptr); }
    CU_LAUNCH_CHECK(ctx, "head_argmax_kernel");
    return ANON_OK;
}

int ner_forward_impl(anon_ctx* ctx, WsCursor& ws, const anon_weights* w, const int32_t* d_ids, const int32_t* d_cu,
                     const int32_t* h_cu, int32_t B, int32_t T, float* d_logits, int32_t* d_labels)
{
    if (!ctx || !w || w->ctx != ctx || B < 0 || T < 0 || !d_cu || !h_cu || (T > 0 && !d_ids)) return ANON_ERR_INVALID_ARG;
    if (h_cu[0] != 0 || h_cu[B] != T) return ANON_ERR_INVALID_ARG;
    const anon_model_desc& d = w->d;
    for (int s = 0; s < B; s++) {
        if (h_cu[s + 1] < h_cu[s]) return ANON_ERR_INVALID_ARG;
        if (h_cu[s + 1] - h_cu[s] > d.max_pos) return ANON_ERR_UNSUPPORTED;
    }
    if (T == 0) return ANON_OK;
    const int H = d.hidden, F = d.ffn, NL = d.num_labels;
    const bool bf = d.dtype == 1;
    cudaStream_t st = ctx->stream;

    // chunk budget: whole sequences, as many tokens as the remaining workspace holds (optionally capped)
    const size_t per_tok = per_token_bytes(d);
    const size_t avail = ws.left() > ((size_t)2 << 20) ? ws.left() - ((size_t)2 << 20) : 0;
    long long cap = (long long)(avail / per_tok);
    if (ctx->chunk_tokens_cap > 0 && cap > ctx->chunk_tokens_cap) cap = ctx->chunk_tokens_cap;
    if (cap < d.max_pos && cap < T) return ANON_ERR_OOM;

    int s0 = 0;
    while (s0 < B) {
        int s1 = s0;
        while (s1 < B && (long long)(h_cu[s1 + 1] - h_cu[s0]) <= cap) s1++;
        if (s1 == s0) return ANON_ERR_OOM;
        const int tok0 = h_cu[s0], nt = h_cu[s1] - tok0, nb = s1 - s0;
        if (nt > 0 && d.arch == 1) {
            const int rc = modern_chunk(ctx, ws, w, d_ids, d_cu, h_cu, B, s0, s1, d_logits, d_labels);
            if (rc) return rc;
        } else if (nt > 0) {
            WsCursor c = ws;          // chunk-local carve (same region reused by every chunk; stream-ordered)
            float* x = (float*)c.take((size_t)nt * H * 4);
            float* y = (float*)c.take((size_t)nt * H * 4);
            __nv_bfloat16* xb = bf ? (__nv_bfloat16*)c.take((size_t)nt * H * 2) : nullptr;
            void* qkv = c.take((size_t)nt * 3 * H * (bf ? 2 : 4));
            void* cx = c.take((size_t)nt * H * (bf ? 2 : 4));
            void* f = c.take((size_t)nt * F * (bf ? 2 : 4));
            if (!x || !y || (bf && !xb) || !qkv || !cx || !f) return ANON_ERR_OOM;
            AttnPlan plan;
            int prc = attention_plan(ctx, c, h_cu + s0, nb, d.dtype, &plan);
            if (prc) return prc;
            double attn_flops = 0;            // 4 n^2 d per (sequence, head): QK^T and PV
            for (int s = s0; s < s1; s++) { const double n = h_cu[s + 1] - h_cu[s]; attn_flops += 4.0 * n * n * H; }
            const unsigned row_grid = (unsigned)((nt + enc::kRowWarps - 1) / enc::kRowWarps);
            const double row_bytes = (double)nt * H * 4 * 2 + (bf ? (double)nt * H * 2 : 0);   // LN: read y, write x (+xb)
            { ProfScope ps(ctx, PROF_ROW, (double)nt * H * (bf ? 2 : 4) + (double)nt * (4 + H * 4 + (bf ? H * 2 : 0)));
            if (bf)
                enc::embed_ln_kernel<__nv_bfloat16><<<row_grid, enc::kRowWarps * 32, 0, st>>>(
                    d_ids, d_cu, B, tok0, nt, (const __nv_bfloat16*)w->E_w, (const __nv_bfloat16*)w->E_p, w->E_t, w->g_e,
                    w->b_e, d.ln_eps, H, d.vocab, d.max_pos, x, xb, ctx->d_status);
            else
                enc::embed_ln_kernel<float><<<row_grid, enc::kRowWarps * 32, 0, st>>>(
                    d_ids, d_cu, B, tok0, nt, (const float*)w->E_w, (const float*)w->E_p, w->E_t, w->g_e, w->b_e,
                    d.ln_eps, H, d.vocab, d.max_pos, x, nullptr, ctx->d_status);
            }
            CU_LAUNCH_CHECK(ctx, "embed_ln_kernel");
            // BF16 path with H = 768 / 1024: the residual stream is carried UN-normalised.  The LayerNorm kernel writes only
            // the BF16 operand copy xb and the row statistics; the next residual GEMM normalises the residual on the fly in
            // its epilogue and writes the new un-normalised rows (ping-pong between x and y: in-place updates measured 20 %
            // slower).  Saves the FP32 write of x (4H bytes per token and LayerNorm).  Only the last LayerNorm writes the
            // normalised FP32 rows (into y) for the classifier head.
            const bool lazy_ln = bf && (H == 768 || H == 1024);
            const float* head_in = x;
            const bool fold = lazy_ln && w->folded && ctx->fold_ln && !(ctx->ablate & 7);
            if (fold) {
                // LN2 FOLDED into the GEMMs around it (the LayerNorm between a layer's FFN and the next layer's attention): the FFN2
                // GEMM (producer) writes the un-normalised FP32 rows x, their BF16 copy (into xb) and per-row partial (sum, sum of
                // squares); the next QKV GEMM (consumer) takes the raw BF16 rows against W_qkv pre-multiplied by gamma_2 and
                // finishes the LayerNorm in its epilogue (free: that epilogue has slack).  LN1 stays a kernel: folding it into FFN1
                // made FFN1 epilogue-bound (+11 ms per step; the GELU epilogue has no slack, profiles/r02_summary.md).
                const int pc = H / 256;
                float2* part2 = (float2*)c.take((size_t)nt * pc * 8);
                float2* stats1 = (float2*)c.take((size_t)nt * 8);
                float2* stats2 = (float2*)c.take((size_t)nt * 8);
                if (!part2 || !stats1 || !stats2) return ANON_ERR_OOM;
                const float* pg = nullptr; const float* pb = nullptr;
                const double ln_bytes = (double)nt * (H * 4 + H * 2 + 8);
                for (int l = 0; l < d.layers; l++) {
                    const LayerW& L = w->layers[l];
                    int rc;
                    { ProfScope ps(ctx, PROF_GEMM, 2.0 * nt * 3 * H * H);
                    if (l == 0) rc = gemm_bf16_impl(ctx, xb, (const __nv_bfloat16*)L.W_qkv, L.b_qkv, nullptr, qkv, nt, 3 * H, H, 0);
                    else rc = gemm_bf16_fold_impl(ctx, xb, (const __nv_bfloat16*)L.Wf_qkv, L.c_qkv, L.s_qkv, part2, H, d.ln_eps, qkv, nt, 3 * H, H); }
                    if (rc) return rc;
                    { ProfScope ps(ctx, PROF_ATTN, attn_flops);
                    rc = attention_run(ctx, plan, qkv, d_cu + s0, tok0, nb, H, d.heads, d.dtype, cx); }
                    if (rc) return rc;
                    { ProfScope ps(ctx, PROF_GEMM_OUT, 2.0 * nt * H * H);
                    rc = gemm_bf16_res_ln_impl(ctx, (const __nv_bfloat16*)cx, (const __nv_bfloat16*)L.W_o, L.b_o, x, l == 0 ? nullptr : stats2, pg, pb, y, nt, H, H); }
                    if (rc) return rc;
                    { ProfScope ps(ctx, PROF_ROW, ln_bytes);
                    launch_layer_norm(st, row_grid, y, nt, H, L.g_1, L.b_1, d.ln_eps, nullptr, xb, stats1); }
                    CU_LAUNCH_CHECK(ctx, "layer_norm_kernel");
                    { ProfScope ps(ctx, PROF_GEMM_FFN1, 2.0 * nt * F * H);
                    rc = gemm_bf16_impl(ctx, xb, (const __nv_bfloat16*)L.W_1, L.b_1f, nullptr, f, nt, F, H, 1); }
                    if (rc) return rc;
                    { ProfScope ps(ctx, PROF_GEMM_FFN2, 2.0 * nt * F * H);
                    rc = gemm_bf16_fold_res_impl(ctx, (const __nv_bfloat16*)f, (const __nv_bfloat16*)L.W_2, L.b_2f, y, nullptr, stats1, L.g_1, L.b_1,
                                                 d.ln_eps, x, xb, part2, nt, H, F); }
                    if (rc) return rc;
                    { ProfScope ps(ctx, PROF_ROW, (double)nt * (pc * 8 + 8));
                    enc::stats_from_partials_kernel<<<(unsigned)((nt + 255) / 256), 256, 0, st>>>(part2, nt, pc, 1.0f / (float)H, d.ln_eps, stats2); }
                    CU_LAUNCH_CHECK(ctx, "stats_from_partials_kernel");
                    pg = L.g_2; pb = L.b_2;
                }
                if (d.layers > 0) {
                    ProfScope ps(ctx, PROF_ROW, (double)nt * (H * 4 + H * 4 + H * 2));
                    launch_layer_norm(st, row_grid, x, nt, H, pg, pb, d.ln_eps, y, xb, nullptr);
                    head_in = y;
                }
                CU_LAUNCH_CHECK(ctx, "layer_norm_kernel");
            } else if (lazy_ln) {
                float2* stats = (float2*)c.take((size_t)nt * 8);
                if (!stats) return ANON_ERR_OOM;
                const float2* pst = nullptr; const float* pg = nullptr; const float* pb = nullptr;   // embedding output: already normal
                const double ln_bytes = (double)nt * (H * 4 + H * 2 + 8);
                for (int l = 0; l < d.layers; l++) {
                    const LayerW& L = w->layers[l];
                    const bool last = l == d.layers - 1;
                    int rc;
                    { ProfScope ps(ctx, PROF_GEMM, 2.0 * nt * 3 * H * H);
                    rc = gemm_bf16_impl(ctx, xb, (const __nv_bfloat16*)L.W_qkv, L.b_qkv, nullptr, qkv, nt, 3 * H, H, 0); }
                    if (rc) return rc;
                    if (!(ctx->ablate & 1)) { ProfScope ps(ctx, PROF_ATTN, attn_flops);
                    rc = attention_run(ctx, plan, qkv, d_cu + s0, tok0, nb, H, d.heads, d.dtype, cx); }
                    if (rc) return rc;
                    if (!(ctx->ablate & 4)) { ProfScope ps(ctx, PROF_GEMM_OUT, 2.0 * nt * H * H);
                    rc = gemm_bf16_res_ln_impl(ctx, (const __nv_bfloat16*)cx, (const __nv_bfloat16*)L.W_o, L.b_o, x, pst, pg, pb, y, nt, H, H); }
                    if (rc) return rc;
                    if (!(ctx->ablate & 2)) { ProfScope ps(ctx, PROF_ROW, ln_bytes);
                    launch_layer_norm(st, row_grid, y, nt, H, L.g_1, L.b_1, d.ln_eps, nullptr, xb, stats); }
                    CU_LAUNCH_CHECK(ctx, "layer_norm_kernel");
                    { ProfScope ps(ctx, PROF_GEMM_FFN1, 2.0 * nt * F * H);
                    rc = gemm_bf16_impl(ctx, xb, (const __nv_bfloat16*)L.W_1, L.b_1f, nullptr, f, nt, F, H, (ctx->ablate & 8) ? 0 : 1); }
                    if (rc) return rc;
                    { ProfScope ps(ctx, PROF_GEMM_FFN2, 2.0 * nt * F * H);
                    rc = gemm_bf16_res_ln_impl(ctx, (const __nv_bfloat16*)f, (const __nv_bfloat16*)L.W_2, L.b_2f, y, stats, L.g_1, L.b_1, x, nt, H, F); }
                    if (rc) return rc;
                    if (!(ctx->ablate & 2) || last) { ProfScope ps(ctx, PROF_ROW, ln_bytes + (last ? (double)nt * H * 4 : 0.0));
                    launch_layer_norm(st, row_grid, x, nt, H, L.g_2, L.b_2, d.ln_eps, last ? y : nullptr, xb, stats); }
                    CU_LAUNCH_CHECK(ctx, "layer_norm_kernel");
                    pst = stats; pg = L.g_2; pb = L.b_2;
                    if (last) head_in = y;
                }
            }
            for (int l = 0; l < ((lazy_ln || fold) ? 0 : d.layers); l++) {
                const LayerW& L = w->layers[l];
                int rc;
                { ProfScope ps(ctx, PROF_GEMM, 2.0 * nt * 3 * H * H);
                if (bf) rc = gemm_bf16_impl(ctx, xb, (const __nv_bfloat16*)L.W_qkv, L.b_qkv, nullptr, qkv, nt, 3 * H, H, 0);
                else rc = sgemm<0>(ctx, x, (const float*)L.W_qkv, L.b_qkv, nullptr, (float*)qkv, nt, 3 * H, H); }
                if (rc) return rc;
                { ProfScope ps(ctx, PROF_ATTN, attn_flops);
                rc = attention_run(ctx, plan, qkv, d_cu + s0, tok0, nb, H, d.heads, d.dtype, cx); }
                if (rc) return rc;
                { ProfScope ps(ctx, PROF_GEMM_OUT, 2.0 * nt * H * H);
                if (bf) rc = gemm_bf16_impl(ctx, (const __nv_bfloat16*)cx, (const __nv_bfloat16*)L.W_o, L.b_o, x, y, nt, H, H, 2);
                else rc = sgemm<2>(ctx, (const float*)cx, (const float*)L.W_o, L.b_o, x, y, nt, H, H); }
                if (rc) return rc;
                { ProfScope ps(ctx, PROF_ROW, row_bytes);
                launch_layer_norm(st, row_grid, y, nt, H, L.g_1, L.b_1, d.ln_eps, x, xb); }
                CU_LAUNCH_CHECK(ctx, "layer_norm_kernel");
                { ProfScope ps(ctx, PROF_GEMM_FFN1, 2.0 * nt * F * H);
                if (bf) rc = gemm_bf16_impl(ctx, xb, (const __nv_bfloat16*)L.W_1, L.b_1f, nullptr, f, nt, F, H, 1);
                else rc = sgemm<1>(ctx, x, (const float*)L.W_1, L.b_1f, nullptr, (float*)f, nt, F, H); }
                if (rc) return rc;
                { ProfScope ps(ctx, PROF_GEMM_FFN2, 2.0 * nt * F * H);
                if (bf) rc = gemm_bf16_impl(ctx, (const __nv_bfloat16*)f, (const __nv_bfloat16*)L.W_2, L.b_2f, x, y, nt, H, F, 2);
                else rc = sgemm<2>(ctx, (const float*)f, (const float*)L.W_2, L.b_2f, x, y, nt, H, F); }
                if (rc) return rc;
                { ProfScope ps(ctx, PROF_ROW, row_bytes);
                launch_layer_norm(st, row_grid, y, nt, H, L.g_2, L.b_2, d.ln_eps, x, xb); }
                CU_LAUNCH_CHECK(ctx, "layer_norm_kernel");
            }
            { ProfScope ps(ctx, PROF_ROW, (double)nt * (H * 4 + (d_logits ? NL * 4 : 0) + (d_labels ? 4 : 0)));
            enc::launch_head_argmax(st, head_in, nt, H, w->W_c, w->b_c, NL, d_logits ? d_logits + (size_t)tok0 * NL : nullptr,
                                    d_labels ? d_labels + tok0 : nullptr); }
            CU_LAUNCH_CHECK(ctx, "head_argmax_kernel");
        }
        s0 = s1;
    }
    return ANON_OK;
}

extern "C" int anon_ner_forward(anon_ctx* ctx, const anon_weights* w, const int32_t* d_token_ids,
                                const int32_t* d_cu_seqlens, int32_t B, int32_t T, float* d_logits, int32_t* d_labels)
{
    if (!ctx || !w || B < 0 || T < 0 || !d_cu_seqlens) return ANON_ERR_INVALID_ARG;
    CU_TRY(ctx, cudaSetDevice(ctx->device));
    std::vector<int32_t> h_cu((size_t)B + 1);
    CU_TRY(ctx, cudaMemcpyAsync(h_cu.data(), d_cu_seqlens, ((size_t)B + 1) * 4, cudaMemcpyDeviceToHost, ctx->stream));
    CU_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    WsCursor ws = ws_begin(ctx);
    return ner_forward_impl(ctx, ws, w, d_token_ids, d_cu_seqlens, h_cu.data(), B, T, d_logits, d_labels);
}
