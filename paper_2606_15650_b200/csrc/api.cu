// api.cu -- context lifecycle, error strings, and the host-buffer pipeline entry point (include/anonshield.h).
#include "common.cuh"

#include <new>
#include <stdlib.h>

extern "C" const char* anon_strerror(int code) {
    switch (code) {
        case ANON_OK: return "ok";
        case ANON_ERR_INVALID_ARG: return "invalid argument";
        case ANON_ERR_UNSUPPORTED: return "unsupported shape or value";
        case ANON_ERR_CAPACITY: return "capacity exceeded (span list / cache / arena / output buffer)";
        case ANON_ERR_KEY_MISMATCH: return "cache is bound to another HMAC key";
        case ANON_ERR_CUDA: return "CUDA error (see anon_last_cuda_error)";
        case ANON_ERR_OOM: return "workspace or device memory too small";
        default: return "unknown error code";
    }
}

extern "C" const char* const* anon_exported_symbols(void) {
    static const char* const names[] = {
        "anon_strerror", "anon_exported_symbols", "anon_ctx_create", "anon_ctx_destroy", "anon_ctx_sync",
        "anon_last_cuda_error", "anon_workspace_bytes", "anon_weights_load", "anon_weights_free", "anon_ner_forward",
        "anon_decode_spans", "anon_gather_spans", "anon_cache_create", "anon_cache_destroy", "anon_cache_stats", "anon_cache_clear",
        "anon_cache_entry", "anon_cache_export", "anon_pseudonymize", "anon_hmac_spans", "anon_pipeline_host", "anon_gemm_bf16",
        "anon_attention", "anon_splice_records", "anon_pipeline_host_text", "anon_ctx_profile", "anon_ctx_profile_read",
        "anon_regex_load", "anon_regex_free", "anon_regex_scan", "anon_merge_spans", "anon_ctx_set_regex", "anon_attention_local", "anon_cache_track_use", "anon_cache_evict", "anon_microbench", "anon_gemm_bf16_fold_res", "anon_gemm_bf16_fold", "anon_decode_spans_static", nullptr};
    return names;
}

extern "C" int anon_ctx_create(anon_ctx** out, int device, void* cuda_stream, size_t workspace_bytes) {
    if (!out || device < 0) return ANON_ERR_INVALID_ARG;
    *out = nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device >= ndev) { cudaGetLastError(); return ANON_ERR_CUDA; }
    anon_ctx* c = new (std::nothrow) anon_ctx();
    if (!c) return ANON_ERR_OOM;
    c->device = device;
    c->stream = (cudaStream_t)cuda_stream;
    { const char* e = getenv("ANON_CHUNK_TOKENS"); c->chunk_tokens_cap = e ? atoll(e) : 0; }
    { const char* e = getenv("ANON_ABLATE"); c->ablate = e ? atoi(e) : 0; }
    { const char* e = getenv("ANON_FOLD_LN"); c->fold_ln = e ? atoi(e) : 1; }
    cudaError_t e = cudaSetDevice(device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, device);
    if (e == cudaSuccess) e = cudaMalloc(&c->d_status, 256);
    if (e == cudaSuccess) e = cudaMemset(c->d_status, 0, 256);
    c->h_pinned_bytes = 4096;
    if (e == cudaSuccess) e = cudaMallocHost(&c->h_pinned, c->h_pinned_bytes);
    if (e != cudaSuccess) { anon_ctx_destroy(c); cudaGetLastError(); return ANON_ERR_CUDA; }
    if (workspace_bytes) {
        e = cudaMalloc(&c->ws, workspace_bytes);
        if (e != cudaSuccess) { anon_ctx_destroy(c); cudaGetLastError(); return ANON_ERR_OOM; }
        c->ws_bytes = workspace_bytes;
    }
    *out = c;
    return ANON_OK;
}

extern "C" void anon_ctx_destroy(anon_ctx* c) {
    if (!c) return;
    for (auto& r : c->prof_recs) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    cudaFree(c->ws);
    cudaFree(c->d_status);
    if (c->h_pinned) cudaFreeHost(c->h_pinned);
    delete c;
}

extern "C" int anon_ctx_sync(anon_ctx* ctx) {
    if (!ctx) return ANON_ERR_INVALID_ARG;
    int* h = (int*)(ctx->h_pinned + 128);
    CU_TRY(ctx, cudaMemcpyAsync(h, ctx->d_status, 4, cudaMemcpyDeviceToHost, ctx->stream));
    CU_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    const int s = *h;
    if (s != 0) {
        CU_TRY(ctx, cudaMemsetAsync(ctx->d_status, 0, 4, ctx->stream));
        CU_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    }
    return s;
}

extern "C" int anon_ctx_profile(anon_ctx* ctx, int enable) {
    if (!ctx) return ANON_ERR_INVALID_ARG;
    CU_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->prof_on = enable != 0;
    ctx->prof_used = 0;
    ctx->n_launches = 0;
    for (int i = 0; i < PROF_NCLASS; i++) { ctx->prof_work[i] = 0; ctx->prof_launches[i] = 0; }
    return ANON_OK;
}

extern "C" int anon_ctx_profile_read(anon_ctx* ctx, double* class_ms, double* class_work, int64_t* class_launches,
                                     int64_t* total_launches) {
    if (!ctx) return ANON_ERR_INVALID_ARG;
    CU_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    double ms[PROF_NCLASS] = {0};
    for (size_t i = 0; i < ctx->prof_used; i++) {
        float t = 0.f;
        if (cudaEventElapsedTime(&t, ctx->prof_recs[i].a, ctx->prof_recs[i].b) == cudaSuccess) ms[ctx->prof_recs[i].cls] += t;
    }
    for (int i = 0; i < PROF_NCLASS; i++) {
        if (class_ms) class_ms[i] = ms[i];
        if (class_work) class_work[i] = ctx->prof_work[i];
        if (class_launches) class_launches[i] = ctx->prof_launches[i];
    }
    if (total_launches) *total_launches = ctx->n_launches;
    return ANON_OK;
}

extern "C" int anon_ctx_set_regex(anon_ctx* ctx, const anon_regex* rx) {
    if (!ctx) return ANON_ERR_INVALID_ARG;
    ctx->regex = rx;
    return ANON_OK;
}

extern "C" const char* anon_last_cuda_error(anon_ctx* ctx) { return ctx ? ctx->cuda_err : ""; }

int splice_records_impl(anon_ctx* ctx, WsCursor& ws, const uint8_t* d_text, size_t text_bytes, const int64_t* d_rec_off, int32_t R,
                        const anon_span* d_spans, int32_t S, const uint8_t* d_tok, const int64_t* d_tok_off,
                        uint8_t* d_new_text, size_t cap, int64_t* d_new_rec_off);

// h_new_text != NULL: the records are also rewritten on the device (NEXT-1) and come back as text
static int pipeline_host_impl(anon_ctx* ctx, const anon_weights* w, anon_cache* cache,
                              const int32_t* h_ids, const int32_t* h_cu, int32_t B, int32_t T,
                              const anon_tok_meta* h_meta, const uint8_t* h_text, size_t text_bytes,
                              const int64_t* h_rec_off, int32_t R, const uint8_t* key, size_t key_len,
                              int32_t slug_len, const char* const* type_names, int32_t num_types,
                              anon_span* h_spans, int32_t span_capacity, int32_t* h_num_spans,
                              uint8_t* h_out_tokens, size_t out_capacity, int64_t* h_out_offsets, uint8_t* h_hit,
                              uint8_t* h_new_text, size_t new_text_capacity, int64_t* h_new_rec_off)
{
    if (!ctx || !w || !cache || !h_ids || !h_cu || !h_meta || !h_text || !h_rec_off || !h_spans || !h_num_spans ||
        !h_out_tokens || !h_out_offsets || B < 0 || T < 0 || R < 0 || span_capacity < 0)
        return ANON_ERR_INVALID_ARG;
    CU_TRY(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    *h_num_spans = 0;
    WsCursor ws = ws_begin(ctx);
    const int NL = weights_desc(w)->num_labels;
    // device staging
    int32_t* d_ids = (int32_t*)ws.take((size_t)T * 4 + 4);
    int32_t* d_cu = (int32_t*)ws.take(((size_t)B + 1) * 4);
    anon_tok_meta* d_meta = (anon_tok_meta*)ws.take((size_t)T * sizeof(anon_tok_meta) + 16);
    uint8_t* d_text = (uint8_t*)ws.take(text_bytes + 16);
    int64_t* d_rec_off = (int64_t*)ws.take(((size_t)R + 1) * 8);
    int32_t* d_labels = (int32_t*)ws.take((size_t)T * 4 + 4);
    anon_span* d_spans = (anon_span*)ws.take((size_t)span_capacity * sizeof(anon_span) + 16);
    int32_t* d_num = (int32_t*)ws.take(16);
    int64_t* d_span_off = (int64_t*)ws.take(((size_t)span_capacity + 1) * 8);
    uint8_t* d_span_type = (uint8_t*)ws.take((size_t)span_capacity + 16);
    int64_t* d_out_off = (int64_t*)ws.take(((size_t)span_capacity + 1) * 8);
    uint8_t* d_hit = (uint8_t*)ws.take((size_t)span_capacity + 16);
    // span bytes can never exceed the text that was scanned
    uint8_t* d_span_bytes = (uint8_t*)ws.take(text_bytes + 16);
    uint8_t* d_out = (uint8_t*)ws.take(out_capacity + 16);
    uint8_t* d_new_text = h_new_text ? (uint8_t*)ws.take(new_text_capacity + 16) : nullptr;
    int64_t* d_new_rec_off = h_new_text ? (int64_t*)ws.take(((size_t)R + 1) * 8) : nullptr;
    // NEXT-4: regex spans and the merged list (only with an attached automaton)
    anon_span* d_rx_spans = ctx->regex ? (anon_span*)ws.take((size_t)span_capacity * sizeof(anon_span) + 16) : nullptr;
    anon_span* d_merged = ctx->regex ? (anon_span*)ws.take((size_t)span_capacity * sizeof(anon_span) + 16) : nullptr;
    if (ctx->regex && (!d_rx_spans || !d_merged)) return ANON_ERR_OOM;
    if (h_new_text && (!d_new_text || !d_new_rec_off || !h_new_rec_off)) return d_new_text ? ANON_ERR_INVALID_ARG : ANON_ERR_OOM;
    if (!d_ids || !d_cu || !d_meta || !d_text || !d_rec_off || !d_labels || !d_spans || !d_num || !d_span_off ||
        !d_span_type || !d_out_off || !d_hit || !d_span_bytes || !d_out)
        return ANON_ERR_OOM;
    CU_TRY(ctx, cudaMemcpyAsync(d_ids, h_ids, (size_t)T * 4, cudaMemcpyHostToDevice, st));
    CU_TRY(ctx, cudaMemcpyAsync(d_cu, h_cu, ((size_t)B + 1) * 4, cudaMemcpyHostToDevice, st));
    CU_TRY(ctx, cudaMemcpyAsync(d_meta, h_meta, (size_t)T * sizeof(anon_tok_meta), cudaMemcpyHostToDevice, st));
    CU_TRY(ctx, cudaMemcpyAsync(d_text, h_text, text_bytes, cudaMemcpyHostToDevice, st));
    CU_TRY(ctx, cudaMemcpyAsync(d_rec_off, h_rec_off, ((size_t)R + 1) * 8, cudaMemcpyHostToDevice, st));

    int rc = ner_forward_impl(ctx, ws, w, d_ids, d_cu, h_cu, B, T, nullptr, d_labels);
    if (rc) return rc;
    {
        WsCursor c = ws;
        rc = decode_spans_impl(ctx, c, d_labels, d_meta, T, NL, d_spans, span_capacity, d_num);
        if (rc) return rc;
    }
    if (ctx->regex) {
        // d_num[0] = NER spans, [1] = regex spans, [2] = merged; a list that overflowed latches CAPACITY (checked below)
        {
            WsCursor c = ws;
            rc = regex_scan_impl(ctx, c, ctx->regex, d_text, text_bytes, d_rec_off, R, d_rx_spans, span_capacity, d_num + 1);
            if (rc) return rc;
        }
        WsCursor c = ws;
        rc = merge_spans_impl(ctx, c, d_spans, d_num, span_capacity, d_rx_spans, d_num + 1, span_capacity, d_merged, span_capacity,
                              d_num + 2);
        if (rc) return rc;
        d_spans = d_merged;
        d_num += 2;
    }
    int* h_n = (int*)(ctx->h_pinned + 256);
    int* h_status = (int*)(ctx->h_pinned + 260);
    CU_TRY(ctx, cudaMemcpyAsync(h_n, d_num, 4, cudaMemcpyDeviceToHost, st));
    CU_TRY(ctx, cudaMemcpyAsync(h_status, ctx->d_status, 4, cudaMemcpyDeviceToHost, st));
    CU_TRY(ctx, cudaStreamSynchronize(st));
    const int S = *h_n;
    *h_num_spans = S;
    if (*h_status != 0) {
        const int s = *h_status;
        CU_TRY(ctx, cudaMemsetAsync(ctx->d_status, 0, 4, st));
        CU_TRY(ctx, cudaStreamSynchronize(st));
        return s;
    }
    if (S > span_capacity) return ANON_ERR_CAPACITY;
    {
        WsCursor c = ws;
        rc = gather_spans_impl(ctx, c, d_text, d_rec_off, d_spans, nullptr, S, d_span_bytes, text_bytes, d_span_off, d_span_type);
        if (rc) return rc;
    }
    {   // a gather overflow (span bytes past their buffer) must stop the pipeline before the probe reads them
        CU_TRY(ctx, cudaMemcpyAsync(h_status, ctx->d_status, 4, cudaMemcpyDeviceToHost, st));
        CU_TRY(ctx, cudaStreamSynchronize(st));
        if (*h_status != 0) {
            const int s = *h_status;
            CU_TRY(ctx, cudaMemsetAsync(ctx->d_status, 0, 4, st));
            CU_TRY(ctx, cudaStreamSynchronize(st));
            return s;
        }
    }
    int64_t out_bytes = 0;
    {
        WsCursor c = ws;
        rc = pseudonymize_impl(ctx, c, cache, d_span_bytes, d_span_off, d_span_type, S, key, key_len, slug_len, type_names,
                               num_types, d_out, out_capacity, d_out_off, h_hit ? d_hit : nullptr, nullptr, nullptr, &out_bytes);
        if (rc) return rc;
    }
    if (h_new_text) {
        // the splice kernels bound-check every write against the capacity and latch CAPACITY; the exact new size
        // (text - span bytes + token bytes) comes back with the new record offsets
        WsCursor c = ws;
        rc = splice_records_impl(ctx, c, d_text, text_bytes, d_rec_off, R, d_spans, S, d_out, d_out_off, d_new_text,
                                 new_text_capacity, d_new_rec_off);
        if (rc) return rc;
        CU_TRY(ctx, cudaMemcpyAsync(h_new_rec_off, d_new_rec_off, ((size_t)R + 1) * 8, cudaMemcpyDeviceToHost, st));
        CU_TRY(ctx, cudaStreamSynchronize(st));
        const int64_t new_bytes = h_new_rec_off[R];
        if (new_bytes < 0 || (uint64_t)new_bytes > new_text_capacity) {
            CU_TRY(ctx, cudaMemsetAsync(ctx->d_status, 0, 4, st));
            CU_TRY(ctx, cudaStreamSynchronize(st));
            return ANON_ERR_CAPACITY;
        }
        if (new_bytes > 0) CU_TRY(ctx, cudaMemcpyAsync(h_new_text, d_new_text, (size_t)new_bytes, cudaMemcpyDeviceToHost, st));
    }
    if (S > 0) {
        CU_TRY(ctx, cudaMemcpyAsync(h_spans, d_spans, (size_t)S * sizeof(anon_span), cudaMemcpyDeviceToHost, st));
        CU_TRY(ctx, cudaMemcpyAsync(h_out_tokens, d_out, (size_t)out_bytes, cudaMemcpyDeviceToHost, st));
        if (h_hit) CU_TRY(ctx, cudaMemcpyAsync(h_hit, d_hit, (size_t)S, cudaMemcpyDeviceToHost, st));
    }
    CU_TRY(ctx, cudaMemcpyAsync(h_out_offsets, d_out_off, ((size_t)S + 1) * 8, cudaMemcpyDeviceToHost, st));
    return anon_ctx_sync(ctx);
}

extern "C" int anon_pipeline_host(anon_ctx* ctx, const anon_weights* w, anon_cache* cache,
                                  const int32_t* h_ids, const int32_t* h_cu, int32_t B, int32_t T,
                                  const anon_tok_meta* h_meta, const uint8_t* h_text, size_t text_bytes,
                                  const int64_t* h_rec_off, int32_t R, const uint8_t* key, size_t key_len,
                                  int32_t slug_len, const char* const* type_names, int32_t num_types,
                                  anon_span* h_spans, int32_t span_capacity, int32_t* h_num_spans,
                                  uint8_t* h_out_tokens, size_t out_capacity, int64_t* h_out_offsets, uint8_t* h_hit)
{
    return pipeline_host_impl(ctx, w, cache, h_ids, h_cu, B, T, h_meta, h_text, text_bytes, h_rec_off, R, key, key_len, slug_len,
                              type_names, num_types, h_spans, span_capacity, h_num_spans, h_out_tokens, out_capacity,
                              h_out_offsets, h_hit, nullptr, 0, nullptr);
}

extern "C" int anon_pipeline_host_text(anon_ctx* ctx, const anon_weights* w, anon_cache* cache,
                                       const int32_t* h_ids, const int32_t* h_cu, int32_t B, int32_t T,
                                       const anon_tok_meta* h_meta, const uint8_t* h_text, size_t text_bytes,
                                       const int64_t* h_rec_off, int32_t R, const uint8_t* key, size_t key_len,
                                       int32_t slug_len, const char* const* type_names, int32_t num_types,
                                       anon_span* h_spans, int32_t span_capacity, int32_t* h_num_spans,
                                       uint8_t* h_out_tokens, size_t out_capacity, int64_t* h_out_offsets, uint8_t* h_hit,
                                       uint8_t* h_new_text, size_t new_text_capacity, int64_t* h_new_record_offsets)
{
    if (!h_new_text || !h_new_record_offsets) return ANON_ERR_INVALID_ARG;
    return pipeline_host_impl(ctx, w, cache, h_ids, h_cu, B, T, h_meta, h_text, text_bytes, h_rec_off, R, key, key_len, slug_len,
                              type_names, num_types, h_spans, span_capacity, h_num_spans, h_out_tokens, out_capacity,
                              h_out_offsets, h_hit, h_new_text, new_text_capacity, h_new_record_offsets);
}
