// encoder_kernels.cuh -- the HBM-bound encoder kernels (K1 embed+LN, K4 LN, K6 head+argmax) and the FP32
// SIMT path for BJ configs[0] (K2f SGEMM, FP32 attention).  S8a A1, A4, A6, A7, A8; S8c O1, O2.
// One warp per token row; every global access is a coalesced 16-byte vector; statistics in FP32 with the
// two-pass (mean, then centred variance) form of O1.
#pragma once
#include "common.cuh"

namespace enc {

constexpr int kMaxVec = 8;           // hidden <= 1024 (8 float4 per lane)
constexpr int kRowWarps = 8;         // warps (token rows) per CTA for the row kernels

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    return v;
}

__device__ __forceinline__ float4 load4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }
__device__ __forceinline__ float4 load4(const __nv_bfloat16* p) {
    const uint2 u = __ldg(reinterpret_cast<const uint2*>(p));
    const __nv_bfloat162 a = *reinterpret_cast<const __nv_bfloat162*>(&u.x);
    const __nv_bfloat162 b = *reinterpret_cast<const __nv_bfloat162*>(&u.y);
    const float2 fa = __bfloat1622float2(a), fb = __bfloat1622float2(b);
    return make_float4(fa.x, fa.y, fb.x, fb.y);
}

// LN over one row held as n4 float4 per lane (element index = 4*(lane + 32k) + c); writes FP32 and optional BF16.
__device__ __forceinline__ void layer_norm_row(float4 (&v)[kMaxVec], int n4, int H, const float* __restrict__ g,
                                               const float* __restrict__ b, float eps, int lane,
                                               float* __restrict__ xo, __nv_bfloat16* __restrict__ xbo) {
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < kMaxVec; k++) if (k < n4) s += (v[k].x + v[k].y) + (v[k].z + v[k].w);
    const float mean = warp_sum(s) / (float)H;
    float q = 0.f;
#pragma unroll
    for (int k = 0; k < kMaxVec; k++) if (k < n4) {
        v[k].x -= mean; v[k].y -= mean; v[k].z -= mean; v[k].w -= mean;
        q += (v[k].x * v[k].x + v[k].y * v[k].y) + (v[k].z * v[k].z + v[k].w * v[k].w);
    }
    const float rstd = 1.0f / sqrtf(warp_sum(q) / (float)H + eps);
#pragma unroll
    for (int k = 0; k < kMaxVec; k++) if (k < n4) {
        const int e = 4 * (lane + 32 * k);
        const float4 gg = load4(g + e), bb = load4(b + e);
        float4 o;
        o.x = v[k].x * rstd * gg.x + bb.x; o.y = v[k].y * rstd * gg.y + bb.y;
        o.z = v[k].z * rstd * gg.z + bb.z; o.w = v[k].w * rstd * gg.w + bb.w;
        if (xo) *reinterpret_cast<float4*>(xo + e) = o;
        if (xbo) {
            __nv_bfloat162 lo = __floats2bfloat162_rn(o.x, o.y), hi = __floats2bfloat162_rn(o.z, o.w);
            uint2 u;
            u.x = *reinterpret_cast<uint32_t*>(&lo); u.y = *reinterpret_cast<uint32_t*>(&hi);
            *reinterpret_cast<uint2*>(xbo + e) = u;
        }
    }
}

// K1: x_j = LN(E_w[id_j] + E_p[pos_j] + E_t).  tok0 = first token of the chunk (absolute index); cu is absolute.
template <class TE>
static __global__ void __launch_bounds__(kRowWarps * 32) embed_ln_kernel(
    const int* __restrict__ ids, const int* __restrict__ cu, int B, int tok0, int ntok, const TE* __restrict__ E_w,
    const TE* __restrict__ E_p, const float* __restrict__ E_t, const float* __restrict__ g, const float* __restrict__ b,
    float eps, int H, int V, int max_pos, float* __restrict__ x, __nv_bfloat16* __restrict__ xb, int* d_status)
{
    const int lane = threadIdx.x & 31;
    const int r = blockIdx.x * kRowWarps + (threadIdx.x >> 5);
    if (r >= ntok) return;
    const int j = tok0 + r;
    int lo = 0, hi = B;                       // largest s with cu[s] <= j  (cu[B] = T > j)
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (__ldg(cu + mid) <= j) lo = mid; else hi = mid; }
    int pos = j - __ldg(cu + lo);
    int id = __ldg(ids + j);
    if (id < 0 || id >= V || pos >= max_pos) {
        if (lane == 0) latch_status(d_status, ANON_ERR_UNSUPPORTED);
        id = id < 0 ? 0 : (id >= V ? V - 1 : id);
        pos = pos >= max_pos ? max_pos - 1 : pos;
    }
    const int n4 = H >> 7;
    float4 v[kMaxVec];
#pragma unroll
    for (int k = 0; k < kMaxVec; k++) if (k < n4) {
        const int e = 4 * (lane + 32 * k);
        const float4 a = load4(E_w + (size_t)id * H + e), p = load4(E_p + (size_t)pos * H + e), t = load4(E_t + e);
        v[k] = make_float4(a.x + p.x + t.x, a.y + p.y + t.y, a.z + p.z + t.z, a.w + p.w + t.w);
    }
    layer_norm_row(v, n4, H, g, b, eps, lane, x + (size_t)r * H, xb ? xb + (size_t)r * H : nullptr);
}

// K4: x = LN(y) (the residual add is fused into the producing GEMM's epilogue), or x = LN(y + res) if res != NULL.
static __global__ void __launch_bounds__(kRowWarps * 32) layer_norm_kernel(
    const float* __restrict__ y, const float* __restrict__ res, int ntok, int H, const float* __restrict__ g,
    const float* __restrict__ b, float eps, float* __restrict__ x, __nv_bfloat16* __restrict__ xb)
{
    const int lane = threadIdx.x & 31;
    const int r = blockIdx.x * kRowWarps + (threadIdx.x >> 5);
    if (r >= ntok) return;
    const int n4 = H >> 7;
    float4 v[kMaxVec];
#pragma unroll
    for (int k = 0; k < kMaxVec; k++) if (k < n4) {
        const int e = 4 * (lane + 32 * k);
        v[k] = load4(y + (size_t)r * H + e);
        if (res) { const float4 o = load4(res + (size_t)r * H + e); v[k].x += o.x; v[k].y += o.y; v[k].z += o.z; v[k].w += o.w; }
    }
    layer_norm_row(v, n4, H, g, b, eps, lane, x + (size_t)r * H, xb ? xb + (size_t)r * H : nullptr);
}

// K4 with the row length known at compile time (H = 128 * N4): the row lives in exactly N4 float4 per lane, which
// lets ptxas keep the kernel at 48 registers and 5 CTAs (40 warps) resident per SM.
template <int N4>
static __global__ void __launch_bounds__(kRowWarps * 32, (N4 <= 6) ? 5 : 4) layer_norm_fixed_kernel(
    const float* __restrict__ y, int ntok, const float* __restrict__ g, const float* __restrict__ b, float eps,
    float* __restrict__ x, __nv_bfloat16* __restrict__ xb, float2* __restrict__ stats)
{
    // x == NULL: the FP32 row is not written; the consumer (the next residual GEMM's epilogue) recomputes it from y and
    // stats[row] = (mean, rstd), which saves 4H bytes of HBM writes per token
    constexpr int H = 128 * N4;
    const int lane = threadIdx.x & 31;
    const int r = blockIdx.x * kRowWarps + (threadIdx.x >> 5);
    if (r >= ntok) return;
    float4 v[N4];
    const float4* src = reinterpret_cast<const float4*>(y + (size_t)r * H) + lane;
#pragma unroll
    for (int k = 0; k < N4; k++) v[k] = __ldcs(src + 32 * k);
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < N4; k++) s += (v[k].x + v[k].y) + (v[k].z + v[k].w);
    const float mean = warp_sum(s) * (1.0f / (float)H);
    float q = 0.f;
#pragma unroll
    for (int k = 0; k < N4; k++) {
        v[k].x -= mean; v[k].y -= mean; v[k].z -= mean; v[k].w -= mean;
        q += (v[k].x * v[k].x + v[k].y * v[k].y) + (v[k].z * v[k].z + v[k].w * v[k].w);
    }
    const float rstd = 1.0f / sqrtf(warp_sum(q) * (1.0f / (float)H) + eps);
    if (stats && lane == 0) stats[r] = make_float2(mean, rstd);
    float4* xo = reinterpret_cast<float4*>(x + (size_t)r * H) + lane;
    uint2* xbo = reinterpret_cast<uint2*>(xb + (size_t)r * H) + lane;
#pragma unroll
    for (int k = 0; k < N4; k++) {
        const int e = 4 * (lane + 32 * k);
        const float4 gg = load4(g + e), bb = load4(b + e);
        float4 o;
        o.x = v[k].x * rstd * gg.x + bb.x; o.y = v[k].y * rstd * gg.y + bb.y;
        o.z = v[k].z * rstd * gg.z + bb.z; o.w = v[k].w * rstd * gg.w + bb.w;
        if (x) xo[32 * k] = o;
        __nv_bfloat162 lo = __floats2bfloat162_rn(o.x, o.y), hi = __floats2bfloat162_rn(o.z, o.w);
        uint2 u;
        u.x = *reinterpret_cast<uint32_t*>(&lo); u.y = *reinterpret_cast<uint32_t*>(&hi);
        xbo[32 * k] = u;
    }
}

// Row statistics from the partial sums a folding residual GEMM wrote (gemm_tcgen05.cu FOLD): part[row][cnt] = (sum, sum of squares)
// over 256 columns each -> stats[row] = (mean, rstd), summed in index order (deterministic).
static __global__ void __launch_bounds__(256) stats_from_partials_kernel(const float2* __restrict__ part, int ntok, int cnt, float inv_h,
                                                                         float eps, float2* __restrict__ stats)
{
    const int r = blockIdx.x * 256 + threadIdx.x;
    if (r >= ntok) return;
    float s = 0.f, q = 0.f;
    for (int i = 0; i < cnt; i++) { const float2 p = __ldg(part + (size_t)r * cnt + i); s += p.x; q += p.y; }
    const float mean = s * inv_h;
    const float var = fmaxf(q * inv_h - mean * mean, 0.f);
    stats[r] = make_float2(mean, 1.0f / sqrtf(var + eps));
}

// K6: logits = x W_c^T + b_c (FP32), label = argmax (ties -> lowest index).
static __global__ void __launch_bounds__(kRowWarps * 32) head_argmax_kernel(
    const float* __restrict__ x, int ntok, int H, const float* __restrict__ W_c, const float* __restrict__ b_c, int NL,
    float* __restrict__ logits, int* __restrict__ labels)
{
    const int lane = threadIdx.x & 31;
    const int r = blockIdx.x * kRowWarps + (threadIdx.x >> 5);
    if (r >= ntok) return;
    const int n4 = H >> 7;
    float4 v[kMaxVec];
#pragma unroll
    for (int k = 0; k < kMaxVec; k++) if (k < n4) v[k] = load4(x + (size_t)r * H + 4 * (lane + 32 * k));
    float best = 0.f; int best_c = 0;
    for (int c = 0; c < NL; c++) {
        float s = 0.f;
#pragma unroll
        for (int k = 0; k < kMaxVec; k++) if (k < n4) {
            const float4 w = load4(W_c + (size_t)c * H + 4 * (lane + 32 * k));
            s += (v[k].x * w.x + v[k].y * w.y) + (v[k].z * w.z + v[k].w * w.w);
        }
        s = warp_sum(s) + __ldg(b_c + c);
        if (logits && lane == 0) logits[(size_t)r * NL + c] = s;
        if (c == 0 || s > best) { best = s; best_c = c; }
    }
    if (labels && lane == 0) labels[r] = best_c;
}

// K6 for NL <= 16 (the paper's 9 / 13 BIO labels): two token rows per warp, all class sums kept per lane as FMA chains (hidden
// loop outside, class loop inside, so a W_c vector serves both rows), then ONE transposed butterfly per row -- at every step a
// lane keeps half of its class sums and trades the other half -- 16 shuffles instead of 5 per class.  Lanes 2c and 2c + 1 end up
// with the logit of class c; the argmax (ties -> lowest index) runs across lanes on those same values.  ncu on the kernel
// above: L1 data pipe 95 % and issue slots 75 % busy at 1,450 instructions per token; this one issues about a third of that.
constexpr int kHeadRows = 2;
static __global__ void __launch_bounds__(kRowWarps * 32, 2) head_argmax16_kernel(
    const float* __restrict__ x, int ntok, int H, const float* __restrict__ W_c, const float* __restrict__ b_c, int NL,
    float* __restrict__ logits, int* __restrict__ labels)
{
    const int lane = threadIdx.x & 31;
    const int r0 = (blockIdx.x * kRowWarps + (threadIdx.x >> 5)) * kHeadRows;
    if (r0 >= ntok) return;
    const int n4 = H >> 7;
    float4 v[kHeadRows][kMaxVec];
#pragma unroll
    for (int i = 0; i < kHeadRows; i++) {
        const int r = min(r0 + i, ntok - 1);          // a row past the end repeats the last one; nothing is stored for it
#pragma unroll
        for (int k = 0; k < kMaxVec; k++) if (k < n4) v[i][k] = load4(x + (size_t)r * H + 4 * (lane + 32 * k));
    }
    float s[kHeadRows][16];
#pragma unroll
    for (int i = 0; i < kHeadRows; i++)
#pragma unroll
        for (int c = 0; c < 16; c++) s[i][c] = 0.f;
#pragma unroll
    for (int k = 0; k < kMaxVec; k++) if (k < n4) {
#pragma unroll
        for (int c = 0; c < 16; c++) if (c < NL) {
            const float4 w = load4(W_c + (size_t)c * H + 4 * (lane + 32 * k));
#pragma unroll
            for (int i = 0; i < kHeadRows; i++)
                s[i][c] = fmaf(v[i][k].w, w.w, fmaf(v[i][k].z, w.z, fmaf(v[i][k].y, w.y, fmaf(v[i][k].x, w.x, s[i][c]))));
        }
    }
    const int cls = lane >> 1;
    const float bias = cls < NL ? __ldg(b_c + cls) : 0.f;
#pragma unroll
    for (int i = 0; i < kHeadRows; i++) {
        float* a = s[i];
#pragma unroll
        for (int half = 8; half >= 1; half >>= 1) {     // lane bit (2 * half) set: keep the upper half of the class sums
            const bool up = (lane & (2 * half)) != 0;
#pragma unroll
            for (int j = 0; j < half; j++) {
                const float keep = up ? a[j + half] : a[j], send = up ? a[j] : a[j + half];
                a[j] = keep + __shfl_xor_sync(0xffffffffu, send, 2 * half);
            }
        }
        float t = a[0] + __shfl_xor_sync(0xffffffffu, a[0], 1) + bias;      // class lane >> 1, summed over all 32 lanes
        const int r = r0 + i;
        if (logits && r < ntok && cls < NL && !(lane & 1)) logits[(size_t)r * NL + cls] = t;
        if (cls >= NL) t = -INFINITY;
        int best_c = cls;
#pragma unroll
        for (int off = 2; off < 32; off <<= 1) {
            const float ot = __shfl_xor_sync(0xffffffffu, t, off);
            const int oc = __shfl_xor_sync(0xffffffffu, best_c, off);
            if (ot > t || (ot == t && oc < best_c)) { t = ot; best_c = oc; }
        }
        if (labels && lane == 0 && r < ntok) labels[r] = best_c;
    }
}

static inline void launch_head_argmax(cudaStream_t st, const float* x, int ntok, int H, const float* W_c, const float* b_c,
                                      int NL, float* logits, int* labels)
{
    if (NL <= 16) {
        const unsigned grid = (unsigned)((ntok + kRowWarps * kHeadRows - 1) / (kRowWarps * kHeadRows));
        head_argmax16_kernel<<<grid, kRowWarps * 32, 0, st>>>(x, ntok, H, W_c, b_c, NL, logits, labels);
    } else {
        const unsigned grid = (unsigned)((ntok + kRowWarps - 1) / kRowWarps);
        head_argmax_kernel<<<grid, kRowWarps * 32, 0, st>>>(x, ntok, H, W_c, b_c, NL, logits, labels);
    }
}

// ---------------------------------------------------------------------------------------------------------
// FP32 SIMT path (BJ configs[0]; TF32 would miss the 1e-4 bound, S7 H5): 64x64x16 tiles, 4x4 per thread
// ---------------------------------------------------------------------------------------------------------
template <int EPI>   // 0: +bias; 1: +bias, erf-GELU; 2: +bias +residual
static __global__ void __launch_bounds__(256) sgemm_tn_kernel(const float* __restrict__ A, const float* __restrict__ W,
                                                       const float* __restrict__ bias, const float* __restrict__ res,
                                                       float* __restrict__ C, int M, int N, int K)
{
    __shared__ float As[16][64 + 4], Ws[16][64 + 4];
    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    const int m0 = blockIdx.y * 64, n0 = blockIdx.x * 64;
    const int lr = tid >> 2, lk = (tid & 3) * 4;
    float acc[4][4] = {};
    for (int k0 = 0; k0 < K; k0 += 16) {
        float4 a = make_float4(0, 0, 0, 0), w = a;
        if (m0 + lr < M && k0 + lk < K) a = load4(A + (size_t)(m0 + lr) * K + k0 + lk);
        if (n0 + lr < N && k0 + lk < K) w = load4(W + (size_t)(n0 + lr) * K + k0 + lk);
        As[lk][lr] = a.x; As[lk + 1][lr] = a.y; As[lk + 2][lr] = a.z; As[lk + 3][lr] = a.w;
        Ws[lk][lr] = w.x; Ws[lk + 1][lr] = w.y; Ws[lk + 2][lr] = w.z; Ws[lk + 3][lr] = w.w;
        __syncthreads();
#pragma unroll
        for (int k = 0; k < 16; k++) {
            const float4 av = *reinterpret_cast<const float4*>(&As[k][ty * 4]);
            const float4 wv = *reinterpret_cast<const float4*>(&Ws[k][tx * 4]);
            const float ar[4] = {av.x, av.y, av.z, av.w}, wr[4] = {wv.x, wv.y, wv.z, wv.w};
#pragma unroll
            for (int i = 0; i < 4; i++)
#pragma unroll
                for (int j = 0; j < 4; j++) acc[i][j] = fmaf(ar[i], wr[j], acc[i][j]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < 4; i++) {
        const int m = m0 + ty * 4 + i;
        if (m >= M) continue;
#pragma unroll
        for (int j = 0; j < 4; j++) {
            const int n = n0 + tx * 4 + j;
            if (n >= N) continue;
            float f = acc[i][j] + __ldg(bias + n);
            if (EPI == 1) f = 0.5f * f * (1.0f + erff(f * 0.70710678118654752f));
            if (EPI == 2) f += res[(size_t)m * N + n];
            C[(size_t)m * N + n] = f;
        }
    }
}

// FP32 varlen attention: one CTA per (sequence, head, block of 32 queries); each warp owns one query at a time; scores in
// shared memory; exact two-pass softmax in FP32.  qkv [T,3H] with q | k | v column blocks; d_head = 64.
// half >= 0 (NEXT-3 local layers): query i sees keys m with |i - m| <= half only.
constexpr int kF32QueryBlock = 32;     // queries per CTA (grid.z = ceil(max sequence length / 32); blocks past a sequence's end exit)
static __global__ void __launch_bounds__(128) attention_f32_kernel(const float* __restrict__ qkv, const int* __restrict__ cu,
                                                            int seq0, int tok0, int H, float* __restrict__ ctx, int half = -1)
{
    __shared__ float sc[4][512];
    __shared__ float qs[4][64];
    const int seq = seq0 + blockIdx.x, head = blockIdx.y;
    const int a = cu[seq] - tok0, n = cu[seq + 1] - cu[seq];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const size_t ld = (size_t)3 * H;
    const float* Q = qkv + (size_t)a * ld + head * 64;
    const float* Kp = Q + H;
    const float* Vp = Q + 2 * H;
    const int i_end = min(n, (int)(blockIdx.z + 1) * kF32QueryBlock);
    for (int i = (int)blockIdx.z * kF32QueryBlock + warp; i < i_end; i += 4) {
        qs[warp][lane] = Q[(size_t)i * ld + lane];
        qs[warp][lane + 32] = Q[(size_t)i * ld + lane + 32];
        __syncwarp();
        const int m_lo = half >= 0 && i - half > 0 ? i - half : 0;
        const int m_hi = half >= 0 && i + half + 1 < n ? i + half + 1 : n;       // exclusive
        float mx = -INFINITY;
        for (int m = m_lo + lane; m < m_hi; m += 32) {
            const float4* kr = reinterpret_cast<const float4*>(Kp + (size_t)m * ld);
            float s = 0.f;
#pragma unroll
            for (int d = 0; d < 16; d++) {
                const float4 kv = __ldg(kr + d);
                s += qs[warp][4 * d] * kv.x + qs[warp][4 * d + 1] * kv.y + qs[warp][4 * d + 2] * kv.z + qs[warp][4 * d + 3] * kv.w;
            }
            s *= 0.125f;
            sc[warp][m] = s;
            mx = fmaxf(mx, s);
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, d));
        float sum = 0.f;
        for (int m = m_lo + lane; m < m_hi; m += 32) { const float e = expf(sc[warp][m] - mx); sc[warp][m] = e; sum += e; }
        sum = warp_sum(sum);
        __syncwarp();
        float o0 = 0.f, o1 = 0.f;
        for (int m = m_lo; m < m_hi; m++) {
            const float p = sc[warp][m];
            o0 = fmaf(p, __ldg(Vp + (size_t)m * ld + lane), o0);
            o1 = fmaf(p, __ldg(Vp + (size_t)m * ld + lane + 32), o1);
        }
        const float inv = 1.0f / sum;
        ctx[(size_t)(a + i) * H + head * 64 + lane] = o0 * inv;
        ctx[(size_t)(a + i) * H + head * 64 + lane + 32] = o1 * inv;
        __syncwarp();
    }
}


// ---- NEXT-3 (ModernBERT-shaped variant, reading D20): position ids, RoPE, GeGLU ---------------------------------------
// pos[t] = index of token t inside its sequence (chunk-local rows; cu points at the chunk's first boundary)
static __global__ void __launch_bounds__(256) token_pos_kernel(const int* __restrict__ cu, int B, int tok0, int ntok, int* __restrict__ pos)
{
    const int t = blockIdx.x * 256 + threadIdx.x;
    if (t >= ntok) return;
    int lo = 0, hi = B;                                   // largest s with cu[s] - tok0 <= t
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (cu[mid] - tok0 <= t) lo = mid; else hi = mid; }
    pos[t] = t - (cu[lo] - tok0);
}

__device__ __forceinline__ float to_f32(float v) { return v; }
__device__ __forceinline__ float to_f32(__nv_bfloat16 v) { return __bfloat162float(v); }
__device__ __forceinline__ void from_f32(float& d, float v) { d = v; }
__device__ __forceinline__ void from_f32(__nv_bfloat16& d, float v) { d = __float2bfloat16_rn(v); }

// 16 bytes of T (4 floats or 8 bf16) moved as one vector
template <class T> struct Vec16 {
    static constexpr int N = 16 / (int)sizeof(T);
    T v[N];
    __device__ __forceinline__ void load(const T* p) { *reinterpret_cast<uint4*>(v) = *reinterpret_cast<const uint4*>(p); }
    __device__ __forceinline__ void store(T* p) const { *reinterpret_cast<uint4*>(p) = *reinterpret_cast<const uint4*>(v); }
};

// In place on the q and k column blocks of qkv [ntok, 3H]: pair (i, i + 32) of every head turns by the angle whose
// (cos, sin) sits in table[pos][i] (float2 [max_pos][32], built in double at weights load).  A thread owns N consecutive
// pairs of one head (N = 4 FP32 / 8 BF16): two 16-byte loads, two 16-byte stores, all coalesced.
template <class T>
static __global__ void __launch_bounds__(256) rope_kernel(T* __restrict__ qkv, const int* __restrict__ pos, int ntok, int H,
                                                           const float2* __restrict__ table)
{
    constexpr int N = Vec16<T>::N;
    const int per_head = 32 / N, per_tok = 2 * (H >> 6) * per_head;       // q heads then k heads: columns [0, 2H)
    const long long gid = (long long)blockIdx.x * 256 + threadIdx.x;
    const int t = (int)(gid / per_tok);
    if (t >= ntok) return;
    const int slot = (int)(gid - (long long)t * per_tok);
    const int hh = slot / per_head, i0 = (slot - hh * per_head) * N;
    T* p = qkv + (size_t)t * 3 * H + hh * 64 + i0;
    const float2* cs = table + (size_t)pos[t] * 32 + i0;
    Vec16<T> x1, x2;
    x1.load(p); x2.load(p + 32);
#pragma unroll
    for (int e = 0; e < N; e++) {
        const float2 r = __ldg(cs + e);
        const float a = to_f32(x1.v[e]), b = to_f32(x2.v[e]);
        from_f32(x1.v[e], a * r.x - b * r.y);
        from_f32(x2.v[e], b * r.x + a * r.y);
    }
    x1.store(p); x2.store(p + 32);
}

// f[t, j] = gelu(u[t, j]) * u[t, F + j] (erf GELU), u [ntok, 2F]; 16 bytes of the activation per thread (F % 8 == 0)
template <class T>
static __global__ void __launch_bounds__(256) geglu_kernel(const T* __restrict__ u, T* __restrict__ f, int ntok, int F)
{
    constexpr int N = Vec16<T>::N;
    const int per_tok = F / N;
    const long long gid = (long long)blockIdx.x * 256 + threadIdx.x;
    const int t = (int)(gid / per_tok);
    if (t >= ntok) return;
    const int j = (int)(gid - (long long)t * per_tok) * N;
    Vec16<T> a, g;
    a.load(u + (size_t)t * 2 * F + j); g.load(u + (size_t)t * 2 * F + F + j);
#pragma unroll
    for (int e = 0; e < N; e++) {
        const float z = to_f32(a.v[e]);
        from_f32(a.v[e], 0.5f * z * (1.0f + erff(z * 0.70710678118654752f)) * to_f32(g.v[e]));
    }
    a.store(f + (size_t)t * F + j);
}

}  // namespace enc
