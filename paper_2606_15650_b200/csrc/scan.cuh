// scan.cuh -- device-wide exclusive transform-scan in three launches (tile reduce, aggregate scan,
// tile apply).  Inputs come from a functor (recomputed in pass 3, never stored) and results go to
// a functor, so callers fuse their own work into the passes.  HBM-bound helper used by the BIO
// decode (A9), span gather (A10) and pseudonymize (A11-A13) stages.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace scan {

constexpr int kThreads = 256;
constexpr int kItems = 8;
constexpr int kTile = kThreads * kItems;   // 2048 items per CTA

struct I64x3 { long long a, b, c; };
struct SumI64x3 {
    __device__ __forceinline__ I64x3 operator()(const I64x3& x, const I64x3& y) const {
        return I64x3{x.a + y.a, x.b + y.b, x.c + y.c};
    }
    __device__ __forceinline__ static I64x3 identity() { return I64x3{0, 0, 0}; }
};
struct SumI64 {
    __device__ __forceinline__ long long operator()(long long x, long long y) const { return x + y; }
    __device__ __forceinline__ static long long identity() { return 0; }
};
struct MaxI32 {
    __device__ __forceinline__ int operator()(int x, int y) const { return x > y ? x : y; }
    __device__ __forceinline__ static int identity() { return -1; }
};

__device__ __forceinline__ int shfl_up(int v, int d) { return __shfl_up_sync(0xffffffffu, v, d); }
__device__ __forceinline__ long long shfl_up(long long v, int d) { return __shfl_up_sync(0xffffffffu, v, d); }
__device__ __forceinline__ I64x3 shfl_up(const I64x3& v, int d) {
    return I64x3{__shfl_up_sync(0xffffffffu, v.a, d), __shfl_up_sync(0xffffffffu, v.b, d),
                 __shfl_up_sync(0xffffffffu, v.c, d)};
}

// Exclusive scan of one value per thread across the CTA; returns the exclusive prefix and the CTA total.
template <class T, class Op>
__device__ __forceinline__ T block_exclusive(T v, Op op, T* smem /*[kThreads/32 + 1]*/, T& total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    T incl = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        T o = shfl_up(incl, d);
        if (lane >= d) incl = op(o, incl);
    }
    if (lane == 31) smem[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        T w = lane < kThreads / 32 ? smem[lane] : Op::identity();
        T wi = w;
#pragma unroll
        for (int d = 1; d < kThreads / 32; d <<= 1) {
            T o = shfl_up(wi, d);
            if (lane >= d) wi = op(o, wi);
        }
        if (lane < kThreads / 32) smem[lane] = wi;          // inclusive warp totals
    }
    __syncthreads();
    T excl = shfl_up(incl, 1);
    if (lane == 0) excl = Op::identity();
    if (warp > 0) excl = op(smem[warp - 1], excl);
    total = smem[kThreads / 32 - 1];
    __syncthreads();
    return excl;
}

// n may live on the device (d_n != nullptr): the grid is sized for n_max and tiles past *d_n idle.
template <class T, class Op, class In>
__global__ void __launch_bounds__(kThreads) tile_reduce(In in, long long n_max, const int* d_n, T* agg) {
    __shared__ T smem[kThreads / 32 + 1];
    const long long n = d_n ? (long long)min((long long)*d_n, n_max) : n_max;
    const long long base = (long long)blockIdx.x * kTile + (long long)threadIdx.x * kItems;
    Op op;
    T acc = Op::identity();
#pragma unroll
    for (int k = 0; k < kItems; k++)
        if (base + k < n) acc = op(acc, in(base + k));
    T total;
    block_exclusive<T, Op>(acc, op, smem, total);
    if (threadIdx.x == 0) agg[blockIdx.x] = total;
}

// Single CTA: agg[0..nb) -> exclusive prefixes in place, agg[nb] = grand total.
template <class T, class Op>
__global__ void __launch_bounds__(kThreads) scan_aggregates(T* agg, int nb) {
    __shared__ T smem[kThreads / 32 + 1];
    Op op;
    T carry = Op::identity();
    for (int b0 = 0; b0 < nb; b0 += kThreads) {
        int i = b0 + threadIdx.x;
        T v = i < nb ? agg[i] : Op::identity();
        T total;
        T excl = block_exclusive<T, Op>(v, op, smem, total);
        if (i < nb) agg[i] = op(carry, excl);
        carry = op(carry, total);
    }
    if (threadIdx.x == 0) agg[nb] = carry;
}

template <class T, class Op, class In, class Out>
__global__ void __launch_bounds__(kThreads) tile_apply(In in, Out out, long long n_max, const int* d_n, const T* agg) {
    __shared__ T smem[kThreads / 32 + 1];
    const long long n = d_n ? (long long)min((long long)*d_n, n_max) : n_max;
    const long long base = (long long)blockIdx.x * kTile + (long long)threadIdx.x * kItems;
    Op op;
    T v[kItems];
    T acc = Op::identity();
#pragma unroll
    for (int k = 0; k < kItems; k++) {
        v[k] = (base + k < n) ? in(base + k) : Op::identity();
        acc = op(acc, v[k]);
    }
    T total;
    T excl = block_exclusive<T, Op>(acc, op, smem, total);
    T run = op(agg[blockIdx.x], excl);
#pragma unroll
    for (int k = 0; k < kItems; k++) {
        if (base + k < n) out(base + k, run, v[k]);
        run = op(run, v[k]);
    }
}

inline int num_tiles(long long n) { return (int)((n + kTile - 1) / kTile); }
// bytes of aggregate scratch for n items
template <class T> inline size_t agg_bytes(long long n) { return (size_t)(num_tiles(n) + 1) * sizeof(T); }

// Runs passes 1+2; the caller launches tile_apply itself (possibly after looking at agg[nb]).
template <class T, class Op, class In>
inline void reduce_and_scan(In in, long long n_max, const int* d_n, T* agg, cudaStream_t st) {
    int nb = num_tiles(n_max);
    if (nb > 0) tile_reduce<T, Op, In><<<nb, kThreads, 0, st>>>(in, n_max, d_n, agg);
    scan_aggregates<T, Op><<<1, kThreads, 0, st>>>(agg, nb);
}
template <class T, class Op, class In, class Out>
inline void apply(In in, Out out, long long n_max, const int* d_n, const T* agg, cudaStream_t st) {
    int nb = num_tiles(n_max);
    if (nb > 0) tile_apply<T, Op, In, Out><<<nb, kThreads, 0, st>>>(in, out, n_max, d_n, agg);
}

}  // namespace scan
