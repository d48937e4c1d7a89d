// stream_probe.cu -- the paper's buffer-copy micro-benchmark (Fig. 5; SURVEY.md
// section 2 row K11), restated for B200 as the library's own HBM roofline probe.
//
// The paper copied a 100 MiB buffer with kernels whose threads move one element each, for the
// element types float, double, float4 (= complex double), an SU(3) matrix and a spinor, and
// found that only the 16-byte element reaches the device's bandwidth while whole-struct (array of
// structures) elements fall far behind.  That finding fixed its storage
// format, and ours.  Here the same experiment:
//   elem 0 float (4 B), 1 double (8 B), 2 16-byte vector: element i of an array, one per access
//   elem 3 su3 AoS (144 B), 4 spinor AoS (192 B): thread <-> struct, 9 / 12 16-byte words each
// and two more access mixes on the plain element types, which bracket the hopping kernel better
// than a 1:1 copy does (it reads 7 bytes for every byte it writes, 1344 : 192):
//   mode 0 COPY  dst[i] = src[i]                                    reads B, writes B
//   mode 1 READ  XOR of all 8-byte words, one word per CTA to dst   reads B, writes ~nothing
//   mode 2 MIX71 dst[i] = src[i] ^ src[n+i] ^ ... ^ src[6n+i]       reads B, writes B/7
// Everything is bit-wise (integer loads, XOR), so the result is exact for any byte pattern and
// the test can state it in one line.  Loads and stores are streaming (ld.global.cs / st.global.cs):
// nothing is reused.
#include "lqcd_internal.h"

#include <cstdint>

namespace lqcd {
namespace {

constexpr int kThreads = 256;
constexpr int kUnroll = 2;

template <typename E> __device__ __forceinline__ E ld_cs(const E* p) { return __ldcs(p); }
template <typename E> __device__ __forceinline__ void st_cs(E* p, E v) { __stcs(p, v); }

__device__ __forceinline__ void xor_into(uint32_t& a, uint32_t b) { a ^= b; }
__device__ __forceinline__ void xor_into(uint2& a, uint2 b) { a.x ^= b.x; a.y ^= b.y; }
__device__ __forceinline__ void xor_into(uint4& a, uint4 b) { a.x ^= b.x; a.y ^= b.y; a.z ^= b.z; a.w ^= b.w; }

// XOR of the 8-byte words of a value; a 4-byte element counts as the low or high half of the
// 8-byte word it lies in (element index parity)
__device__ __forceinline__ unsigned long long fold(uint32_t v, size_t i) {
    return (i & 1) ? ((unsigned long long)v << 32) : (unsigned long long)v;
}
__device__ __forceinline__ unsigned long long fold(uint2 v, size_t) {
    return ((unsigned long long)v.y << 32) | v.x;
}
__device__ __forceinline__ unsigned long long fold(uint4 v, size_t) {
    return (((unsigned long long)v.y << 32) | v.x) ^ (((unsigned long long)v.w << 32) | v.z);
}

// n = number of elements written (COPY, MIX71) or read (READ); tiles of kUnroll * kThreads elements,
// the kUnroll (x 7) loads of a thread issued before their uses; the loop runs once unless the grid is capped
template <typename E, int MODE>
__global__ void __launch_bounds__(kThreads) stream_kernel(const E* __restrict__ src, E* __restrict__ dst, size_t n) {
    const size_t tile = (size_t)kUnroll * kThreads;
    unsigned long long acc = 0;
    for (size_t base = (size_t)blockIdx.x * tile; base < n; base += (size_t)gridDim.x * tile) {
        E v[kUnroll];
#pragma unroll
        for (int k = 0; k < kUnroll; ++k) {
            const size_t i = base + (size_t)k * kThreads + threadIdx.x;
            if (i < n) {
                v[k] = ld_cs(src + i);
                if (MODE == 2) {
#pragma unroll
                    for (int pl = 1; pl < 7; ++pl) xor_into(v[k], ld_cs(src + (size_t)pl * n + i));
                }
            }
        }
#pragma unroll
        for (int k = 0; k < kUnroll; ++k) {
            const size_t i = base + (size_t)k * kThreads + threadIdx.x;
            if (i < n) {
                if (MODE == 1) acc ^= fold(v[k], i);
                else st_cs(dst + i, v[k]);
            }
        }
    }
    if (MODE == 1) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc ^= __shfl_xor_sync(0xffffffffu, acc, o);
        __shared__ unsigned long long part[kThreads / 32];
        if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = acc;
        __syncthreads();
        if (threadIdx.x == 0) {
            unsigned long long t = 0;
#pragma unroll
            for (int w = 0; w < kThreads / 32; ++w) t ^= part[w];
            reinterpret_cast<unsigned long long*>(dst)[blockIdx.x] = t;
        }
    }
}

// array of structures: thread <-> struct of W 16-byte words (the layout the paper started from,
// PAPER.md:209-217); lanes of a warp are W * 16 bytes apart
template <int W>
__global__ void __launch_bounds__(kThreads) aos_copy_kernel(const uint4* __restrict__ src, uint4* __restrict__ dst,
                                                            size_t n_struct) {
    for (size_t s = (size_t)blockIdx.x * kThreads + threadIdx.x; s < n_struct; s += (size_t)gridDim.x * kThreads) {
        uint4 v[W];
#pragma unroll
        for (int j = 0; j < W; ++j) v[j] = ld_cs(src + s * W + j);
#pragma unroll
        for (int j = 0; j < W; ++j) st_cs(dst + s * W + j, v[j]);
    }
}

// FP64 pipe probe ("measure with a DFMA micro-benchmark"): every thread runs
// 8 independent chains x <- fma(x, a, b), `iters` links each; out[t] = sum of its 8 chains, chain c
// starting at t + c.  2 x 8 x iters flop per thread.
__global__ void __launch_bounds__(kThreads) dfma_kernel(double a, double b, int iters, double* __restrict__ out) {
    const int t = blockIdx.x * kThreads + threadIdx.x;
    double x[8];
#pragma unroll
    for (int c = 0; c < 8; ++c) x[c] = (double)(t + c);
#pragma unroll 4
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int c = 0; c < 8; ++c) x[c] = fma(x[c], a, b);
    }
    out[t] = ((x[0] + x[1]) + (x[2] + x[3])) + ((x[4] + x[5]) + (x[6] + x[7]));
}

template <typename E>
cudaError_t launch_typed(int mode, const void* src, void* dst, size_t n, int grid, cudaStream_t st) {
    const E* s = reinterpret_cast<const E*>(src);
    E* d = reinterpret_cast<E*>(dst);
    if (mode == 0)      stream_kernel<E, 0><<<grid, kThreads, 0, st>>>(s, d, n);
    else if (mode == 1) stream_kernel<E, 1><<<grid, kThreads, 0, st>>>(s, d, n);
    else                stream_kernel<E, 2><<<grid, kThreads, 0, st>>>(s, d, n);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_stream_probe(int elem, int mode, const void* src, void* dst, size_t bytes, cudaStream_t st) {
    static const size_t elem_bytes[5] = {4, 8, 16, 144, 192};
    const size_t read_elems = bytes / elem_bytes[elem];
    const size_t n = (mode == 2) ? read_elems / 7 : read_elems;
    if (n == 0) return cudaSuccess;
    count_launch();
    ProfScope prof(4, st);
    // READ leaves one word per CTA, so its grid is fixed (grid-stride loop); COPY and MIX71 take one CTA per
    // tile: measured at 2.1 GB on B200, one tile per CTA copies at 6.9 TB/s, the same kernel as a
    // grid-stride loop over 1184 CTAs at 5.9 (the memcpy engine: 6.5).  Tiles of 2 elements per thread
    // beat 1, 4 and 8 (MIX71: 7.06 TB/s against 7.19 / 6.93 / 6.51 for 1 / 4 / 8; COPY 6.92 against 6.64 / 6.85 / 6.21).
    // Cache hints (.cs on loads, on stores, on neither) move the plain element types by < 2%.
    const size_t per_cta = (elem >= 3) ? (size_t)kThreads : (size_t)kUnroll * kThreads;
    const size_t tiles = (n + per_cta - 1) / per_cta;
    if (tiles > 0x7fffffffull) return cudaErrorInvalidValue;
    const int grid = (mode == 1) ? kStreamProbeBlocks : (int)tiles;
    switch (elem) {
        case 0: return launch_typed<uint32_t>(mode, src, dst, n, grid, st);
        case 1: return launch_typed<uint2>(mode, src, dst, n, grid, st);
        case 2: return launch_typed<uint4>(mode, src, dst, n, grid, st);
        case 3: aos_copy_kernel<9><<<grid, kThreads, 0, st>>>((const uint4*)src, (uint4*)dst, n); break;
        default: aos_copy_kernel<12><<<grid, kThreads, 0, st>>>((const uint4*)src, (uint4*)dst, n); break;
    }
    return cudaGetLastError();
}

cudaError_t launch_dfma_probe(double a, double b, int iters, double* out, cudaStream_t st) {
    count_launch();
    ProfScope prof(4, st);
    dfma_kernel<<<kStreamProbeBlocks, kThreads, 0, st>>>(a, b, iters, out);
    return cudaGetLastError();
}

}  // namespace lqcd
