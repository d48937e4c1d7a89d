// pack.cu -- canonical (array-of-structures, complex double; include/lqcd.h) <-> internal
// structure-of-arrays layout (lqcd_internal.h).  The paper hides the same conversion
// behind accessor functions and performs it on host<->device copies;
// here it is a device kernel so that the interchange format never reaches the hot path.
#include "lqcd_internal.h"

namespace lqcd {
namespace {

constexpr int PBLOCK = 128;

__device__ __forceinline__ int site_r(const Geometry& g, int e, int parity) {
    int t = e / g.N0h;
    const int x1 = t % g.N1; t /= g.N1;
    const int x2 = t % g.N2;
    const int x3 = t / g.N2;
    return (x1 + x2 + x3 + parity) & 1;
}

// one thread per (parity, mu, e): reads the 144-byte link U[lex][mu], lex = 2e + r, and writes
// it into group e >> 5, lane e & 31 of the grouped layout (lqcd_internal.h)
template <typename T, int RECON>
__global__ void __launch_bounds__(PBLOCK) pack_gauge_kernel(Geometry g, const double2* __restrict__ canon,
                                                            void* __restrict__ internal) {
    const size_t tid = (size_t)blockIdx.x * PBLOCK + threadIdx.x;
    const size_t Vh = g.Vh;
    if (tid >= 8 * Vh) return;
    const int e = (int)(tid % Vh);
    const int pm = (int)(tid / Vh);  // parity * 4 + mu
    const int parity = pm >> 2, mu = pm & 3;
    const size_t lex = 2 * (size_t)e + site_r(g, e, parity);
    const double2* src = canon + (lex * 4 + mu) * 9;
    double2 u[9];
#pragma unroll
    for (int j = 0; j < 9; ++j) u[j] = src[j];
    const size_t grp = gauge_block(parity, mu, g.Gg, e >> 5);
    const int lane = e & 31;
    if (sizeof(T) == 8) {
        double2* dst = (double2*)internal + grp * ((RECON / 2) * 32) + lane;
#pragma unroll
        for (int j = 0; j < RECON / 2; ++j) dst[j * 32] = u[j];
    } else if (RECON == 12) {
        float4* dst = (float4*)internal + grp * (3 * 32) + lane;
#pragma unroll
        for (int j = 0; j < 3; ++j)
            dst[j * 32] = make_float4((float)u[2 * j].x, (float)u[2 * j].y, (float)u[2 * j + 1].x,
                                      (float)u[2 * j + 1].y);
    } else {
        float* blk = (float*)internal + grp * (18 * 32);
        float4* dst = (float4*)blk + lane;
#pragma unroll
        for (int j = 0; j < 4; ++j)
            dst[j * 32] = make_float4((float)u[2 * j].x, (float)u[2 * j].y, (float)u[2 * j + 1].x,
                                      (float)u[2 * j + 1].y);
        ((float2*)(blk + 16 * 32))[lane] = make_float2((float)u[8].x, (float)u[8].y);
    }
}

// internal -> canonical U[lex][mu] (row 2 rebuilt as conj(row0 x row1) for 12-real storage)
template <typename T, int RECON>
__global__ void __launch_bounds__(PBLOCK) unpack_gauge_kernel(Geometry g, const void* __restrict__ internal,
                                                              double2* __restrict__ canon) {
    const size_t tid = (size_t)blockIdx.x * PBLOCK + threadIdx.x;
    const size_t Vh = g.Vh;
    if (tid >= 8 * Vh) return;
    const int e = (int)(tid % Vh);
    const int pm = (int)(tid / Vh);
    const int parity = pm >> 2, mu = pm & 3;
    const size_t lex = 2 * (size_t)e + site_r(g, e, parity);
    const size_t grp = gauge_block(parity, mu, g.Gg, e >> 5);
    const int lane = e & 31;
    double2 u[9];
    if (sizeof(T) == 8) {
        const double2* src = (const double2*)internal + grp * ((RECON / 2) * 32) + lane;
#pragma unroll
        for (int j = 0; j < RECON / 2; ++j) u[j] = src[j * 32];
    } else if (RECON == 12) {
        const float4* src = (const float4*)internal + grp * (3 * 32) + lane;
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            const float4 v = src[j * 32];
            u[2 * j] = make_double2(v.x, v.y);
            u[2 * j + 1] = make_double2(v.z, v.w);
        }
    } else {
        const float* blk = (const float*)internal + grp * (18 * 32);
        const float4* src = (const float4*)blk + lane;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const float4 v = src[j * 32];
            u[2 * j] = make_double2(v.x, v.y);
            u[2 * j + 1] = make_double2(v.z, v.w);
        }
        const float2 w = ((const float2*)(blk + 16 * 32))[lane];
        u[8] = make_double2(w.x, w.y);
    }
    if (RECON == 12) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {   // conj(row0 x row1)_c, in the storage precision's values widened to double
            const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
            const double2 a = u[c1], b = u[3 + c2], cc = u[c2], d = u[3 + c1];
            const double re = (a.x * b.x - a.y * b.y) - (cc.x * d.x - cc.y * d.y);
            const double im = (a.x * b.y + a.y * b.x) - (cc.x * d.y + cc.y * d.x);
            u[6 + c] = make_double2(re, -im);
        }
    }
    double2* dst = canon + (lex * 4 + mu) * 9;
#pragma unroll
    for (int j = 0; j < 9; ++j) dst[j] = u[j];
}

// canonical half spinor psi_p[e][c] -> internal s[e >> 5][c][e & 31]; pad sites get zeros
template <typename T>
__global__ void __launch_bounds__(PBLOCK) pack_spinor_kernel(int Vh, int G, const double2* __restrict__ canon,
                                                             void* __restrict__ internal) {
    const int e = blockIdx.x * PBLOCK + threadIdx.x;
    if (e >= G * 32) return;
    double2 s[12];
    if (e < Vh) {
        const double2* src = canon + (size_t)e * 12;
#pragma unroll
        for (int c = 0; c < 12; ++c) s[c] = src[c];
    } else {
#pragma unroll
        for (int c = 0; c < 12; ++c) s[c] = make_double2(0.0, 0.0);
    }
    if (sizeof(T) == 8) {
        double2* dst = (double2*)internal + (size_t)(e >> 5) * (12 * 32) + (e & 31);
#pragma unroll
        for (int c = 0; c < 12; ++c) dst[c * 32] = s[c];
    } else {
        float4* dst = (float4*)internal + (size_t)(e >> 5) * (6 * 32) + (e & 31);
#pragma unroll
        for (int k = 0; k < 6; ++k)
            dst[k * 32] = make_float4((float)s[2 * k].x, (float)s[2 * k].y, (float)s[2 * k + 1].x,
                                      (float)s[2 * k + 1].y);
    }
}

template <typename T>
__global__ void __launch_bounds__(PBLOCK) unpack_spinor_kernel(int Vh, const void* __restrict__ internal,
                                                               double2* __restrict__ canon) {
    const int e = blockIdx.x * PBLOCK + threadIdx.x;
    if (e >= Vh) return;
    double2 s[12];
    if (sizeof(T) == 8) {
        const double2* src = (const double2*)internal + (size_t)(e >> 5) * (12 * 32) + (e & 31);
#pragma unroll
        for (int c = 0; c < 12; ++c) s[c] = src[c * 32];
    } else {
        const float4* src = (const float4*)internal + (size_t)(e >> 5) * (6 * 32) + (e & 31);
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            const float4 v = src[k * 32];
            s[2 * k] = make_double2(v.x, v.y);
            s[2 * k + 1] = make_double2(v.z, v.w);
        }
    }
    double2* dst = canon + (size_t)e * 12;
#pragma unroll
    for (int c = 0; c < 12; ++c) dst[c] = s[c];
}

}  // namespace

cudaError_t launch_pack_gauge(int precision, int recon, const Geometry& g, const void* canon,
                              void* internal, cudaStream_t st) {
    const size_t n = 8 * (size_t)g.Vh;
    const int grid = (int)((n + PBLOCK - 1) / PBLOCK);
    count_launch();
    ProfScope prof(4, st);
    const double2* c = (const double2*)canon;
    if (precision == 0) {
        if (recon == 12) pack_gauge_kernel<double, 12><<<grid, PBLOCK, 0, st>>>(g, c, internal);
        else             pack_gauge_kernel<double, 18><<<grid, PBLOCK, 0, st>>>(g, c, internal);
    } else {
        if (recon == 12) pack_gauge_kernel<float, 12><<<grid, PBLOCK, 0, st>>>(g, c, internal);
        else             pack_gauge_kernel<float, 18><<<grid, PBLOCK, 0, st>>>(g, c, internal);
    }
    return cudaGetLastError();
}

cudaError_t launch_unpack_gauge(int precision, int recon, const Geometry& g, const void* internal, void* canon,
                                cudaStream_t st) {
    const size_t n = 8 * (size_t)g.Vh;
    const int grid = (int)((n + PBLOCK - 1) / PBLOCK);
    count_launch();
    ProfScope prof(4, st);
    double2* c = (double2*)canon;
    if (precision == 0) {
        if (recon == 12) unpack_gauge_kernel<double, 12><<<grid, PBLOCK, 0, st>>>(g, internal, c);
        else             unpack_gauge_kernel<double, 18><<<grid, PBLOCK, 0, st>>>(g, internal, c);
    } else {
        if (recon == 12) unpack_gauge_kernel<float, 12><<<grid, PBLOCK, 0, st>>>(g, internal, c);
        else             unpack_gauge_kernel<float, 18><<<grid, PBLOCK, 0, st>>>(g, internal, c);
    }
    return cudaGetLastError();
}

cudaError_t launch_pack_spinor(int precision, const Geometry& g, const void* canon, void* internal,
                               int /*parity*/, cudaStream_t st) {
    const int grid = (g.G * 32 + PBLOCK - 1) / PBLOCK;
    count_launch();
    ProfScope prof(4, st);
    if (precision == 0) pack_spinor_kernel<double><<<grid, PBLOCK, 0, st>>>(g.Vh, g.G, (const double2*)canon, internal);
    else                pack_spinor_kernel<float><<<grid, PBLOCK, 0, st>>>(g.Vh, g.G, (const double2*)canon, internal);
    return cudaGetLastError();
}

cudaError_t launch_unpack_spinor(int precision, const Geometry& g, const void* internal, void* canon,
                                 int /*parity*/, cudaStream_t st) {
    const int grid = (g.Vh + PBLOCK - 1) / PBLOCK;
    count_launch();
    ProfScope prof(4, st);
    if (precision == 0) unpack_spinor_kernel<double><<<grid, PBLOCK, 0, st>>>(g.Vh, internal, (double2*)canon);
    else                unpack_spinor_kernel<float><<<grid, PBLOCK, 0, st>>>(g.Vh, internal, (double2*)canon);
    return cudaGetLastError();
}

}  // namespace lqcd
