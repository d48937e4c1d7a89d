// site_ops.cuh -- per-site device building blocks shared by the hopping kernel (hopping.cu) and
// the fermion-force kernel (force.cu): field access in the grouped layout (lqcd_internal.h),
// 12-real link reconstruction, the spin-projection table, SU(3) x half-spinor products.
//
// Spin projection table (gamma basis of include/lqcd.h; reading G4),
// (1 + S gamma_mu) psi = (h0, h1, conj(c0) h0 or h1 ...):
//   h0 = psi_0 + c0 psi_j0,  h1 = psi_1 + c1 psi_j1,  j1 = 5 - j0,
//   row j0 of the result = conj(c0) h0, row j1 = conj(c1) h1.
//   S = -1:  mu=x: j0=3 c0=+i c1=+i | y: j0=3 c0=+1 c1=-1 | z: j0=2 c0=+i c1=-i | t: j0=2 c0=-1 c1=-1
//   S = +1:  all c negated.
#pragma once

#include "lqcd_internal.h"

namespace lqcd {
namespace {

__device__ __forceinline__ double fma_(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ float fma_(float a, float b, float c) { return fmaf(a, b, c); }

// arguments of a hopping launch (hopping.cu, hopping_staged.cu)
struct HopArgs {
    const void* gauge;
    const void* in;
    void* out;
    const void* aux;
    const void* dotw;   // MODE 4, 5: the field w of <w, out>
    const void* dotw2;  // MODE 5: a second such field
    Geometry g;
    Epilogue ep;
    int out_parity;
    int reverse;   // traverse the sites in descending order (see lqcd_internal.h "snake order")
    Reduction red;
    CgScalars* scal;
    SiteRange rg;
    // variant 6 (TILE): a CTA of four warps takes the four groups {g, g + Gy, g + Gy N2, g + Gy (N2 + 1)} -- the
    // groups of a 2 x 2 block in (z, t) -- instead of four consecutive groups; Gy = groups per z plane
    int tile_gy, tile_n2h;   // Gy and N2 / 2 (0: linear order)
    int general_phases;      // variant 7: the branch-per-hop kernel even where every phase is +-1 (for A/B timing)
};

// ----------------------------------------------------------------------------- field access
// Grouped layout (lqcd_internal.h): one address per site, compile-time offsets per component.
__device__ __forceinline__ void load_spinor(const void* base, int idx, double (&psi)[24]) {
    const double2* p = reinterpret_cast<const double2*>(base) + (size_t)(idx >> 5) * (12 * 32) + (idx & 31);
#pragma unroll
    for (int c = 0; c < 12; ++c) {
        const double2 v = __ldg(p + c * 32);
        psi[2 * c] = v.x;
        psi[2 * c + 1] = v.y;
    }
}
__device__ __forceinline__ void load_spinor(const void* base, int idx, float (&psi)[24]) {
    const float4* p = reinterpret_cast<const float4*>(base) + (size_t)(idx >> 5) * (6 * 32) + (idx & 31);
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        const float4 v = __ldg(p + k * 32);
        psi[4 * k] = v.x;
        psi[4 * k + 1] = v.y;
        psi[4 * k + 2] = v.z;
        psi[4 * k + 3] = v.w;
    }
}
// plain (coherent) loads for a field the same kernel also writes (MODE 3 reads r before storing it)
__device__ __forceinline__ void load_spinor_rw(const void* base, int idx, double (&psi)[24]) {
    const double2* p = reinterpret_cast<const double2*>(base) + (size_t)(idx >> 5) * (12 * 32) + (idx & 31);
#pragma unroll
    for (int c = 0; c < 12; ++c) {
        const double2 v = p[c * 32];
        psi[2 * c] = v.x;
        psi[2 * c + 1] = v.y;
    }
}
__device__ __forceinline__ void load_spinor_rw(const void* base, int idx, float (&psi)[24]) {
    const float4* p = reinterpret_cast<const float4*>(base) + (size_t)(idx >> 5) * (6 * 32) + (idx & 31);
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        const float4 v = p[k * 32];
        psi[4 * k] = v.x;
        psi[4 * k + 1] = v.y;
        psi[4 * k + 2] = v.z;
        psi[4 * k + 3] = v.w;
    }
}
__device__ __forceinline__ void store_spinor(void* base, int idx, const double (&o)[24]) {
    double2* p = reinterpret_cast<double2*>(base) + (size_t)(idx >> 5) * (12 * 32) + (idx & 31);
#pragma unroll
    for (int c = 0; c < 12; ++c) p[c * 32] = make_double2(o[2 * c], o[2 * c + 1]);
}
__device__ __forceinline__ void store_spinor(void* base, int idx, const float (&o)[24]) {
    float4* p = reinterpret_cast<float4*>(base) + (size_t)(idx >> 5) * (6 * 32) + (idx & 31);
#pragma unroll
    for (int k = 0; k < 6; ++k)
        p[k * 32] = make_float4(o[4 * k], o[4 * k + 1], o[4 * k + 2], o[4 * k + 3]);
}

// third row of an SU(3) matrix from the first two: row2 = conj(row0 x row1)  (G9)
template <typename T>
__device__ __forceinline__ void reconstruct_row2(T (&u)[18]) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
        // (row0 x row1)_c = u0[c1] u1[c2] - u0[c2] u1[c1]
        const T ar = u[2 * c1], ai = u[2 * c1 + 1], br = u[6 + 2 * c2], bi = u[6 + 2 * c2 + 1];
        const T cr = u[2 * c2], ci = u[2 * c2 + 1], dr = u[6 + 2 * c1], di = u[6 + 2 * c1 + 1];
        const T re = fma_(ci, di, fma_(-cr, dr, fma_(-ai, bi, ar * br)));
        const T im = fma_(-ci, dr, fma_(-cr, di, fma_(ai, br, ar * bi)));
        u[12 + 2 * c] = re;
        u[12 + 2 * c + 1] = -im;
    }
}

template <int RECON>
__device__ __forceinline__ void load_link(const void* gauge, int G, int par, int mu, int idx,
                                          double (&u)[18]) {
    const double2* p = reinterpret_cast<const double2*>(gauge) +
                       gauge_block(par, mu, G, idx >> 5) * ((RECON / 2) * 32) + (idx & 31);
#pragma unroll
    for (int j = 0; j < RECON / 2; ++j) {
        const double2 v = __ldcs(p + j * 32);
        u[2 * j] = v.x;
        u[2 * j + 1] = v.y;
    }
    if (RECON == 12) reconstruct_row2(u);
}
template <int RECON>
__device__ __forceinline__ void load_link(const void* gauge, int G, int par, int mu, int idx,
                                          float (&u)[18]) {
    if (RECON == 12) {
        const float4* p = reinterpret_cast<const float4*>(gauge) +
                          gauge_block(par, mu, G, idx >> 5) * (3 * 32) + (idx & 31);
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            const float4 v = __ldcs(p + j * 32);
            u[4 * j] = v.x;
            u[4 * j + 1] = v.y;
            u[4 * j + 2] = v.z;
            u[4 * j + 3] = v.w;
        }
        reconstruct_row2(u);
    } else {
        const float* blk = reinterpret_cast<const float*>(gauge) +
                           gauge_block(par, mu, G, idx >> 5) * (18 * 32);
        const float4* p = reinterpret_cast<const float4*>(blk) + (idx & 31);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const float4 v = __ldcs(p + j * 32);
            u[4 * j] = v.x;
            u[4 * j + 1] = v.y;
            u[4 * j + 2] = v.z;
            u[4 * j + 3] = v.w;
        }
        const float2 w = __ldcs(reinterpret_cast<const float2*>(blk + 16 * 32) + (idx & 31));
        u[16] = w.x;
        u[17] = w.y;
    }
}

// ----------------------------------------------------------------------------- spin algebra
// o = a + c b with c = i^C  (C: 0 -> +1, 1 -> +i, 2 -> -1, 3 -> -i)
template <int C, typename T>
__device__ __forceinline__ void add_c(T& ore, T& oim, T are, T aim, T bre, T bim) {
    if (C == 0) { ore = are + bre; oim = aim + bim; }
    if (C == 1) { ore = are - bim; oim = aim + bre; }
    if (C == 2) { ore = are - bre; oim = aim - bim; }
    if (C == 3) { ore = are + bim; oim = aim - bre; }
}

template <int MU, int S>
struct Proj {
    static constexpr int j0 = (MU < 2) ? 3 : 2;
    static constexpr int j1 = 5 - j0;
    static constexpr int c0m = (MU == 0) ? 1 : (MU == 1) ? 0 : (MU == 2) ? 1 : 2;  // S = -1 table
    static constexpr int c1m = (MU == 0) ? 1 : (MU == 1) ? 2 : (MU == 2) ? 3 : 2;
    static constexpr int c0 = (S < 0) ? c0m : (c0m + 2) % 4;
    static constexpr int c1 = (S < 0) ? c1m : (c1m + 2) % 4;
    static constexpr int c0conj = (4 - c0) % 4;
    static constexpr int c1conj = (4 - c1) % 4;
};

// h[k][a], k = 0,1: index 2*(3k+a)
template <int MU, int S, typename T>
__device__ __forceinline__ void project(const T (&psi)[24], T (&h)[12]) {
    typedef Proj<MU, S> P;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        add_c<P::c0>(h[2 * a], h[2 * a + 1], psi[2 * a], psi[2 * a + 1], psi[2 * (3 * P::j0 + a)],
                     psi[2 * (3 * P::j0 + a) + 1]);
        add_c<P::c1>(h[2 * (3 + a)], h[2 * (3 + a) + 1], psi[2 * (3 + a)], psi[2 * (3 + a) + 1],
                     psi[2 * (3 * P::j1 + a)], psi[2 * (3 * P::j1 + a) + 1]);
    }
}

template <int MU, int S, typename T>
__device__ __forceinline__ void accumulate(T (&acc)[24], const T (&chi)[12]) {
    typedef Proj<MU, S> P;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        acc[2 * a] += chi[2 * a];
        acc[2 * a + 1] += chi[2 * a + 1];
        acc[2 * (3 + a)] += chi[2 * (3 + a)];
        acc[2 * (3 + a) + 1] += chi[2 * (3 + a) + 1];
        add_c<P::c0conj>(acc[2 * (3 * P::j0 + a)], acc[2 * (3 * P::j0 + a) + 1],
                         acc[2 * (3 * P::j0 + a)], acc[2 * (3 * P::j0 + a) + 1], chi[2 * a],
                         chi[2 * a + 1]);
        add_c<P::c1conj>(acc[2 * (3 * P::j1 + a)], acc[2 * (3 * P::j1 + a) + 1],
                         acc[2 * (3 * P::j1 + a)], acc[2 * (3 * P::j1 + a) + 1], chi[2 * (3 + a)],
                         chi[2 * (3 + a) + 1]);
    }
}

// acc += sg * (the four spin rows of chi), sg real: the same additions as accumulate() written as multiply-adds, so
// that a boundary phase of +-1 (periodic / antiperiodic directions) needs no branch and no extra instruction;
// fma(1, b, a) = a + b and fma(-1, b, a) = a - b exactly, i.e. the same bits as the branch would give.
template <int C, typename T>
__device__ __forceinline__ void add_c_scaled(T& ore, T& oim, T are, T aim, T bre, T bim, T sg, T msg) {
    if (C == 0) { ore = fma_(sg, bre, are);  oim = fma_(sg, bim, aim); }
    if (C == 1) { ore = fma_(msg, bim, are); oim = fma_(sg, bre, aim); }
    if (C == 2) { ore = fma_(msg, bre, are); oim = fma_(msg, bim, aim); }
    if (C == 3) { ore = fma_(sg, bim, are);  oim = fma_(msg, bre, aim); }
}
template <int MU, int S, typename T>
__device__ __forceinline__ void accumulate_scaled(T (&acc)[24], const T (&chi)[12], T sg) {
    typedef Proj<MU, S> P;
    const T msg = -sg;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        acc[2 * a] = fma_(sg, chi[2 * a], acc[2 * a]);
        acc[2 * a + 1] = fma_(sg, chi[2 * a + 1], acc[2 * a + 1]);
        acc[2 * (3 + a)] = fma_(sg, chi[2 * (3 + a)], acc[2 * (3 + a)]);
        acc[2 * (3 + a) + 1] = fma_(sg, chi[2 * (3 + a) + 1], acc[2 * (3 + a) + 1]);
        add_c_scaled<P::c0conj>(acc[2 * (3 * P::j0 + a)], acc[2 * (3 * P::j0 + a) + 1],
                                acc[2 * (3 * P::j0 + a)], acc[2 * (3 * P::j0 + a) + 1], chi[2 * a], chi[2 * a + 1], sg, msg);
        add_c_scaled<P::c1conj>(acc[2 * (3 * P::j1 + a)], acc[2 * (3 * P::j1 + a) + 1],
                                acc[2 * (3 * P::j1 + a)], acc[2 * (3 * P::j1 + a) + 1], chi[2 * (3 + a)],
                                chi[2 * (3 + a) + 1], sg, msg);
    }
}

// chi_{k,a} = sum_b U_ab h_{k,b}
template <typename T>
__device__ __forceinline__ void su3_mul(const T (&u)[18], const T (&h)[12], T (&chi)[12]) {
#pragma unroll
    for (int k = 0; k < 2; ++k)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            // explicit FMA chains: 4 FMA per complex multiply-add (the a*b - c*d form
            // compiles to MUL + FMA + ADD, 50% more FP64 issue slots and energy)
            T re = u[2 * (3 * a)] * h[2 * (3 * k)];
            T im = u[2 * (3 * a)] * h[2 * (3 * k) + 1];
            re = fma_(-u[2 * (3 * a) + 1], h[2 * (3 * k) + 1], re);
            im = fma_(u[2 * (3 * a) + 1], h[2 * (3 * k)], im);
#pragma unroll
            for (int b = 1; b < 3; ++b) {
                const T ur = u[2 * (3 * a + b)], ui = u[2 * (3 * a + b) + 1];
                const T hr = h[2 * (3 * k + b)], hi = h[2 * (3 * k + b) + 1];
                re = fma_(ur, hr, re);
                re = fma_(-ui, hi, re);
                im = fma_(ur, hi, im);
                im = fma_(ui, hr, im);
            }
            chi[2 * (3 * k + a)] = re;
            chi[2 * (3 * k + a) + 1] = im;
        }
}

// chi_{k,a} = sum_b conj(U_ba) h_{k,b}
template <typename T>
__device__ __forceinline__ void su3_dag_mul(const T (&u)[18], const T (&h)[12], T (&chi)[12]) {
#pragma unroll
    for (int k = 0; k < 2; ++k)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            T re = u[2 * a] * h[2 * (3 * k)];
            T im = u[2 * a] * h[2 * (3 * k) + 1];
            re = fma_(u[2 * a + 1], h[2 * (3 * k) + 1], re);
            im = fma_(-u[2 * a + 1], h[2 * (3 * k)], im);
#pragma unroll
            for (int b = 1; b < 3; ++b) {
                const T ur = u[2 * (3 * b + a)], ui = u[2 * (3 * b + a) + 1];
                const T hr = h[2 * (3 * k + b)], hi = h[2 * (3 * k + b) + 1];
                re = fma_(ur, hr, re);
                re = fma_(ui, hi, re);
                im = fma_(ur, hi, im);
                im = fma_(-ui, hr, im);
            }
            chi[2 * (3 * k + a)] = re;
            chi[2 * (3 * k + a) + 1] = im;
        }
}

}  // namespace
}  // namespace lqcd
