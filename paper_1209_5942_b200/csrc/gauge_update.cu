// gauge_update.cu -- the paper's second workload: pure-gauge heatbath and overrelaxation
// (Fig. 2; Table 2 rows "heatbath" / "overrelax", PAPER.md:237-238;
// SURVEY.md section 8(f) row 4; readings G17-G21), plus the average plaquette.
//
// One launch = one sub-sweep: every link U_mu(x) with parity(x) = p, one thread per link.  Those
// links are independent: the 6 staples of U_mu(x) hold links of the other directions, and
// direction-mu links only at x +- nu, which have the other parity.  Per link (Fig. 2):
//   A = sum_{nu != mu} [ U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag + U_nu(x+mu-nu)^dag U_mu(x-nu)^dag U_nu(x-nu) ]
//   for the subgroups (0,1), (1,2), (0,2):  W = L A;  w = project(W);  v = update(w);  L = extend(v) L
// with update = Kennedy-Pendleton heatbath (v w = g, g ~ sqrt(1 - g0^2) exp(lambda g0), lambda =
// 2 beta k / 3) or overrelaxation (v w = w^dag).  The 3x3 products run in the storage precision
// T; the SU(2) step (projection, k, the random draws, the accept/reject decision, v) always runs
// in double, so that single-precision fields take the same decisions as a double evaluation of
// the same W.  Random numbers: the counter-based generator of the input
// recipe (reading G21), re-implemented here.
//
// Traffic: the paper's kernel moved 2880 B per link (19 links read, 1 written, no reuse).  A
// sub-sweep needs every link of the lattice once (4 V links) and writes V/2: algorithmic
// 9 x 144 = 1296 B per updated link in double/18; the 2.1-fold reuse of the 18 loads is left to
// L1/L2, as for the neighbour spinors of the hopping kernel.
#include "site_ops.cuh"
#include "../../include/lqcd.h"
#include <cstdlib>

// Measured at 32^3 x 64 (us per sub-sweep, heatbath / overrelaxation): double with 2 CTAs per SM
// (246 registers) 460 / 289, with 3 (168 registers, 8 B of spills) 415 / 291, with the staple loop
// unrolled as well 403 / 267; single with 3, 4, 5, 6 CTAs 331 / 172, 310 / 164, 306 / 178, 307 / 169,
// unrolled at 4 CTAs 310 / 149.  Re-measured: double at 4 CTAs (128 registers, 60-80 B of spills) 406 / 279.
// Kennedy-Pendleton draws of the first two attempts precomputed ahead of the staple loads
// (kp_precompute): heatbath 401 -> 395 (double), 310 -> 279 (single/18), 331 -> 308 (single/12).
// Round 2: CTAs on a 2 x 2 block in (z, t) of one group instead of four consecutive groups (the staple links shared
// between sites one step apart in z, t then meet in one CTA's L1): overrelaxation 264.4 / 153.0 / 245.7 / 152.3 us
// (double/18, single/18, double/12, single/12) against 266.4 / 151.0 / 242.5 / 150.2 in linear order, heatbath 401.7
// against 397.8 -- no gain, not kept (the same order of sites moved nothing in the hopping kernel either).
// CTAs per SM re-measured on the final kernels (overrelaxation sub-sweep, us, A B A B on one box): single/18 at 3 / 4 / 5 / 6
// CTAs 139.8 / 131.6-132.9 / 144.0 / 143.1, single/12 131.7 / 119.9 / 121.0 / 123.3; double/18 at 2 / 3 CTAs 262.9 /
// 242.8-245.0, double/12 232.6 / 210-219 (4 CTAs: 259.7, profiles/r02_heatbath.md).  The constants below stay.
constexpr int kGaugeMinBlocksDouble = 3;   // CTAs of 128 threads per SM the register allocation aims at
constexpr int kGaugeMinBlocksFloat = 4;

namespace lqcd {
namespace {

struct GaugeArgs {
    void* gauge;
    Geometry g;
    int mu, parity;
    double beta;
    double c_il;            // 3 / (2 beta): 1 / lambda = c_il / k (heatbath)
    unsigned long long seed, tag;
    Reduction red;          // plaquette only
};

// ------------------------------------------------------------------------------- indexing
struct SiteIdx {
    int e, x0h, x1, x2, x3, r;   // r = x0 mod 2
};

__device__ __forceinline__ SiteIdx site_of(const Geometry& g, int e, int parity) {
    SiteIdx s;
    s.e = e;
    site_coords(g, e, s.x0h, s.x1, s.x2, s.x3);
    s.r = (s.x1 + s.x2 + s.x3 + parity) & 1;
    return s;
}

// neighbour in direction dir, sgn = +1 / -1 (periodic; the neighbour has the other parity).  Written with selects only:
// a branch per step would cut the kernel into basic blocks and keep ptxas from carrying link loads across them.
__device__ __forceinline__ SiteIdx step(const Geometry& g, SiteIdx s, int dir, int sgn) {
    // direction 0: the even-odd index moves only when the parity bit r allows it (x0 = 2 x0h + r)
    const bool up = sgn > 0;
    const bool move0 = up ? (s.r != 0) : (s.r == 0);
    const int n = (dir == 0) ? g.N0h : (dir == 1) ? g.N1 : (dir == 2) ? g.N2 : g.N3;
    const int stride = (dir == 0) ? 1 : (dir == 1) ? g.N0h : (dir == 2) ? g.N0h * g.N1 : g.N0h * g.N1 * g.N2;
    const int c = (dir == 0) ? s.x0h : (dir == 1) ? s.x1 : (dir == 2) ? s.x2 : s.x3;
    const bool moves = (dir != 0) || move0;
    const bool wrap = up ? (c == n - 1) : (c == 0);
    const int dc = !moves ? 0 : up ? (wrap ? -(n - 1) : 1) : (wrap ? (n - 1) : -1);
    s.e += dc * stride;
    s.x0h += (dir == 0) ? dc : 0;
    s.x1 += (dir == 1) ? dc : 0;
    s.x2 += (dir == 2) ? dc : 0;
    s.x3 += (dir == 3) ? dc : 0;
    s.r ^= (dir == 0) ? 1 : 0;
    return s;
}

// ------------------------------------------------------------------------------- link access
// Links are reused by several threads here (unlike in the hopping kernel), so they are read
// with default caching, not evict-first.  COHERENT = the link this thread rewrites.
template <int RECON, bool COHERENT>
__device__ __forceinline__ void gload(const void* gauge, int G, int par, int mu, int idx, double (&u)[18]) {
    const double2* p = reinterpret_cast<const double2*>(gauge) +
                       gauge_block(par, mu, G, idx >> 5) * ((RECON / 2) * 32) + (idx & 31);
#pragma unroll
    for (int j = 0; j < RECON / 2; ++j) {
        const double2 v = COHERENT ? p[j * 32] : __ldg(p + j * 32);
        u[2 * j] = v.x;
        u[2 * j + 1] = v.y;
    }
    if (RECON == 12) reconstruct_row2(u);
}
template <int RECON, bool COHERENT>
__device__ __forceinline__ void gload(const void* gauge, int G, int par, int mu, int idx, float (&u)[18]) {
    if (RECON == 12) {
        const float4* p = reinterpret_cast<const float4*>(gauge) +
                          gauge_block(par, mu, G, idx >> 5) * (3 * 32) + (idx & 31);
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            const float4 v = COHERENT ? p[j * 32] : __ldg(p + j * 32);
            u[4 * j] = v.x; u[4 * j + 1] = v.y; u[4 * j + 2] = v.z; u[4 * j + 3] = v.w;
        }
        reconstruct_row2(u);
    } else {
        const float* blk = reinterpret_cast<const float*>(gauge) + gauge_block(par, mu, G, idx >> 5) * (18 * 32);
        const float4* p = reinterpret_cast<const float4*>(blk) + (idx & 31);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const float4 v = COHERENT ? p[j * 32] : __ldg(p + j * 32);
            u[4 * j] = v.x; u[4 * j + 1] = v.y; u[4 * j + 2] = v.z; u[4 * j + 3] = v.w;
        }
        const float2* q = reinterpret_cast<const float2*>(blk + 16 * 32) + (idx & 31);
        const float2 w = COHERENT ? *q : __ldg(q);
        u[16] = w.x;
        u[17] = w.y;
    }
}
// 12-real storage keeps rows 0, 1 and rebuilds row 2 = conj(row0 x row1) on every load.  A rounding
// defect eps of the stored rows comes back as 2 eps in the rebuilt row and is mixed into rows 0, 1
// by the (1,2) and (0,2) subgroup steps: measured growth x1.35 per overrelaxation sweep in single
// precision (unitarity defect 1e-5 -> 0.1 in 30 sweeps) where 18-real storage only random-walks
// (2e-6).  So the two rows are re-orthonormalised (Gram-Schmidt) before they are stored.
template <typename T>
__device__ __forceinline__ void orthonormalise_rows01(T (&u)[18]) {
    T n0 = 0;
#pragma unroll
    for (int i = 0; i < 6; ++i) n0 = fma_(u[i], u[i], n0);
    const T i0 = rsqrt(n0);
#pragma unroll
    for (int i = 0; i < 6; ++i) u[i] *= i0;
    T dr = 0, di = 0;   // <row0, row1> = sum conj(row0_c) row1_c
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        dr = fma_(u[2 * c], u[6 + 2 * c], fma_(u[2 * c + 1], u[6 + 2 * c + 1], dr));
        di = fma_(u[2 * c], u[6 + 2 * c + 1], fma_(-u[2 * c + 1], u[6 + 2 * c], di));
    }
    T n1 = 0;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const T re = u[6 + 2 * c] - (dr * u[2 * c] - di * u[2 * c + 1]);
        const T im = u[6 + 2 * c + 1] - (dr * u[2 * c + 1] + di * u[2 * c]);
        u[6 + 2 * c] = re;
        u[6 + 2 * c + 1] = im;
        n1 = fma_(re, re, fma_(im, im, n1));
    }
    const T i1 = rsqrt(n1);
#pragma unroll
    for (int i = 6; i < 12; ++i) u[i] *= i1;
}

template <int RECON>
__device__ __forceinline__ void gstore(void* gauge, int G, int par, int mu, int idx, const double (&u)[18]) {
    double2* p = reinterpret_cast<double2*>(gauge) + gauge_block(par, mu, G, idx >> 5) * ((RECON / 2) * 32) + (idx & 31);
#pragma unroll
    for (int j = 0; j < RECON / 2; ++j) p[j * 32] = make_double2(u[2 * j], u[2 * j + 1]);
}
template <int RECON>
__device__ __forceinline__ void gstore(void* gauge, int G, int par, int mu, int idx, const float (&u)[18]) {
    if (RECON == 12) {
        float4* p = reinterpret_cast<float4*>(gauge) + gauge_block(par, mu, G, idx >> 5) * (3 * 32) + (idx & 31);
#pragma unroll
        for (int j = 0; j < 3; ++j) p[j * 32] = make_float4(u[4 * j], u[4 * j + 1], u[4 * j + 2], u[4 * j + 3]);
    } else {
        float* blk = reinterpret_cast<float*>(gauge) + gauge_block(par, mu, G, idx >> 5) * (18 * 32);
        float4* p = reinterpret_cast<float4*>(blk) + (idx & 31);
#pragma unroll
        for (int j = 0; j < 4; ++j) p[j * 32] = make_float4(u[4 * j], u[4 * j + 1], u[4 * j + 2], u[4 * j + 3]);
        reinterpret_cast<float2*>(blk + 16 * 32)[idx & 31] = make_float2(u[16], u[17]);
    }
}

// c (+)= op(a) op(b), op = identity or dagger; 3x3 complex, row-major, explicit FMA chains
template <bool DA, bool DB, bool ACC, typename T>
__device__ __forceinline__ void mm3(const T (&a)[18], const T (&b)[18], T (&c)[18]) {
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            T re = ACC ? c[2 * (3 * i + j)] : (T)0, im = ACC ? c[2 * (3 * i + j) + 1] : (T)0;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const T ar = DA ? a[2 * (3 * k + i)] : a[2 * (3 * i + k)];
                const T ai = DA ? -a[2 * (3 * k + i) + 1] : a[2 * (3 * i + k) + 1];
                const T br = DB ? b[2 * (3 * j + k)] : b[2 * (3 * k + j)];
                const T bi = DB ? -b[2 * (3 * j + k) + 1] : b[2 * (3 * k + j) + 1];
                re = fma_(ar, br, re);
                re = fma_(-ai, bi, re);
                im = fma_(ar, bi, im);
                im = fma_(ai, br, im);
            }
            c[2 * (3 * i + j)] = re;
            c[2 * (3 * i + j) + 1] = im;
        }
}

// ------------------------------------------------------------------------------- random numbers
// uniform in (0,1]: bits = splitmix64_mix(seed * GOLD + (stream << 40) + counter), top 53 bits
__device__ __forceinline__ double uniform01(unsigned long long seed, unsigned long long stream,
                                            unsigned long long counter) {
    unsigned long long z = seed * 0x9E3779B97F4A7C15ULL + (stream << 40) + counter;
    z += 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return ((double)(z >> 11) + 1.0) * (1.0 / 9007199254740992.0);
}

constexpr int MAXTRY = 32;   // reading G20

// Kennedy-Pendleton: g0 with density sqrt(1 - g0^2) exp(lambda g0), direction uniform.
// Counters: attempt t uses base + 4 t + (0..3), the direction base + 4 MAXTRY + (0, 1).
//
// Everything but the division by lambda depends on the random numbers alone, i.e. on the link id,
// not on the fields: X_t = -(ln r1 + cos^2(2 pi r2) ln r3), q_t = r4^2, and the direction.  So the
// first KP_PRE attempts and the direction of all three subgroups are worked out at the start of the
// kernel -- straight-line code with three-fold instruction-level parallelism that overlaps the
// staple loads -- and parked in shared memory; the serial, divergent accept loop that used to
// follow the staple sum only remains for the lanes that reject KP_PRE times (0.5% at beta = 5.7).
// A divergent attempt costs a warp as much as a full one, so computing attempt 1 for every lane
// costs nothing extra.  Values and decisions are bit-identical to the one-loop form.
constexpr int KP_PRE = 2;
constexpr int KP_SLOTS = 2 * KP_PRE + 4;   // X_t, q_t for t < KP_PRE; sin(theta), cos(theta), sin(phi), cos(phi)

// ln x for x in (0, 1], x a multiple of 2^-53 (a uniform01 draw): the exponent, a 128-entry table on the top seven
// mantissa bits (kp_log_table.h: ln m = log_c + log1p(m inv_c - 1), |m inv_c - 1| <= 2^-8) and the series of log1p to
// the seventh power, 12 FP64 instructions against ~35 of the library's log with its special cases; the result is within
// 2.3e-16 max(|ln x|, 1) of the correctly rounded one (checked over 3e5 arguments against glibc when the table was
// made), which is what the draws need: a flip of an accept/reject decision against the oracle takes a difference of the
// size of |r4^2 - (1 - delta / 2)|.
#include "kp_log_table.h"
__device__ __forceinline__ double kp_log(double x) {
    const long long b = __double_as_longlong(x);
    const int e = (int)(b >> 52) - 1023;
    const double m = __longlong_as_double((b & 0x000fffffffffffffLL) | 0x3ff0000000000000LL);
    const double2 t = __ldg(&kp_log_tab[(int)(b >> 45) & 127]);
    const double eps = fma(m, t.x, -1.0);
    double p = fma(eps, 1.0 / 7.0, -1.0 / 6.0);
    p = fma(p, eps, 0.2);
    p = fma(p, eps, -0.25);
    p = fma(p, eps, 1.0 / 3.0);
    p = fma(p, eps, -0.5);
    p = fma(p * eps, eps, eps);
    const double de = (double)e;
    return fma(de, KP_LN2_HI, t.y) + fma(de, KP_LN2_LO, p);
}

__device__ __forceinline__ void kp_attempt(unsigned long long seed, unsigned long long tag, unsigned long long c,
                                           double& X, double& q) {
    const double r1 = uniform01(seed, tag, c), r2 = uniform01(seed, tag, c + 1);
    const double r3 = uniform01(seed, tag, c + 2), r4 = uniform01(seed, tag, c + 3);
    const double cs = cospi(2.0 * r2);
    X = -(kp_log(r1) + cs * cs * kp_log(r3));
    q = r4 * r4;
}

// pre[slot * stride]: the thread's KP_SLOTS values of one subgroup
__device__ __forceinline__ void kp_precompute(unsigned long long seed, unsigned long long tag, unsigned long long base,
                                              double* pre, int stride) {
#pragma unroll
    for (int t = 0; t < KP_PRE; ++t) {
        double X, q;
        kp_attempt(seed, tag, base + 4ull * t, X, q);
        pre[(2 * t) * stride] = X;
        pre[(2 * t + 1) * stride] = q;
    }
    const unsigned long long cd = base + 4ull * MAXTRY;
    const double r5 = uniform01(seed, tag, cd), r6 = uniform01(seed, tag, cd + 1);
    const double ct = 2.0 * r5 - 1.0;
    const double st = sqrt(1.0 - ct * ct);
    double sp, cp;
    sincospi(2.0 * r6, &sp, &cp);
    pre[(2 * KP_PRE) * stride] = st;
    pre[(2 * KP_PRE + 1) * stride] = ct;
    pre[(2 * KP_PRE + 2) * stride] = sp;
    pre[(2 * KP_PRE + 3) * stride] = cp;
}

// il = 1 / lambda = (3 / (2 beta)) (1 / k), handed in as a product of the two reciprocals the caller already has: X * il is
// within two ulp of the X / lambda of the definition, and the subgroup step has no division left.
__device__ __forceinline__ bool kp_sample(double il, unsigned long long seed, unsigned long long tag,
                                          unsigned long long base, const double* pre, int stride, double (&g)[4]) {
    bool ok = false;
    double delta = 0.0;
#pragma unroll
    for (int t = 0; t < KP_PRE; ++t) {
        if (!ok) {
            delta = pre[(2 * t) * stride] * il;
            ok = pre[(2 * t + 1) * stride] <= 1.0 - 0.5 * delta;
        }
    }
    for (int t = KP_PRE; t < MAXTRY && !ok; ++t) {
        double X, q;
        kp_attempt(seed, tag, base + 4ull * t, X, q);
        delta = X * il;
        ok = q <= 1.0 - 0.5 * delta;
    }
    if (!ok) return false;
    const double st = pre[(2 * KP_PRE) * stride], ct = pre[(2 * KP_PRE + 1) * stride];
    const double sp = pre[(2 * KP_PRE + 2) * stride], cp = pre[(2 * KP_PRE + 3) * stride];
    const double g0 = 1.0 - delta;
    const double rad = sqrt(1.0 - g0 * g0);
    g[0] = g0;
    g[1] = rad * st * cp;
    g[2] = rad * st * sp;
    g[3] = rad * ct;
    return true;
}

// One subgroup step of Fig. 2 on the link L with staple sum A: subgroup (P, Q), I = its index.
// SU(2) elements are quaternions (a0, a1, a2, a3) = a0 + i a.sigma
//   = [[a0 + i a3, a2 + i a1], [-a2 + i a1, a0 - i a3]]   (reading G19);
// (a0, a)(b0, b) = (a0 b0 - a.b, a0 b + b0 a - a x b).
template <int MODE, int I, int P, int Q, typename T>
__device__ __forceinline__ void subgroup_step(T (&L)[18], const T (&A)[18], double c_il, unsigned long long seed,
                                              unsigned long long tag, unsigned long long link_id, const double* pre,
                                              int stride) {
    // the four entries (P,P), (P,Q), (Q,P), (Q,Q) of W = L A
    T wr[4], wi[4];
#pragma unroll
    for (int n = 0; n < 4; ++n) {
        const int i = (n < 2) ? P : Q, j = (n & 1) ? Q : P;
        T re = 0, im = 0;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const T ar = L[2 * (3 * i + k)], ai = L[2 * (3 * i + k) + 1];
            const T br = A[2 * (3 * k + j)], bi = A[2 * (3 * k + j) + 1];
            re = fma_(ar, br, re);
            re = fma_(-ai, bi, re);
            im = fma_(ar, bi, im);
            im = fma_(ai, br, im);
        }
        wr[n] = re;
        wi[n] = im;
    }
    double w0 = 0.5 * ((double)wr[0] + (double)wr[3]);
    double w1 = 0.5 * ((double)wi[1] + (double)wi[2]);
    double w2 = 0.5 * ((double)wr[1] - (double)wr[2]);
    double w3 = 0.5 * ((double)wi[0] - (double)wi[3]);
    const double k2 = w0 * w0 + w1 * w1 + w2 * w2 + w3 * w3;
    if (!(k2 > 0.0)) return;
    const double ik = rsqrt(k2);       // 1 / k from one reciprocal square root (no sqrt, no division)
    w0 *= ik; w1 *= ik; w2 *= ik; w3 *= ik;
    double v0, v1, v2, v3;
    if (MODE == 0) {   // heatbath: v = g w^dag
        double g[4];
        const unsigned long long base = ((link_id * 3ull + (unsigned long long)I) * (unsigned long long)(MAXTRY + 1)) * 4ull;
        if (!kp_sample(c_il * ik, seed, tag, base, pre + (size_t)I * KP_SLOTS * stride, stride, g)) return;
        v0 = g[0] * w0 + (g[1] * w1 + g[2] * w2 + g[3] * w3);
        v1 = w0 * g[1] - g[0] * w1 + (g[2] * w3 - g[3] * w2);
        v2 = w0 * g[2] - g[0] * w2 + (g[3] * w1 - g[1] * w3);
        v3 = w0 * g[3] - g[0] * w3 + (g[1] * w2 - g[2] * w1);
    } else {           // overrelaxation: v = (w^dag)^2
        v0 = w0 * w0 - (w1 * w1 + w2 * w2 + w3 * w3);
        v1 = -2.0 * w0 * w1;
        v2 = -2.0 * w0 * w2;
        v3 = -2.0 * w0 * w3;
    }
    // L <- extend(v) L: rows P, Q become v00 L_P + v01 L_Q and v10 L_P + v11 L_Q
    const T ar = (T)v0, ai = (T)v3, br = (T)v2, bi = (T)v1;   // v00 = a, v01 = b, v10 = -conj(b), v11 = conj(a)
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const T pr = L[2 * (3 * P + c)], pi = L[2 * (3 * P + c) + 1];
        const T qr = L[2 * (3 * Q + c)], qi = L[2 * (3 * Q + c) + 1];
        L[2 * (3 * P + c)]     = fma_(-bi, qi, fma_(br, qr, fma_(-ai, pi, ar * pr)));
        L[2 * (3 * P + c) + 1] = fma_(bi, qr, fma_(br, qi, fma_(ai, pr, ar * pi)));
        L[2 * (3 * Q + c)]     = fma_(ai, qi, fma_(ar, qr, fma_(-bi, pi, -br * pr)));
        L[2 * (3 * Q + c) + 1] = fma_(-ai, qr, fma_(ar, qi, fma_(bi, pr, -br * pi)));
    }
}

// Rows 0, 1 of op(a) op(b) (a product of SU(3) matrices is in SU(3): its third row follows from these two).
template <bool DA, bool DB, typename T>
__device__ __forceinline__ void mm3_rows01(const T (&a)[18], const T (&b)[18], T (&c)[12]) {
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            T re = 0, im = 0;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const T ar = DA ? a[2 * (3 * k + i)] : a[2 * (3 * i + k)];
                const T ai = DA ? -a[2 * (3 * k + i) + 1] : a[2 * (3 * i + k) + 1];
                const T br = DB ? b[2 * (3 * j + k)] : b[2 * (3 * k + j)];
                const T bi = DB ? -b[2 * (3 * j + k) + 1] : b[2 * (3 * k + j) + 1];
                re = fma_(ar, br, re);
                re = fma_(-ai, bi, re);
                im = fma_(ar, bi, im);
                im = fma_(ai, br, im);
            }
            c[2 * (3 * i + j)] = re;
            c[2 * (3 * i + j) + 1] = im;
        }
}
// A += S, S the SU(3) matrix whose rows 0, 1 are t01 op(b): rows 0, 1 as computed, row 2 = conj(row0 x row1) accumulated
// straight into A (8 multiply-adds per entry, the same count as the direct product of a third row would need for ONE of
// the two products it saves).
template <bool DB, typename T>
__device__ __forceinline__ void add_staple_rows01(const T (&t)[12], const T (&b)[18], T (&A)[18]) {
    T s[12];
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            T re = 0, im = 0;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const T ar = t[2 * (3 * i + k)], ai = t[2 * (3 * i + k) + 1];
                const T br = DB ? b[2 * (3 * j + k)] : b[2 * (3 * k + j)];
                const T bi = DB ? -b[2 * (3 * j + k) + 1] : b[2 * (3 * k + j) + 1];
                re = fma_(ar, br, re);
                re = fma_(-ai, bi, re);
                im = fma_(ar, bi, im);
                im = fma_(ai, br, im);
            }
            s[2 * (3 * i + j)] = re;
            s[2 * (3 * i + j) + 1] = im;
        }
#pragma unroll
    for (int i = 0; i < 12; ++i) A[i] += s[i];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
        const T ar = s[2 * c1], ai = s[2 * c1 + 1], br = s[6 + 2 * c2], bi = s[6 + 2 * c2 + 1];
        const T cr = s[2 * c2], ci = s[2 * c2 + 1], dr = s[6 + 2 * c1], di = s[6 + 2 * c1 + 1];
        // A2_c += conj(s0[c1] s1[c2] - s0[c2] s1[c1])
        A[12 + 2 * c] = fma_(ci, di, fma_(-cr, dr, fma_(-ai, bi, fma_(ar, br, A[12 + 2 * c]))));
        A[12 + 2 * c + 1] = fma_(ci, dr, fma_(cr, di, fma_(-ai, br, fma_(-ar, bi, A[12 + 2 * c + 1]))));
    }
}

// the two products of a staple, full (t of 18 reals) or two-row (t of 12)
template <bool DA, bool DB, typename T>
__device__ __forceinline__ void staple_first(const T (&a)[18], const T (&b)[18], T (&t)[18]) { mm3<DA, DB, false>(a, b, t); }
template <bool DA, bool DB, typename T>
__device__ __forceinline__ void staple_first(const T (&a)[18], const T (&b)[18], T (&t)[12]) { mm3_rows01<DA, DB>(a, b, t); }
template <bool DB, typename T>
__device__ __forceinline__ void staple_second(const T (&t)[18], const T (&b)[18], T (&A)[18]) { mm3<false, DB, true>(t, b, A); }
template <bool DB, typename T>
__device__ __forceinline__ void staple_second(const T (&t)[12], const T (&b)[18], T (&A)[18]) { add_staple_rows01<DB>(t, b, A); }

// A += the six staples of U_mu(x) (Fig. 2).  All neighbour indices first, then one straight line of 18 link loads and
// 12 products, written software-pipelined: the first link of the next direction nu is asked for BEFORE the last product
// of the current one, so that the three passes do not each begin with nothing in flight (ptxas keeps to the order it
// is given across these blocks: with the loads of a pass issued only after the pass before had finished, a thread sat
// through four exposed round trips instead of one).
// The link itself, L = U_mu(x), is asked for before the very last product for the same reason.
template <typename T, int RECON>
__device__ __forceinline__ void staple_sum(const GaugeArgs& a, const SiteIdx& x, const SiteIdx& xpm, T (&A)[18], T (&L)[18]) {
    const int G = a.g.G, mu = a.mu, p = a.parity;
    int nu[3], e_pn[3], e_mn[3], e_pmmn[3];
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        nu[j] = (mu + j + 1) & 3;   // the three directions nu != mu
        e_pn[j] = step(a.g, x, nu[j], +1).e;
        e_mn[j] = step(a.g, x, nu[j], -1).e;
        e_pmmn[j] = step(a.g, xpm, nu[j], -1).e;
    }
    // Two-row form of the products (mm3_rows01 / add_staple_rows01: a staple is a product of SU(3) matrices, so its
    // third row is conj(row0 x row1) and a third of the first product need not be computed): 36 of 216 multiply-adds per
    // staple less.  Measured at 32^3 x 64 (us per sub-sweep, heatbath / overrelaxation, A B A B on one box, full / two-row):
    // double/12 321-323 / 212 -> 283-284 / 205-213, single/12 216 / 120 -> 199 / 106, single/18 202 / 134-135 -> 198 / 130-133;
    // double/18 326-329 / 246-253 -> 342-345 / 274-275: the full products stay there.  (Not the spills and not the shape of
    // the source: the same products formed one row at a time with all three operands in registers give 343-344 / 273, and
    // with the loads the two-row form drops kept alive 373-375 / 307-308.  ncu, profiles/r02_heatbath.md: 16% fewer
    // instructions, 12% fewer bytes from L2, and more exposed load latency.)
    constexpr bool TWOROW = !(sizeof(T) == 8 && RECON == 18);
    T u[18], w[18], t[TWOROW ? 12 : 18], nx[18];
    gload<RECON, false>(a.gauge, G, 1 - p, nu[0], xpm.e, nx);            // U_nu(x+mu) of the first direction
#pragma unroll
    for (int j = 0; j < 3; ++j) {
#pragma unroll
        for (int i = 0; i < 18; ++i) u[i] = nx[i];
        gload<RECON, false>(a.gauge, G, 1 - p, mu, e_pn[j], w);          // U_mu(x+nu)
        staple_first<false, true>(u, w, t);
        gload<RECON, false>(a.gauge, G, p, nu[j], x.e, u);               // U_nu(x)
        staple_second<true>(t, u, A);
        gload<RECON, false>(a.gauge, G, p, nu[j], e_pmmn[j], u);         // U_nu(x+mu-nu)
        gload<RECON, false>(a.gauge, G, 1 - p, mu, e_mn[j], w);          // U_mu(x-nu)
        staple_first<true, true>(u, w, t);
        gload<RECON, false>(a.gauge, G, 1 - p, nu[j], e_mn[j], u);       // U_nu(x-nu)
        if (j < 2) gload<RECON, false>(a.gauge, G, 1 - p, nu[j + 1], xpm.e, nx);   // next pass: U_nu'(x+mu)
        else       gload<RECON, true>(a.gauge, G, p, mu, x.e, L);                  // after the last pass: the link itself
        staple_second<false>(t, u, A);
    }
}

template <typename T, int RECON, int MODE>
__global__ void __launch_bounds__(128, sizeof(T) == 8 ? kGaugeMinBlocksDouble : kGaugeMinBlocksFloat)
gauge_update_kernel(const GaugeArgs a) {
    const int e = blockIdx.x * 128 + (threadIdx.x & 127);
    if (e >= a.g.Vh) return;
    const int G = a.g.G, mu = a.mu, p = a.parity;
    const SiteIdx x = site_of(a.g, e, p);
    const SiteIdx xpm = step(a.g, x, mu, +1);
    // link id of reading G21: 4 lex(x) + mu, lex(x) = 2 e + r
    const unsigned long long link_id = 4ull * (2ull * (unsigned long long)e + (unsigned long long)x.r) + (unsigned long long)mu;
    // heatbath: the random-number part of the three Kennedy-Pendleton steps (see kp_precompute)
    __shared__ double pre_s[MODE == 0 ? 3 * KP_SLOTS * 128 : 1];
    double* pre = pre_s + threadIdx.x;
    if (MODE == 0) {
#pragma unroll
        for (int i = 0; i < 3; ++i)
            kp_precompute(a.seed, a.tag, ((link_id * 3ull + (unsigned long long)i) * (unsigned long long)(MAXTRY + 1)) * 4ull,
                          pre + (size_t)i * KP_SLOTS * 128, 128);
    }
    T A[18];
#pragma unroll
    for (int i = 0; i < 18; ++i) A[i] = 0;
    T L[18];
    staple_sum<T, RECON>(a, x, xpm, A, L);
    subgroup_step<MODE, 0, 0, 1>(L, A, a.c_il, a.seed, a.tag, link_id, pre, 128);
    subgroup_step<MODE, 1, 1, 2>(L, A, a.c_il, a.seed, a.tag, link_id, pre, 128);
    subgroup_step<MODE, 2, 0, 2>(L, A, a.c_il, a.seed, a.tag, link_id, pre, 128);
    if (RECON == 12) orthonormalise_rows01(L);
    gstore<RECON>(a.gauge, G, p, mu, e, L);
}


// Heatbath, warp-specialised (LQCD_HEATBATH_WS=1; not the default, see the end of this comment): a CTA of 256 threads is two warpgroups working on the same 128
// links.  Warpgroup 1 does nothing but the field-independent part of the three Kennedy-Pendleton steps (kp_precompute:
// 30 uniforms, 12 logarithms, 6 cospi, 3 sincospi and 3 square roots per link, ~2000 instructions, FP64/integer pipes)
// and parks the 24 doubles per link in shared memory; warpgroup 0 is the update kernel proper (staple loads and
// products, latency bound) and meets it at a named barrier before the subgroup steps.  The two instruction streams
// overlap instead of following each other inside one thread, and setmaxnreg moves the registers to where they are
// needed: the CTA is launched at 80 registers per thread (three CTAs per SM), warpgroup 1 drops to 40, warpgroup 0
// takes 120.  Same counters, same values, same decisions as the one-thread form (gauge_update_kernel<.., 0>).
// Measured at 32^3 x 64 (us per sub-sweep, this kernel / one thread per link): double/18 431 / 398, single/18 307 / 279,
// double/12 435 / 411, single/12 330 / 307.  The Kennedy-Pendleton arithmetic costs the same ~130 us wherever it runs:
// it is bound by the FP64 pipe (about 1500 FP64 instructions per link on top of the 2250 of the staple products),
// not by latency another warp could hide.
template <typename T, int RECON>
__global__ void __launch_bounds__(256, 3) heatbath_ws_kernel(const GaugeArgs a) {
    __shared__ double pre_s[3 * KP_SLOTS * 128];
    const int wg = threadIdx.x >> 7, tl = threadIdx.x & 127;
    const int e = blockIdx.x * 128 + (threadIdx.x & 127);
    const int G = a.g.G, mu = a.mu, p = a.parity;
    const bool live = e < a.g.Vh;
    if (wg == 1) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;\n" ::);
        if (live) {
            int x0h, x1, x2, x3;
            site_coords(a.g, e, x0h, x1, x2, x3);
            const int r = (x1 + x2 + x3 + p) & 1;
            const unsigned long long link_id = 4ull * (2ull * (unsigned long long)e + (unsigned long long)r) + (unsigned long long)mu;
#pragma unroll 1
            for (int i = 0; i < 3; ++i)
                kp_precompute(a.seed, a.tag, ((link_id * 3ull + (unsigned long long)i) * (unsigned long long)(MAXTRY + 1)) * 4ull,
                              pre_s + tl + (size_t)i * KP_SLOTS * 128, 128);
        }
        __threadfence_block();
        asm volatile("bar.arrive 1, 256;\n" ::);
        return;
    }
    asm volatile("setmaxnreg.inc.sync.aligned.u32 120;\n" ::);
    T L[18], A[18];
    unsigned long long link_id = 0;
    if (live) {
        const SiteIdx x = site_of(a.g, e, p);
        const SiteIdx xpm = step(a.g, x, mu, +1);
        link_id = 4ull * (2ull * (unsigned long long)e + (unsigned long long)x.r) + (unsigned long long)mu;
#pragma unroll
        for (int i = 0; i < 18; ++i) A[i] = 0;
        staple_sum<T, RECON>(a, x, xpm, A, L);
    }
    asm volatile("bar.sync 1, 256;\n" ::: "memory");
    if (live) {
        const double* pre = pre_s + tl;
        subgroup_step<0, 0, 0, 1>(L, A, a.c_il, a.seed, a.tag, link_id, pre, 128);
        subgroup_step<0, 1, 1, 2>(L, A, a.c_il, a.seed, a.tag, link_id, pre, 128);
        subgroup_step<0, 2, 0, 2>(L, A, a.c_il, a.seed, a.tag, link_id, pre, 128);
        if (RECON == 12) orthonormalise_rows01(L);
        gstore<RECON>(a.gauge, G, p, mu, e, L);
    }
}

// Average plaquette: one thread per site of parity blockIdx.y, 6 plaquettes
//   P_mu_nu(x) = U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag,  mu < nu;
// one partial sum of Re tr per warp (fixed-order two-stage sum, lqcd_internal.h).
template <typename T, int RECON>
__global__ void __launch_bounds__(128, 3) plaquette_kernel(const GaugeArgs a) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    const int p = blockIdx.y;
    const int G = a.g.G;
    double sum = 0.0;
    if (e < a.g.Vh) {
        const SiteIdx x = site_of(a.g, e, p);
#pragma unroll 1
        for (int mu = 0; mu < 3; ++mu) {
            const SiteIdx xpm = step(a.g, x, mu, +1);
            T um[18];
            gload<RECON, false>(a.gauge, G, p, mu, e, um);
#pragma unroll 1
            for (int nu = mu + 1; nu < 4; ++nu) {
                const SiteIdx xpn = step(a.g, x, nu, +1);
                T u[18], t[18], s[18];
                gload<RECON, false>(a.gauge, G, 1 - p, nu, xpm.e, u);
                mm3<false, false, false>(um, u, t);                    // U_mu(x) U_nu(x+mu)
                gload<RECON, false>(a.gauge, G, 1 - p, mu, xpn.e, u);
                mm3<false, true, false>(t, u, s);                      // ... U_mu(x+nu)^dag
                gload<RECON, false>(a.gauge, G, p, nu, e, u);
                // Re tr(s U_nu(x)^dag) = sum_ij Re(s_ij conj(u_ij))
#pragma unroll
                for (int i = 0; i < 18; ++i) sum += (double)s[i] * (double)u[i];
            }
        }
    }
    sum = warp_sum(sum);
    if ((threadIdx.x & 31) == 0)
        a.red.partials[(size_t)p * (gridDim.x * (blockDim.x >> 5)) + ((blockIdx.x * blockDim.x + threadIdx.x) >> 5)] = sum;
}

}  // namespace

cudaError_t launch_gauge_update(int precision, int recon, int mode, const Geometry& g, void* gauge, int mu,
                                int parity, double beta, unsigned long long seed, unsigned long long tag,
                                cudaStream_t st) {
    GaugeArgs a;
    a.gauge = gauge; a.g = g; a.mu = mu; a.parity = parity; a.beta = beta; a.c_il = (beta != 0.0) ? 1.5 / beta : 0.0; a.seed = seed; a.tag = tag;
    a.red.partials = nullptr;
    const int grid = (g.Vh + 127) / 128;
    count_launch();
    ProfScope prof(7, st);
    // heatbath: LQCD_HEATBATH_WS=1 selects the warp-specialised kernel (measured slower: profiles/r02_heatbath.md)
    static const bool ws = getenv("LQCD_HEATBATH_WS") && atoi(getenv("LQCD_HEATBATH_WS")) != 0;
#define LQCD_GU(TT, RR)                                                                   \
    do {                                                                                  \
        if (mode == 0 && ws) heatbath_ws_kernel<TT, RR><<<grid, 256, 0, st>>>(a);         \
        else if (mode == 0)  gauge_update_kernel<TT, RR, 0><<<grid, 128, 0, st>>>(a);     \
        else                 gauge_update_kernel<TT, RR, 1><<<grid, 128, 0, st>>>(a);     \
    } while (0)
    if (precision == 0) { if (recon == 12) LQCD_GU(double, 12); else LQCD_GU(double, 18); }
    else                { if (recon == 12) LQCD_GU(float, 12);  else LQCD_GU(float, 18); }
#undef LQCD_GU
    return cudaGetLastError();
}

int plaquette_partials(int Vh) { return 2 * ((Vh + 127) / 128) * 4; }

cudaError_t launch_plaquette(int precision, int recon, const Geometry& g, const void* gauge, Reduction red,
                             cudaStream_t st) {
    GaugeArgs a;
    a.gauge = const_cast<void*>(gauge); a.g = g; a.mu = 0; a.parity = 0; a.beta = 0; a.c_il = 0; a.seed = 0; a.tag = 0;
    a.red = red;
    const dim3 grid((g.Vh + 127) / 128, 2);
    count_launch();
    ProfScope prof(8, st);
    if (precision == 0) {
        if (recon == 12) plaquette_kernel<double, 12><<<grid, 128, 0, st>>>(a);
        else             plaquette_kernel<double, 18><<<grid, 128, 0, st>>>(a);
    } else {
        if (recon == 12) plaquette_kernel<float, 12><<<grid, 128, 0, st>>>(a);
        else             plaquette_kernel<float, 18><<<grid, 128, 0, st>>>(a);
    }
    return cudaGetLastError();
}


// ---------------------------------------------------------------------------------------------------------------------
// The average plaquette with no allocation anywhere on the path (lqcd_plaquette_static, include/lqcd.h): the per-warp
// partial sums go to a file-scope device array instead of the context's cudaMalloc'ed buffer.  Every GPU that loads the
// library holds the array (LQCD_PLAQUETTE_STATIC_MAX_PARTIALS doubles = 512 KiB) until exit.  All calls share it: calls
// that overlap on the GPU (two streams, two host threads) race on it.  Nothing in it has to start at zero -- a call
// rewrites every partial it later reads -- so it keeps the last call's contents and is never cleared.
// ---------------------------------------------------------------------------------------------------------------------
}  // namespace lqcd

static __device__ __align__(256) double g_plaquette_static_partials[LQCD_PLAQUETTE_STATIC_MAX_PARTIALS];

namespace lqcd {
namespace {

// fixed-order sum of the n partials; device code names the array directly
__global__ void __launch_bounds__(256) plaquette_static_sum_kernel(int n, double inv_norm, double* out) {
    __shared__ double sh[256];
    double s = 0.0;
    for (int i = threadIdx.x; i < n; i += 256) s += g_plaquette_static_partials[i];
    sh[threadIdx.x] = s;
    __syncthreads();
#pragma unroll
    for (int w = 128; w > 0; w >>= 1) {
        if ((int)threadIdx.x < w) sh[threadIdx.x] += sh[threadIdx.x + w];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = sh[0] * inv_norm;
}

// In host code the array's name is a host-side stand-in, not a device address: the kernel gets what
// cudaGetSymbolAddress returns, looked up once per device with that device current.
constexpr int kMaxDevices = 64;
double* g_static_partials_ptr[kMaxDevices] = {};

cudaError_t plaquette_static_ptr(double** ptr) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    if (!g_static_partials_ptr[dev]) {
        double* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, g_plaquette_static_partials);
        if (e != cudaSuccess) return e;
        g_static_partials_ptr[dev] = p;
    }
    *ptr = g_static_partials_ptr[dev];
    return cudaSuccess;
}

}  // namespace

cudaError_t launch_plaquette_static(int precision, int recon, const Geometry& g, const void* gauge, double* out_dev,
                                    cudaStream_t st) {
    double* scratch = nullptr;
    cudaError_t e = plaquette_static_ptr(&scratch);
    if (e != cudaSuccess) return e;
    GaugeArgs a;
    a.gauge = const_cast<void*>(gauge); a.g = g; a.mu = 0; a.parity = 0; a.beta = 0; a.c_il = 0; a.seed = 0; a.tag = 0;
    a.red.partials = scratch;
    const dim3 grid((g.Vh + 127) / 128, 2);
    count_launch(2);
    if (precision == 0) {
        if (recon == 12) plaquette_kernel<double, 12><<<grid, 128, 0, st>>>(a);
        else             plaquette_kernel<double, 18><<<grid, 128, 0, st>>>(a);
    } else {
        if (recon == 12) plaquette_kernel<float, 12><<<grid, 128, 0, st>>>(a);
        else             plaquette_kernel<float, 18><<<grid, 128, 0, st>>>(a);
    }
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    // sum of Re tr over the 6 V plaquettes -> average of Re tr / 3
    plaquette_static_sum_kernel<<<1, 256, 0, st>>>(plaquette_partials(g.Vh), 1.0 / (3.0 * 6.0 * 2.0 * (double)g.Vh), out_dev);
    return cudaGetLastError();
}

}  // namespace lqcd
