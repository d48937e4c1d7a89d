// vector_ops.cu -- fused CG vector kernels (the paper's
// "saxpy" and "LAPACK operations", written there
// "in a straightforward manner").  Here: two passes per iteration instead of five,
// 128-bit loads, warp-shuffle block sums written as one partial per block, and a separate
// one-block finalize_kernel that adds the partials in a fixed order and applies the scalar
// recurrence, so that alpha, beta and the convergence decision never leave the device.
//
//   cg_init      x = 0, r = p = b; finalize(FIN_BB): rho = bb = |b|^2
//   (r -= alpha q and |r|^2 live in the epilogue of the iteration's last hopping launch,
//    hopping.cu MODE 3: q is never stored)
//                finalize(FIN_RHO): iters++, done = (rho' <= tol^2 bb), beta = rho'/rho, rho = rho'
//   cg_update_xp x += alpha p; p = r + beta p (p only while not converged)  (5 fields of traffic)
//   true_resid   |b - Ax|^2; finalize(FIN_TRUE)
// i.e. 5 + 2 (r read/written by the hopping launch) field transfers per iteration instead of
// the 12 of unfused BLAS-1.
// Reductions accumulate in double whatever the field precision.
#include "lqcd_internal.h"

namespace lqcd {
namespace {

constexpr int VBLOCK = 256;
constexpr int VUNROLL = 4;

template <typename T> struct VecOf;
template <> struct VecOf<double> { typedef double2 type; static constexpr int width = 2; };
template <> struct VecOf<float>  { typedef float4 type;  static constexpr int width = 4; };

__device__ __forceinline__ double2 axpy(double a, double2 x, double2 y) {
    return make_double2(fma(a, x.x, y.x), fma(a, x.y, y.y));
}
__device__ __forceinline__ float4 axpy(double a, float4 x, float4 y) {
    const float f = (float)a;
    return make_float4(fmaf(f, x.x, y.x), fmaf(f, x.y, y.y), fmaf(f, x.z, y.z), fmaf(f, x.w, y.w));
}
__device__ __forceinline__ double2 sub(double2 x, double2 y) { return make_double2(x.x - y.x, x.y - y.y); }
__device__ __forceinline__ float4 sub(float4 x, float4 y) {
    return make_float4(x.x - y.x, x.y - y.y, x.z - y.z, x.w - y.w);
}
__device__ __forceinline__ double norm2(double2 v) { return v.x * v.x + v.y * v.y; }
__device__ __forceinline__ double norm2(float4 v) {
    return (double)v.x * v.x + (double)v.y * v.y + (double)v.z * v.z + (double)v.w * v.w;
}
__device__ __forceinline__ void zero(double2& v) { v = make_double2(0.0, 0.0); }
__device__ __forceinline__ void zero(float4& v) { v = make_float4(0.f, 0.f, 0.f, 0.f); }

// fixed-order block sum; thread 0 stores the block's partial (no fence, no atomic)
__device__ __forceinline__ void block_partial(double v, Reduction red) {
    __shared__ double sm[VBLOCK / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    v = warp_sum(v);
    if (lane == 0) sm[warp] = v;
    __syncthreads();
    if (warp == 0) {
        v = (lane < VBLOCK / 32) ? sm[lane] : 0.0;
        v = warp_sum(v);
        if (lane == 0) red.partials[blockIdx.x] = v;
    }
}

// One block: adds the partials in index order (thread-strided, then a fixed tree) and applies
// the scalar step of the recurrence on the device.
//
// Slab mode (several ranks, lqcd_slab_*) splits it around the all-reduce of the caller:
//   sum_io != null, apply = 0: only the rank's own sum is formed and stored to *sum_io;
//   sum_io != null, apply = 1: no summation, the (all-reduced) value of *sum_io is applied.
__global__ void __launch_bounds__(1024) finalize_kernel(int fin, Reduction red, int n, double tol,
                                                        CgScalars* scal, double* sum_io, int apply) {
    chain_prologue();
    __shared__ double sm[32];
    if (fin != FIN_BB && fin != FIN_TRUE && scal->done) {
        if (fin == FIN_RHO && threadIdx.x == 0 && (sum_io == nullptr || apply)) scal->upd = 0;  // nothing for cg_update_xp to apply
        if (sum_io != nullptr && !apply && threadIdx.x == 0) *sum_io = 0.0;
        return;
    }
    double s = 0.0;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (sum_io != nullptr && apply) {
        if (threadIdx.x != 0) return;
        s = *sum_io;
    } else {
        for (int i = threadIdx.x; i < n; i += 1024) s += red.partials[i];
        s = warp_sum(s);
        if (lane == 0) sm[warp] = s;
        __syncthreads();
        if (warp != 0) return;
        s = warp_sum(sm[lane]);
        if (lane != 0) return;
        if (sum_io != nullptr) { *sum_io = s; return; }
    }
    if (fin == FIN_PAP) {
        const double rho = scal->rho;
        scal->pAp = s;
        if (!(s > 0.0) || !isfinite(s) || !isfinite(rho)) {  // breakdown: r and x stay untouched
            scal->status = -5;
            scal->done = 1;
            scal->upd = 0;
        } else {
            scal->alpha = rho / s;
            scal->inv_alpha = s / rho;
        }
    } else if (fin == FIN_BB) {
        scal->bb = s;
        scal->rho = s;
        scal->pAp = 0.0;
        scal->beta = 0.0;
        scal->tol2bb = tol * tol * s;
        scal->resid_true = 0.0;
        scal->iters = 0;
        scal->done = (s == 0.0) ? 1 : 0;
        scal->status = (s == 0.0) ? 0 : 1;
        scal->upd = 0;
    } else if (fin == FIN_RHO) {
        const double rho = scal->rho;
        scal->iters += 1;
        scal->upd = 1;
        if (s <= scal->tol2bb) {
            scal->done = 1;
            scal->status = 0;
        }
        scal->beta = s / rho;
        scal->rho = s;
    } else if (fin == FIN_TRUE) {
        scal->resid_true = s;
    }
}

template <typename T>
__global__ void __launch_bounds__(VBLOCK) cg_init_kernel(size_t nvec, const void* b_, void* x_, void* r_,
                                                         void* p_, Reduction red) {
    chain_prologue();
    typedef typename VecOf<T>::type V;
    const V* b = (const V*)b_;
    V *x = (V*)x_, *r = (V*)r_, *p = (V*)p_;
    const size_t base = (size_t)blockIdx.x * (VBLOCK * VUNROLL) + threadIdx.x;
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < VUNROLL; ++k) {
        const size_t i = base + (size_t)k * VBLOCK;
        if (i < nvec) {
            const V v = b[i];
            V z;
            zero(z);
            x[i] = z;
            r[i] = v;
            p[i] = v;
            s += norm2(v);
        }
    }
    block_partial(s, red);
}

template <typename T>
__global__ void __launch_bounds__(VBLOCK) cg_update_xp_kernel(size_t nvec, void* x_, void* p_,
                                                              const void* r_, int reverse,
                                                              CgScalars* scal) {
    typedef typename VecOf<T>::type V;
    chain_prologue();
    if (!scal->upd) return;            // no r-update happened in this iteration
    const bool more = !scal->done;     // converged in this iteration: x gets its last update, p is dead
    const double alpha = scal->alpha, beta = scal->beta;
    V *x = (V*)x_, *p = (V*)p_;
    const V* r = (const V*)r_;
    const size_t blk = reverse ? (gridDim.x - 1 - blockIdx.x) : blockIdx.x;
    const size_t base = blk * (VBLOCK * VUNROLL) + threadIdx.x;
    V xv[VUNROLL], pv[VUNROLL], rv[VUNROLL];
#pragma unroll
    for (int k = 0; k < VUNROLL; ++k) {
        const size_t i = base + (size_t)k * VBLOCK;
        if (i < nvec) { xv[k] = x[i]; pv[k] = p[i]; if (more) rv[k] = __ldg(r + i); }
    }
#pragma unroll
    for (int k = 0; k < VUNROLL; ++k) {
        const size_t i = base + (size_t)k * VBLOCK;
        if (i < nvec) {
            x[i] = axpy(alpha, pv[k], xv[k]);
            if (more) p[i] = axpy(beta, pv[k], rv[k]);
        }
    }
}

template <typename T>
__global__ void __launch_bounds__(VBLOCK) true_resid_kernel(size_t nvec, const void* b_, const void* ax_,
                                                            Reduction red) {
    chain_prologue();
    typedef typename VecOf<T>::type V;
    const V *b = (const V*)b_, *ax = (const V*)ax_;
    const size_t base = (size_t)blockIdx.x * (VBLOCK * VUNROLL) + threadIdx.x;
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < VUNROLL; ++k) {
        const size_t i = base + (size_t)k * VBLOCK;
        if (i < nvec) s += norm2(sub(__ldg(b + i), __ldg(ax + i)));
    }
    block_partial(s, red);
}

// ---- mixed-precision helpers.  Double field: double2 d[G][12][32]; float field: float4 f[G][6][32]
// with f[g][k][l] = (d[g][2k][l], d[g][2k+1][l]).  One thread per float4 element.
__global__ void __launch_bounds__(VBLOCK) convert_d2f_kernel(size_t nf4, const double2* __restrict__ d,
                                                             float4* __restrict__ f, double scale) {
    const size_t i = (size_t)blockIdx.x * VBLOCK + threadIdx.x;
    if (i >= nf4) return;
    const size_t g = i / 192, r = i - g * 192, k = r >> 5, l = r & 31;
    const double2* p = d + g * 384 + (2 * k) * 32 + l;
    const double2 a = __ldcs(p), b = __ldcs(p + 32);
    f[i] = make_float4((float)(a.x * scale), (float)(a.y * scale), (float)(b.x * scale), (float)(b.y * scale));
}

__global__ void __launch_bounds__(VBLOCK) axpy_f2d_kernel(size_t nf4, double a, const float4* __restrict__ x,
                                                          double2* __restrict__ y) {
    const size_t i = (size_t)blockIdx.x * VBLOCK + threadIdx.x;
    if (i >= nf4) return;
    const size_t g = i / 192, r = i - g * 192, k = r >> 5, l = r & 31;
    const float4 v = __ldcs(x + i);
    double2* y0 = y + g * 384 + (2 * k) * 32 + l;
    double2* y1 = y0 + 32;
    const double2 u0 = *y0, u1 = *y1;
    *y0 = make_double2(fma(a, (double)v.x, u0.x), fma(a, (double)v.y, u0.y));
    *y1 = make_double2(fma(a, (double)v.z, u1.x), fma(a, (double)v.w, u1.y));
}

__global__ void __launch_bounds__(VBLOCK) residual_kernel(size_t nvec, const double2* __restrict__ b,
                                                          const double2* __restrict__ ax,
                                                          double2* __restrict__ r, Reduction red) {
    const size_t base = (size_t)blockIdx.x * (VBLOCK * VUNROLL) + threadIdx.x;
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < VUNROLL; ++k) {
        const size_t i = base + (size_t)k * VBLOCK;
        if (i < nvec) {
            const double2 v = sub(__ldg(b + i), __ldcs(ax + i));
            r[i] = v;
            s += norm2(v);
        }
    }
    block_partial(s, red);
}

// out = a_chi * in per site, a_chi complex per chirality (upper: components 0..5, lower: 6..11):
// the diagonal term (1 + i c gamma5) or its inverse on a whole half field.  One thread per
// double2 / float4 element of the grouped layout (lqcd_internal.h).
__global__ void __launch_bounds__(VBLOCK) diag_scale_kernel_d(size_t nvec, const double2* __restrict__ in,
                                                              double2* __restrict__ out, double ur, double ui,
                                                              double dr, double di) {
    const size_t i = (size_t)blockIdx.x * VBLOCK + threadIdx.x;
    if (i >= nvec) return;
    const bool upper = ((i % 384) >> 5) < 6;
    const double ar = upper ? ur : dr, ai = upper ? ui : di;
    const double2 v = in[i];
    out[i] = make_double2(ar * v.x - ai * v.y, ar * v.y + ai * v.x);
}
__global__ void __launch_bounds__(VBLOCK) diag_scale_kernel_f(size_t nvec, const float4* __restrict__ in,
                                                              float4* __restrict__ out, float ur, float ui,
                                                              float dr, float di) {
    const size_t i = (size_t)blockIdx.x * VBLOCK + threadIdx.x;
    if (i >= nvec) return;
    const bool upper = ((i % 192) >> 5) < 3;
    const float ar = upper ? ur : dr, ai = upper ? ui : di;
    const float4 v = in[i];
    out[i] = make_float4(ar * v.x - ai * v.y, ar * v.y + ai * v.x, ar * v.z - ai * v.w, ar * v.w + ai * v.z);
}

// ----------------------------------------------------------------------------- BiCGStab on Mhat
// (PAPER.md:94 names CG and BiCGStab; reading G15 for the recurrence).  Complex
// scalars live in BiScalars on the device; one iteration is
//   v = Mhat p, <rhat,v> from the hopping launch (MODE 4) -> alpha | bicg_s: s = r - alpha v |
//   t = Mhat s, <s,t>, |t|^2 from the hopping launch -> omega | bicg_xr: x += alpha p + omega s,
//   r = s - omega t, |r|^2, <rhat,r> -> beta, convergence | bicg_p: p = r + beta (p - omega v)
//   bicg_xrp: the last two in one pass, possible because rho' = <rhat, r'> = (rho - alpha sigma) - omega <rhat, t>
//   is known before r' exists (<rhat, t> comes out of the hopping launch as well, MODE 5), so beta is too
// = 3 + 8 field transfers in vector kernels + two (rhat, twice) read by hopping launches, besides the
// four hopping launches (18 + 4 when every step is a kernel of its own: bicg_sigma, bicg_omega, bicg_xr,
// bicg_p, which remain as the plain form of the recurrence).
struct cd { double re, im; };
__device__ __forceinline__ cd cmul(cd a, cd b) { return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
__device__ __forceinline__ cd cdiv(cd a, cd b) {
    const double d = b.re * b.re + b.im * b.im;
    return {(a.re * b.re + a.im * b.im) / d, (a.im * b.re - a.re * b.im) / d};
}
__device__ __forceinline__ bool cbad(cd a) { return (a.re == 0.0 && a.im == 0.0) || !isfinite(a.re) || !isfinite(a.im); }

// y + a x, a complex, on one (double2) or two (float4) complex numbers
__device__ __forceinline__ double2 caxpy(cd a, double2 x, double2 y) {
    return make_double2(fma(-a.im, x.y, fma(a.re, x.x, y.x)), fma(a.im, x.x, fma(a.re, x.y, y.y)));
}
__device__ __forceinline__ float4 caxpy(cd a, float4 x, float4 y) {
    const float ar = (float)a.re, ai = (float)a.im;
    return make_float4(fmaf(-ai, x.y, fmaf(ar, x.x, y.x)), fmaf(ai, x.x, fmaf(ar, x.y, y.y)),
                       fmaf(-ai, x.w, fmaf(ar, x.z, y.z)), fmaf(ai, x.z, fmaf(ar, x.w, y.w)));
}
// sum conj(a_i) b_i accumulated in double
__device__ __forceinline__ void cdot_acc(double2 a, double2 b, double& re, double& im) {
    re += a.x * b.x + a.y * b.y;
    im += a.x * b.y - a.y * b.x;
}
__device__ __forceinline__ void cdot_acc(float4 a, float4 b, double& re, double& im) {
    re += (double)a.x * b.x + (double)a.y * b.y + (double)a.z * b.z + (double)a.w * b.w;
    im += (double)a.x * b.y - (double)a.y * b.x + (double)a.z * b.w - (double)a.w * b.z;
}

// K block sums at once; partial k of block b goes to red.partials[k * gridDim.x + b]
template <int K>
__device__ __forceinline__ void block_partials(double (&v)[K], Reduction red) {
    __shared__ double sm[K][VBLOCK / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        v[k] = warp_sum(v[k]);
        if (lane == 0) sm[k][warp] = v[k];
    }
    __syncthreads();
    if (warp == 0) {
#pragma unroll
        for (int k = 0; k < K; ++k) {
            double w = (lane < VBLOCK / 32) ? sm[k][lane] : 0.0;
            w = warp_sum(w);
            if (lane == 0) red.partials[(size_t)k * gridDim.x + blockIdx.x] = w;
        }
    }
}

__global__ void __launch_bounds__(1024) bicg_finalize_kernel(int fin, Reduction red, int n, double tol,
                                                             BiScalars* bs) {
    chain_prologue();
    __shared__ double sm[5][32];
    if (fin != FIN_BI_INIT && bs->cg.done) return;
    double s[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    const int K = (fin == FIN_BI_INIT || fin == FIN_BI_R2) ? 1 : (fin == FIN_BI_SIGMA) ? 2 : (fin == FIN_BI_OMEGA_BETA) ? 5 : 3;
    const int fin_in = fin;
    for (int k = 0; k < K; ++k)
        for (int i = threadIdx.x; i < n; i += 1024) s[k] += red.partials[(size_t)k * n + i];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int k = 0; k < K; ++k) {
        s[k] = warp_sum(s[k]);
        if (lane == 0) sm[k][warp] = s[k];
    }
    __syncthreads();
    if (warp != 0) return;
    for (int k = 0; k < K; ++k) s[k] = warp_sum(sm[k][lane]);
    if (lane != 0) return;
    if (fin_in == FIN_BI_SIGMA_HOP) {        // (|v|^2, <rhat, v>) -> (<rhat, v>)
        s[0] = s[1]; s[1] = s[2];
        fin = FIN_BI_SIGMA;
    } else if (fin_in == FIN_BI_OMEGA_HOP) { // (|t|^2, <s, t>) -> (<t, s> = conj <s, t>, |t|^2)
        const double tt = s[0];
        s[0] = s[1]; s[1] = -s[2]; s[2] = tt;
        fin = FIN_BI_OMEGA;
    }
    if (fin == FIN_BI_INIT) {           // s0 = |b|^2; rhat = r = b so rho = <rhat, r> = |b|^2
        CgScalars& c = bs->cg;
        c.bb = s[0]; c.rho = s[0]; c.pAp = 0.0; c.beta = 0.0; c.alpha = 0.0; c.inv_alpha = 0.0;
        c.tol2bb = tol * tol * s[0]; c.resid_true = 0.0; c.iters = 0;
        c.done = (s[0] == 0.0) ? 1 : 0;
        c.status = (s[0] == 0.0) ? 0 : 1;
        c.upd = 0;
        bs->rho_re = s[0]; bs->rho_im = 0.0;
        bs->alpha_re = bs->alpha_im = bs->omega_re = bs->omega_im = bs->beta_re = bs->beta_im = 0.0;
        bs->sigma_re = bs->sigma_im = 0.0;
        bs->pend = 0;
    } else if (fin == FIN_BI_SIGMA) {   // sigma = <rhat, v>; alpha = rho / sigma
        const cd sigma = {s[0], s[1]};
        if (cbad(sigma)) { bs->cg.status = -5; bs->cg.done = 1; return; }
        const cd a = cdiv({bs->rho_re, bs->rho_im}, sigma);
        bs->alpha_re = a.re; bs->alpha_im = a.im;
        bs->sigma_re = sigma.re; bs->sigma_im = sigma.im;
    } else if (fin == FIN_BI_OMEGA) {   // omega = <t, s> / |t|^2 (0 if t = 0)
        const double tt = s[2];
        bs->omega_re = tt > 0.0 ? s[0] / tt : 0.0;
        bs->omega_im = tt > 0.0 ? s[1] / tt : 0.0;
    } else if (fin == FIN_BI_OMEGA_BETA) {   // s = (|t|^2, <s,t>, <rhat,t>)
        const double tt = s[0];
        const cd omega = {tt > 0.0 ? s[1] / tt : 0.0, tt > 0.0 ? -s[2] / tt : 0.0};   // <t,s> / |t|^2, <t,s> = conj <s,t>
        bs->omega_re = omega.re; bs->omega_im = omega.im;
        const cd rho = {bs->rho_re, bs->rho_im}, alpha = {bs->alpha_re, bs->alpha_im};
        const cd as = cmul(alpha, {bs->sigma_re, bs->sigma_im});
        const cd ot = cmul(omega, {s[3], s[4]});
        const cd rho1 = {(rho.re - as.re) - ot.re, (rho.im - as.im) - ot.im};
        if (cbad(rho1) || cbad(omega)) {   // decided by FIN_BI_R2, once |r'| is known
            bs->pend = 1;
            bs->beta_re = bs->beta_im = 0.0;
        } else {
            const cd beta = cmul(cdiv(rho1, rho), cdiv(alpha, omega));
            bs->beta_re = beta.re; bs->beta_im = beta.im;
            bs->rho_re = rho1.re; bs->rho_im = rho1.im;
        }
    } else if (fin == FIN_BI_R2) {      // s0 = |r'|^2
        CgScalars& c = bs->cg;
        c.iters += 1;
        c.rho = s[0];
        if (s[0] <= c.tol2bb) { c.done = 1; c.status = 0; return; }
        if (bs->pend || !isfinite(s[0])) { c.status = -5; c.done = 1; }
    } else if (fin == FIN_BI_R) {       // s0 = |r|^2, (s1, s2) = rho' = <rhat, r>
        CgScalars& c = bs->cg;
        c.iters += 1;
        c.rho = s[0];
        if (s[0] <= c.tol2bb) { c.done = 1; c.status = 0; return; }
        const cd rho1 = {s[1], s[2]}, omega = {bs->omega_re, bs->omega_im};
        if (cbad(rho1) || cbad(omega) || !isfinite(s[0])) { c.status = -5; c.done = 1; return; }
        const cd beta = cmul(cdiv(rho1, {bs->rho_re, bs->rho_im}), cdiv({bs->alpha_re, bs->alpha_im}, omega));
        bs->beta_re = beta.re; bs->beta_im = beta.im;
        bs->rho_re = rho1.re; bs->rho_im = rho1.im;
    }
}

#define LQCD_VEC_INDEX                                                              \
    const size_t blk = reverse ? (gridDim.x - 1 - blockIdx.x) : blockIdx.x;         \
    const size_t base = blk * (VBLOCK * VUNROLL) + threadIdx.x

template <typename T>
__global__ void __launch_bounds__(VBLOCK) bicg_sigma_kernel(size_t nvec, const void* rhat_, const void* v_,
                                                            int reverse, Reduction red, const BiScalars* bs) {
    typedef typename VecOf<T>::type V;
    if (bs->cg.done) return;
    const V *rhat = (const V*)rhat_, *v = (const V*)v_;
    LQCD_VEC_INDEX;
    double s[2] = {0.0, 0.0};
#pragma unroll
    for (int k = 0; k < VUNROLL; ++k) {
        const size_t i = base + (size_t)k * VBLOCK;
        if (i < nvec) cdot_acc(__ldg(rhat + i), __ldg(v + i), s[0], s[1]);
    }
    block_partials<2>(s, red);
}

template <typename T>
__global__ void __launch_bounds__(VBLOCK) bicg_s_kernel(size_t nvec, const void* r_, const void* v_, void* s_,
                                                        int reverse, const BiScalars* bs) {
    chain_prologue();
    typedef typename VecOf<T>::type V;
    if (bs->cg.done) return;
    const cd ma = {-bs->alpha_re, -bs->alpha_im};
    const V *r = (const V*)r_, *v = (const V*)v_;
    V* s = (V*)s_;
    LQCD_VEC_INDEX;
#pragma unroll
    for (int k = 0; k < VUNROLL; ++k) {
        const size_t i = base + (size_t)k * VBLOCK;
        if (i < nvec) s[i] = caxpy(ma, __ldg(v + i), __ldg(r + i));
    }
}

template <typename T>
__global__ void __launch_bounds__(VBLOCK) bicg_omega_kernel(size_t nvec, const void* t_, const void* s_,
                                                            int reverse, Reduction red, const BiScalars* bs) {
    typedef typename VecOf<T>::type V;
    if (bs->cg.done) return;
    const V *t = (const V*)t_, *s = (const V*)s_;
    LQCD_VEC_INDEX;
    double a[3] = {0.0, 0.0, 0.0};
#pragma unroll
    for (int k = 0; k < VUNROLL; ++k) {
        const size_t i = base + (size_t)k * VBLOCK;
        if (i < nvec) {
            const V tv = __ldg(t + i);
            cdot_acc(tv, __ldg(s + i), a[0], a[1]);
            a[2] += norm2(tv);
        }
    }
    block_partials<3>(a, red);
}

template <typename T>
__global__ void __launch_bounds__(VBLOCK) bicg_xr_kernel(size_t nvec, void* x_, const void* p_, const void* s_,
                                                         const void* t_, const void* rhat_, void* r_,
                                                         int reverse, Reduction red, const BiScalars* bs) {
    typedef typename VecOf<T>::type V;
    if (bs->cg.done) return;
    const cd alpha = {bs->alpha_re, bs->alpha_im}, omega = {bs->omega_re, bs->omega_im};
    const cd momega = {-omega.re, -omega.im};
    V *x = (V*)x_, *r = (V*)r_;
    const V *p = (const V*)p_, *s = (const V*)s_, *t = (const V*)t_, *rhat = (const V*)rhat_;
    LQCD_VEC_INDEX;
    double a[3] = {0.0, 0.0, 0.0};
#pragma unroll
    for (int k = 0; k < VUNROLL; ++k) {
        const size_t i = base + (size_t)k * VBLOCK;
        if (i < nvec) {
            const V sv = __ldg(s + i);
            x[i] = caxpy(omega, sv, caxpy(alpha, __ldg(p + i), x[i]));
            const V rn = caxpy(momega, __ldcs(t + i), sv);
            r[i] = rn;
            a[0] += norm2(rn);
            cdot_acc(__ldg(rhat + i), rn, a[1], a[2]);
        }
    }
    block_partials<3>(a, red);
}

// the merged pass: x += alpha p + omega s;  r' = s - omega t;  p' = r' + beta (p - omega v);  |r'|^2
template <typename T>
__global__ void __launch_bounds__(VBLOCK) bicg_xrp_kernel(size_t nvec, void* x_, void* p_, const void* s_, const void* t_,
                                                          const void* v_, void* r_, int reverse, Reduction red,
                                                          const BiScalars* bs) {
    chain_prologue();
    typedef typename VecOf<T>::type V;
    if (bs->cg.done) return;
    const cd alpha = {bs->alpha_re, bs->alpha_im}, omega = {bs->omega_re, bs->omega_im}, beta = {bs->beta_re, bs->beta_im};
    const cd momega = {-omega.re, -omega.im};
    V *x = (V*)x_, *r = (V*)r_, *p = (V*)p_;
    const V *s = (const V*)s_, *t = (const V*)t_, *v = (const V*)v_;
    LQCD_VEC_INDEX;
    double a[1] = {0.0};
#pragma unroll
    for (int k = 0; k < VUNROLL; ++k) {
        const size_t i = base + (size_t)k * VBLOCK;
        if (i < nvec) {
            const V sv = __ldcs(s + i), pv = p[i];
            x[i] = caxpy(omega, sv, caxpy(alpha, pv, x[i]));
            const V rn = caxpy(momega, __ldcs(t + i), sv);
            r[i] = rn;
            a[0] += norm2(rn);
            p[i] = caxpy(beta, caxpy(momega, __ldcs(v + i), pv), rn);
        }
    }
    block_partials<1>(a, red);
}

template <typename T>
__global__ void __launch_bounds__(VBLOCK) bicg_p_kernel(size_t nvec, void* p_, const void* r_, const void* v_,
                                                        int reverse, const BiScalars* bs) {
    typedef typename VecOf<T>::type V;
    if (bs->cg.done) return;
    const cd beta = {bs->beta_re, bs->beta_im}, momega = {-bs->omega_re, -bs->omega_im};
    V* p = (V*)p_;
    const V *r = (const V*)r_, *v = (const V*)v_;
    LQCD_VEC_INDEX;
#pragma unroll
    for (int k = 0; k < VUNROLL; ++k) {
        const size_t i = base + (size_t)k * VBLOCK;
        if (i < nvec) p[i] = caxpy(beta, caxpy(momega, __ldcs(v + i), p[i]), __ldg(r + i));
    }
}

inline int grid_for(size_t nvec) { return (int)((nvec + VBLOCK * VUNROLL - 1) / (VBLOCK * VUNROLL)); }

}  // namespace

int vector_grid(size_t n) { return grid_for(n / 2); }  // upper bound over both precisions

cudaError_t launch_finalize(int fin, Reduction red, int n_partials, double tol, CgScalars* scal,
                            cudaStream_t st, double* sum_io, int apply) {
    count_launch();
    ProfScope prof(3, st);
    return launch_chained(chained_launches(st), finalize_kernel, 1, 1024, 0, st, fin, red, n_partials, tol, scal, sum_io, apply);
}

cudaError_t launch_diag_scale(int precision, size_t n, const void* in, void* out, double ur, double ui,
                              double dr, double di, cudaStream_t st) {
    count_launch();
    ProfScope prof(3, st);
    if (precision == 0) {
        const size_t nv = n / 2;
        diag_scale_kernel_d<<<(int)((nv + VBLOCK - 1) / VBLOCK), VBLOCK, 0, st>>>(nv, (const double2*)in, (double2*)out,
                                                                             ur, ui, dr, di);
    } else {
        const size_t nv = n / 4;
        diag_scale_kernel_f<<<(int)((nv + VBLOCK - 1) / VBLOCK), VBLOCK, 0, st>>>(nv, (const float4*)in, (float4*)out,
                                                                             (float)ur, (float)ui, (float)dr, (float)di);
    }
    return cudaGetLastError();
}

cudaError_t launch_convert_d2f(size_t n, const void* src_d, void* dst_f, double scale, cudaStream_t st) {
    const size_t nf4 = n / 4;
    count_launch();
    ProfScope prof(3, st);
    convert_d2f_kernel<<<(int)((nf4 + VBLOCK - 1) / VBLOCK), VBLOCK, 0, st>>>(nf4, (const double2*)src_d,
                                                                              (float4*)dst_f, scale);
    return cudaGetLastError();
}

cudaError_t launch_axpy_f2d(size_t n, double a, const void* x_f, void* y_d, cudaStream_t st) {
    const size_t nf4 = n / 4;
    count_launch();
    ProfScope prof(3, st);
    axpy_f2d_kernel<<<(int)((nf4 + VBLOCK - 1) / VBLOCK), VBLOCK, 0, st>>>(nf4, a, (const float4*)x_f,
                                                                           (double2*)y_d);
    return cudaGetLastError();
}

cudaError_t launch_residual(size_t n, const void* b, const void* ax, void* r, Reduction red,
                            CgScalars* scal, cudaStream_t st) {
    const size_t nv = n / 2;
    count_launch(2);
    ProfScope prof(3, st);
    residual_kernel<<<grid_for(nv), VBLOCK, 0, st>>>(nv, (const double2*)b, (const double2*)ax, (double2*)r, red);
    finalize_kernel<<<1, 1024, 0, st>>>(FIN_TRUE, red, grid_for(nv), 0.0, scal, nullptr, 0);
    return cudaGetLastError();
}

cudaError_t launch_cg_init(int precision, size_t n, const void* b, void* x, void* r, void* p,
                           double tol, Reduction red, CgScalars* scal, cudaStream_t st, double* sum_io) {
    count_launch(2);
    ProfScope prof(3, st);
    if (precision == 0) {
        const size_t nv = n / 2;
        cg_init_kernel<double><<<grid_for(nv), VBLOCK, 0, st>>>(nv, b, x, r, p, red);
        finalize_kernel<<<1, 1024, 0, st>>>(FIN_BB, red, grid_for(nv), tol, scal, sum_io, 0);
    } else {
        const size_t nv = n / 4;
        cg_init_kernel<float><<<grid_for(nv), VBLOCK, 0, st>>>(nv, b, x, r, p, red);
        finalize_kernel<<<1, 1024, 0, st>>>(FIN_BB, red, grid_for(nv), tol, scal, sum_io, 0);
    }
    return cudaGetLastError();
}

cudaError_t launch_cg_update_xp(int precision, size_t n, void* x, void* p, const void* r, int reverse,
                                CgScalars* scal, cudaStream_t st) {
    count_launch();
    ProfScope prof(3, st);
    if (precision == 0) {
        const size_t nv = n / 2;
        return launch_chained(chained_launches(st), cg_update_xp_kernel<double>, grid_for(nv), VBLOCK, 0, st, nv, x, p, r, reverse, scal);
    } else {
        const size_t nv = n / 4;
        return launch_chained(chained_launches(st), cg_update_xp_kernel<float>, grid_for(nv), VBLOCK, 0, st, nv, x, p, r, reverse, scal);
    }
    return cudaGetLastError();
}

cudaError_t launch_true_resid(int precision, size_t n, const void* b, const void* ax, Reduction red,
                              CgScalars* scal, cudaStream_t st, double* sum_io) {
    count_launch(2);
    ProfScope prof(3, st);
    if (precision == 0) {
        const size_t nv = n / 2;
        true_resid_kernel<double><<<grid_for(nv), VBLOCK, 0, st>>>(nv, b, ax, red);
        finalize_kernel<<<1, 1024, 0, st>>>(FIN_TRUE, red, grid_for(nv), 0.0, scal, sum_io, 0);
    } else {
        const size_t nv = n / 4;
        true_resid_kernel<float><<<grid_for(nv), VBLOCK, 0, st>>>(nv, b, ax, red);
        finalize_kernel<<<1, 1024, 0, st>>>(FIN_TRUE, red, grid_for(nv), 0.0, scal, sum_io, 0);
    }
    return cudaGetLastError();
}

// ---- BiCGStab launchers (nv = 128-bit elements of one field)
#define LQCD_BICG_DISPATCH(KERNEL, ...)                                                        \
    do {                                                                                       \
        if (precision == 0) { const size_t nv = n / 2; KERNEL<double><<<grid_for(nv), VBLOCK, 0, st>>>(nv, __VA_ARGS__); } \
        else                { const size_t nv = n / 4; KERNEL<float><<<grid_for(nv), VBLOCK, 0, st>>>(nv, __VA_ARGS__); }  \
    } while (0)
// the same for the kernels of the production iteration, which begin with chain_prologue() (lqcd_internal.h)
#define LQCD_BICG_DISPATCH_CHAINED(KERNEL, ...)                                                \
    do {                                                                                       \
        const bool ch_ = chained_launches(st);                                                 \
        if (precision == 0) { const size_t nv = n / 2; (void)launch_chained(ch_, KERNEL<double>, grid_for(nv), VBLOCK, 0, st, nv, __VA_ARGS__); } \
        else                { const size_t nv = n / 4; (void)launch_chained(ch_, KERNEL<float>, grid_for(nv), VBLOCK, 0, st, nv, __VA_ARGS__); }  \
    } while (0)

static int bicg_grid(int precision, size_t n) { return grid_for(precision == 0 ? n / 2 : n / 4); }

cudaError_t launch_bicg_init(int precision, size_t n, const void* b, void* x, void* r, void* p, double tol,
                             Reduction red, BiScalars* bs, cudaStream_t st) {
    count_launch(2);
    ProfScope prof(3, st);
    LQCD_BICG_DISPATCH(cg_init_kernel, b, x, r, p, red);
    bicg_finalize_kernel<<<1, 1024, 0, st>>>(FIN_BI_INIT, red, bicg_grid(precision, n), tol, bs);
    return cudaGetLastError();
}

cudaError_t launch_bicg_sigma(int precision, size_t n, const void* rhat, const void* v, int reverse,
                              Reduction red, BiScalars* bs, cudaStream_t st) {
    count_launch(2);
    ProfScope prof(3, st);
    LQCD_BICG_DISPATCH(bicg_sigma_kernel, rhat, v, reverse, red, bs);
    bicg_finalize_kernel<<<1, 1024, 0, st>>>(FIN_BI_SIGMA, red, bicg_grid(precision, n), 0.0, bs);
    return cudaGetLastError();
}

cudaError_t launch_bicg_s(int precision, size_t n, const void* r, const void* v, void* s, int reverse,
                          BiScalars* bs, cudaStream_t st) {
    count_launch();
    ProfScope prof(3, st);
    LQCD_BICG_DISPATCH_CHAINED(bicg_s_kernel, r, v, s, reverse, bs);
    return cudaGetLastError();
}

cudaError_t launch_bicg_omega(int precision, size_t n, const void* t, const void* s, int reverse,
                              Reduction red, BiScalars* bs, cudaStream_t st) {
    count_launch(2);
    ProfScope prof(3, st);
    LQCD_BICG_DISPATCH(bicg_omega_kernel, t, s, reverse, red, bs);
    bicg_finalize_kernel<<<1, 1024, 0, st>>>(FIN_BI_OMEGA, red, bicg_grid(precision, n), 0.0, bs);
    return cudaGetLastError();
}

cudaError_t launch_bicg_xr(int precision, size_t n, void* x, const void* p, const void* s, const void* t,
                           const void* rhat, void* r, int reverse, Reduction red, BiScalars* bs,
                           cudaStream_t st) {
    count_launch(2);
    ProfScope prof(3, st);
    LQCD_BICG_DISPATCH(bicg_xr_kernel, x, p, s, t, rhat, r, reverse, red, bs);
    bicg_finalize_kernel<<<1, 1024, 0, st>>>(FIN_BI_R, red, bicg_grid(precision, n), 0.0, bs);
    return cudaGetLastError();
}

cudaError_t launch_bicg_xrp(int precision, size_t n, void* x, void* p, const void* s, const void* t, const void* v,
                            void* r, int reverse, Reduction red, BiScalars* bs, cudaStream_t st) {
    count_launch(2);
    ProfScope prof(3, st);
    LQCD_BICG_DISPATCH_CHAINED(bicg_xrp_kernel, x, p, s, t, v, r, reverse, red, bs);
    (void)launch_chained(chained_launches(st), bicg_finalize_kernel, 1, 1024, 0, st, (int)FIN_BI_R2, red, bicg_grid(precision, n), 0.0, bs);
    return cudaGetLastError();
}

cudaError_t launch_bicg_finalize(int fin, Reduction red, int n_partials, BiScalars* bs, cudaStream_t st) {
    count_launch();
    ProfScope prof(3, st);
    (void)launch_chained(chained_launches(st), bicg_finalize_kernel, 1, 1024, 0, st, fin, red, n_partials, 0.0, bs);
    return cudaGetLastError();
}

cudaError_t launch_bicg_p(int precision, size_t n, void* p, const void* r, const void* v, int reverse,
                          BiScalars* bs, cudaStream_t st) {
    count_launch();
    ProfScope prof(3, st);
    LQCD_BICG_DISPATCH(bicg_p_kernel, p, r, v, reverse, bs);
    return cudaGetLastError();
}

}  // namespace lqcd
