// force.cu -- the fermion force F = -dS/dU of the HMC (eq. 9-10; Table 2 row
// F_fermion; reading G16).
//
// For two spinor fields X, Y on the whole lattice and the link U_mu(x),
//   F^a_mu(x) = 2 kappa Im tr_colour [ T^a W ],   T^a = lambda^a / 2,
//   W = eta   sum_k (U h-_k[X(x+mu)]) (x) h-_k[Y(x)]^dag
//     - eta^* sum_k  h+_k[X(x)]       (x) (U h+_k[Y(x+mu)])^dag ,
// where h-+ are the half-spinor projections with (1 -+ gamma_mu) (site_ops.cuh: since
// (1 -+ gamma)^2 = 2 (1 -+ gamma), the four-row spin trace equals the two-row sum over k),
// eta the boundary phase of the hop (1 unless it wraps) and (u (x) v^dag)_cd = u_c conj(v_d).
// The paper's kernel moved 4736 B per site and direction with no reuse (4 spinors, link,
// force read + written); here one thread owns one link, the four warps of a CTA take the four
// directions of the same 32 sites so X(x), Y(x) are shared through L1, and neighbour reuse is
// left to L2 as in the hopping kernel.  Algorithmic bytes per site of V: 576 (links) + 2 x 192
// (X, Y once each) + 256 (force written) = 1216 in double/18.
#include "site_ops.cuh"

namespace lqcd {
namespace {

struct ForceArgs {
    const void* gauge;
    const void* x[2];   // X on even / odd sites (internal half-spinor layout)
    const void* y[2];
    double* force;      // double2 f[2][4][G][4][32]
    Geometry g;
    double kappa;
    double sx_odd, sy_odd;   // the odd halves handed in are sx_odd * X_o, sy_odd * Y_o (+-1)
};

// w[c][d] += (cr + i ci) * u_c conj(v_d), summed over the two half-spinor rows k
template <typename T>
__device__ __forceinline__ void outer_acc(T (&w)[18], const T (&u)[12], const T (&v)[12], T cr, T ci) {
#pragma unroll
    for (int k = 0; k < 2; ++k)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            // s = coefficient * u_c
            const T ur = u[2 * (3 * k + c)], ui = u[2 * (3 * k + c) + 1];
            const T sr = fma_(-ci, ui, cr * ur), si = fma_(ci, ur, cr * ui);
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                const T vr = v[2 * (3 * k + d)], vi = v[2 * (3 * k + d) + 1];
                w[2 * (3 * c + d)] = fma_(si, vi, fma_(sr, vr, w[2 * (3 * c + d)]));
                w[2 * (3 * c + d) + 1] = fma_(-sr, vi, fma_(si, vr, w[2 * (3 * c + d) + 1]));
            }
        }
}

template <typename T, int RECON, int MU>
__device__ __forceinline__ void force_link(const ForceArgs& a, int p, int e, int e_nb, bool wrap) {
    T u[18], psi[24], h[12], uh[12], v[12], w[18];
#pragma unroll
    for (int i = 0; i < 18; ++i) w[i] = 0;
    load_link<RECON>(a.gauge, a.g.G, p, MU, e, u);
    // boundary phase of this hop and the signs of the odd halves (file header)
    const T er = wrap ? (T)a.g.ph_re[MU] : (T)1, ei = wrap ? (T)a.g.ph_im[MU] : (T)0;
    const T s1 = (T)(p == 0 ? a.sx_odd : a.sy_odd);   // term 1 holds X(x+mu), Y(x)
    const T s2 = (T)(p == 0 ? a.sy_odd : a.sx_odd);   // term 2 holds X(x), Y(x+mu)

    load_spinor(a.x[1 - p], e_nb, psi);
    project<MU, -1>(psi, h);
    su3_mul(u, h, uh);
    load_spinor(a.y[p], e, psi);
    project<MU, -1>(psi, v);
    outer_acc(w, uh, v, s1 * er, s1 * ei);

    load_spinor(a.y[1 - p], e_nb, psi);
    project<MU, +1>(psi, h);
    su3_mul(u, h, uh);
    load_spinor(a.x[p], e, psi);
    project<MU, +1>(psi, v);
    outer_acc(w, v, uh, -s2 * er, s2 * ei);     // - conj(eta) X(x) (x) (U Y(x+mu))^dag

    // F^a = 2 kappa Im tr(T^a W), T^a = lambda^a / 2  (w[2(3c+d)] = Re W_cd)
    const double k = a.kappa;
    const double f1 = k * ((double)w[2 * 3 + 1] + (double)w[2 * 1 + 1]);            // Im(W10 + W01)
    const double f2 = k * ((double)w[2 * 1] - (double)w[2 * 3]);                    // Re(W01 - W10)
    const double f3 = k * ((double)w[1] - (double)w[2 * 4 + 1]);                    // Im(W00 - W11)
    const double f4 = k * ((double)w[2 * 6 + 1] + (double)w[2 * 2 + 1]);            // Im(W20 + W02)
    const double f5 = k * ((double)w[2 * 2] - (double)w[2 * 6]);                    // Re(W02 - W20)
    const double f6 = k * ((double)w[2 * 7 + 1] + (double)w[2 * 5 + 1]);            // Im(W21 + W12)
    const double f7 = k * ((double)w[2 * 5] - (double)w[2 * 7]);                    // Re(W12 - W21)
    const double f8 = k * 0.57735026918962576451 *
                      ((double)w[1] + (double)w[2 * 4 + 1] - 2.0 * (double)w[2 * 8 + 1]);  // Im(W00 + W11 - 2 W22)/sqrt 3
    double2* out = reinterpret_cast<double2*>(a.force) +
                   ((size_t)(p * 4 + MU) * a.g.G + (e >> 5)) * (4 * 32) + (e & 31);
    out[0] = make_double2(f1, f2);
    out[32] = make_double2(f3, f4);
    out[64] = make_double2(f5, f6);
    out[96] = make_double2(f7, f8);
}

// grid = 2 G blocks of 128 threads: block b works on the 32 sites of group b mod G of parity
// b / G; warp w takes direction mu = w.
template <typename T, int RECON>
__global__ void __launch_bounds__(128, 3) force_kernel(const ForceArgs a) {
    const int G = a.g.G;
    const int p = (int)blockIdx.x >= G ? 1 : 0;
    const int e = ((int)blockIdx.x - p * G) * 32 + (threadIdx.x & 31);
    const int mu = threadIdx.x >> 5;
    if (e >= a.g.Vh) {   // pad sites of the last group: zero force
        double2* out = reinterpret_cast<double2*>(a.force) + ((size_t)(p * 4 + mu) * G + (e >> 5)) * (4 * 32) + (e & 31);
#pragma unroll
        for (int j = 0; j < 4; ++j) out[32 * j] = make_double2(0.0, 0.0);
        return;
    }
    const int N0h = a.g.N0h, N1 = a.g.N1, N2 = a.g.N2, N3 = a.g.N3;
    int t = e;
    const int x0h = t % N0h; t /= N0h;
    const int x1 = t % N1;   t /= N1;
    const int x2 = t % N2;
    const int x3 = t / N2;
    const int r = (x1 + x2 + x3 + p) & 1;
    const int s1 = N0h, s2 = N0h * N1, s3 = N0h * N1 * N2;
    if (mu == 0) {
        const bool wf = (r == 1) && (x0h == N0h - 1);
        force_link<T, RECON, 0>(a, p, e, wf ? e - (N0h - 1) : e + r, wf);
    } else if (mu == 1) {
        const bool wf = (x1 == N1 - 1);
        force_link<T, RECON, 1>(a, p, e, wf ? e - (N1 - 1) * s1 : e + s1, wf);
    } else if (mu == 2) {
        const bool wf = (x2 == N2 - 1);
        force_link<T, RECON, 2>(a, p, e, wf ? e - (N2 - 1) * s2 : e + s2, wf);
    } else {
        const bool wf = (x3 == N3 - 1);
        force_link<T, RECON, 3>(a, p, e, wf ? e - (N3 - 1) * s3 : e + s3, wf);
    }
}

// internal double2 f[2][4][G][4][32] -> canonical double F[lex(x)][mu][8]
__global__ void __launch_bounds__(128) unpack_force_kernel(Geometry g, const double2* __restrict__ f,
                                                           double2* __restrict__ canon) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;   // (parity, e)
    if (i >= 2 * g.Vh) return;
    const int p = i / g.Vh, e = i - p * g.Vh;
    int t = e;
    const int x0h = t % g.N0h; t /= g.N0h;
    const int x1 = t % g.N1;   t /= g.N1;
    const int x2 = t % g.N2;
    const int x3 = t / g.N2;
    const int r = (x1 + x2 + x3 + p) & 1;
    const size_t lexi = (size_t)2 * e + r;   // x0 = 2 x0h + r
    (void)x0h;
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
        const double2* src = f + ((size_t)(p * 4 + mu) * g.G + (e >> 5)) * (4 * 32) + (e & 31);
#pragma unroll
        for (int j = 0; j < 4; ++j) canon[(lexi * 4 + mu) * 4 + j] = src[32 * j];
    }
}

}  // namespace

cudaError_t launch_fermion_force(int precision, int recon, const Geometry& g, const void* gauge,
                                 const void* x_even, const void* x_odd, const void* y_even,
                                 const void* y_odd, void* force, double kappa, double sx_odd, double sy_odd,
                                 cudaStream_t st) {
    ForceArgs a;
    a.gauge = gauge;
    a.x[0] = x_even; a.x[1] = x_odd; a.y[0] = y_even; a.y[1] = y_odd;
    a.force = (double*)force;
    a.g = g; a.kappa = kappa; a.sx_odd = sx_odd; a.sy_odd = sy_odd;
    count_launch();
    ProfScope prof(6, st);
    const int grid = 2 * g.G;
    if (precision == 0) {
        if (recon == 12) force_kernel<double, 12><<<grid, 128, 0, st>>>(a);
        else             force_kernel<double, 18><<<grid, 128, 0, st>>>(a);
    } else {
        if (recon == 12) force_kernel<float, 12><<<grid, 128, 0, st>>>(a);
        else             force_kernel<float, 18><<<grid, 128, 0, st>>>(a);
    }
    return cudaGetLastError();
}

cudaError_t launch_unpack_force(const Geometry& g, const void* force, void* canon, cudaStream_t st) {
    count_launch();
    ProfScope prof(4, st);
    unpack_force_kernel<<<(2 * g.Vh + 127) / 128, 128, 0, st>>>(g, (const double2*)force, (double2*)canon);
    return cudaGetLastError();
}

}  // namespace lqcd
