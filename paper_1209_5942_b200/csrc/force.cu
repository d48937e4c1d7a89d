// force.cu -- the fermion force F = -dS/dU of the HMC (eq. 9-10; Table 2 row
// F_fermion; reading G16).
//
// For two spinor fields X, Y on the whole lattice and the link U_mu(x),
//   F^a_mu(x) = 2 kappa Im tr_colour [ T^a W ],   T^a = lambda^a / 2,
//   W = sum_k (eta U h-_k[X(x+mu)]) (x) h-_k[Y(x)]^dag
//     - sum_k  h+_k[X(x)]           (x) (eta U h+_k[Y(x+mu)])^dag ,
// where h-+ are the half-spinor projections with (1 -+ gamma_mu) (site_ops.cuh: since
// (1 -+ gamma)^2 = 2 (1 -+ gamma), the four-row spin trace equals the two-row sum over k),
// eta the boundary phase of the hop (1 unless it wraps) and (u (x) v^dag)_cd = u_c conj(v_d).
// The paper's kernel moved 4736 B per site and direction with no reuse (4 spinors, link,
// force read + written); here one thread owns one link, the four warps of a CTA take the four
// directions of the same 32 sites so X(x), Y(x) are shared through L1, and neighbour reuse is
// left to L2 as in the hopping kernel.  Algorithmic bytes per site of V: 576 (links) + 2 x 192
// (X, Y once each) + 256 (force written) = 1216 in double/18.
#include "site_ops.cuh"

// CTAs of 128 threads per SM (per format: table below).  Round 1: the kernel is latency bound (ncu: DRAM traffic =
// algorithmic bytes, DRAM throughput 62%, 12 warps/SM): in double 4 CTAs (128 registers, no spills) run 460 us at
// 32^3 x 64 against 497 us with 3 (168 registers) and 497 us with 5 (96 registers, 140 B of spills).
// Tried and dropped: two threads per link (one per term of W, CTAs of 256, partial sums combined through
// shared memory; 80 registers, 24 warps/SM): 581 us -- the link is fetched twice and the local spinors
// lose their L1 sharing, which costs more than the extra warps hide.  X(x), Y(x) of the CTA's 32 sites staged
// once in shared memory instead of read through L1 by each direction-warp: 480 us (no change: the
// L2 -> L1 traffic it removes is not the limiter).  One thread per site looping over the four directions
// with the staged X(x), Y(x) (64-thread CTAs, 168 registers): 513 us; at 128 registers 707 us.
//
// Round 2 (us per launch at 32^3 x 64 in the sweep's power-capped loop, A B A B on one box; d18 / d12 / s18 / s12):
//   as above, 4 CTAs                                     505-510 / 422-443 / 270-280 / 258-267
//   loads first (LF below) at 3 / 4 / 6 / 8 CTAs          487-489 / 420     / 263-270 / 235     <- used, except d12
//   (the build as committed, another box: 472 / 433 / 262 / 237 = 0.83 / 0.76 / 0.90 / 0.87 of the measured copy bandwidth)
//   loads first at 4 / 3 / 5 / 6 CTAs                     531     / 448-452 / 276     / 242
// ptxas issues the link and X(x+mu) up front (21 LDG.128) and the second neighbour spinor only when registers free up, so a
// thread waits on DRAM twice; LF names all three DRAM-latency reads before any arithmetic (33 LDG.128 up front, 168
// registers in double/18).  Tried on top of both and dropped:
// * a grid that fills the GPU once, every CTA walking the blocks b, b + gridDim.x, ... with no barrier between its warps
//   (ncu: 12.8 of 16 resident warps active, the rest is CTA turnover): 576 us at 4 CTAs per SM, 530 at 8, 553 at 16 (d18);
// * cp.async.bulk.prefetch.L2 of the link group and the two neighbour groups of the block 296 ... 9472 blocks ahead (five
//   instructions per warp): 549 / 531 / 600 / 774 / 757 us (d18) -- the prefetched lines compete with the demand loads.
// * the two combined as a software pipeline: persistent CTAs, the next block's link and neighbour spinors fetched with
//   cp.async into a per-thread slot of shared memory (33 x 16 B per thread, 68 KB per CTA) while the current block is
//   worked on from registers: 704 us at 3 CTAs per SM, 586 at 2 (d18), 575 / 521 (d12), results identical.  Every form
//   that runs the memory requests further ahead of the arithmetic is slower: what the short-lived CTAs give the kernel is
//   a spread over the phases of a link's life, and with it an even load on the memory system.
constexpr int kForceMinBlocks = 4;       // double/12
constexpr int kForceMinBlocksD18 = 3;    // loads first: 168 registers
constexpr int kForceMinBlocksF18 = 6;    // loads first: 80 registers
constexpr int kForceMinBlocksF12 = 8;    // loads first: 64 registers

namespace lqcd {
namespace {

struct ForceArgs {
    const void* gauge;
    const void* x[2];   // X on even / odd sites (internal half-spinor layout)
    const void* y[2];
    double* force;      // double2 f[2][4][G][4][32]
    Geometry g;
    double kappa;       // kappa times the common sign of the odd halves handed in (lqcd_force_tm)
};

// Only the traceless anti-Hermitian part of W enters Im tr(T^a W); with W = sum u (x) v^dag it is
// spanned by nine real numbers,
//   s[cd] = Im(W_cd + W_dc), r[cd] = Re(W_cd - W_dc) for cd = 01, 02, 12, and d[c] = Im W_cc,
// accumulated here over the two half-spinor rows k: 30 FMA per row instead of the 36 of the full
// 3 x 3 complex outer product, and 9 accumulators instead of 18.
template <typename T>
struct AntiHerm { T s[3], r[3], d[3]; };

template <typename T>
__device__ __forceinline__ void outer_acc(AntiHerm<T>& w, const T (&u)[12], const T (&v)[12]) {
#pragma unroll
    for (int k = 0; k < 2; ++k) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const T ur = u[2 * (3 * k + c)], ui = u[2 * (3 * k + c) + 1];
            const T vr = v[2 * (3 * k + c)], vi = v[2 * (3 * k + c) + 1];
            w.d[c] = fma_(-ur, vi, fma_(ui, vr, w.d[c]));            // Im(u_c conj v_c)
        }
#pragma unroll
        for (int q = 0; q < 3; ++q) {
            const int c = (q == 2) ? 1 : 0, d = (q == 0) ? 1 : 2;
            const T ucr = u[2 * (3 * k + c)], uci = u[2 * (3 * k + c) + 1];
            const T udr = u[2 * (3 * k + d)], udi = u[2 * (3 * k + d) + 1];
            const T vcr = v[2 * (3 * k + c)], vci = v[2 * (3 * k + c) + 1];
            const T vdr = v[2 * (3 * k + d)], vdi = v[2 * (3 * k + d) + 1];
            // Im(u_c conj v_d) + Im(u_d conj v_c)
            w.s[q] = fma_(-udr, vci, fma_(udi, vcr, fma_(-ucr, vdi, fma_(uci, vdr, w.s[q]))));
            // Re(u_c conj v_d) - Re(u_d conj v_c)
            w.r[q] = fma_(-udi, vci, fma_(-udr, vcr, fma_(uci, vdi, fma_(ucr, vdr, w.r[q]))));
        }
    }
}

template <typename T>
__device__ __forceinline__ void phase_mul(T (&chi)[12], T pr, T pi) {
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        const T re = chi[2 * i], im = chi[2 * i + 1];
        chi[2 * i] = fma_(-pi, im, pr * re);
        chi[2 * i + 1] = fma_(pi, re, pr * im);
    }
}

// The second term of W is -h+[X(x)] (x) (eta U h+[Y(x+mu)])^dag; its anti-Hermitian part equals
// that of +(eta U h+[Y(x+mu)]) (x) h+[X(x)]^dag, so both terms go through the same accumulation
// with the transported half spinor first.
// REALPH (every boundary phase +-1, Geometry::real_ph): both terms carry the same real eta, so it multiplies the link's
// whole W and is applied once, with kappa, when the force is stored -- no branch, no phase multiplication.
// LF ("loads first"): the link and BOTH neighbour spinors -- the three DRAM-latency reads of the thread -- are named before
// any arithmetic, so they are in flight together; the local spinors, shared through L1 by the four direction-warps, follow.
template <typename T, int RECON, int MU, bool REALPH, bool LF>
__device__ __forceinline__ void force_link(const ForceArgs& a, int p, int e, int e_nb, bool wrap) {
    AntiHerm<T> w;
#pragma unroll
    for (int i = 0; i < 3; ++i) w.s[i] = w.r[i] = w.d[i] = 0;
    const T er = (T)a.g.ph_re[MU], ei = (T)a.g.ph_im[MU];   // boundary phase, used on the wrapping hop only
    if (LF) {
        T u[18], xn[24], yn[24], h[12], uh1[12], uh2[12], v[12];
        load_link<RECON>(a.gauge, a.g.G, p, MU, e, u);
        load_spinor(a.x[1 - p], e_nb, xn);
        load_spinor(a.y[1 - p], e_nb, yn);
        project<MU, -1>(xn, h);
        su3_mul(u, h, uh1);
        project<MU, +1>(yn, h);
        su3_mul(u, h, uh2);
        if (!REALPH && wrap) {
            phase_mul(uh1, er, ei);
            phase_mul(uh2, er, ei);
        }
        load_spinor(a.y[p], e, xn);
        project<MU, -1>(xn, v);
        outer_acc(w, uh1, v);
        load_spinor(a.x[p], e, yn);
        project<MU, +1>(yn, v);
        outer_acc(w, uh2, v);
    } else {
        T u[18], psi[24], h[12], uh[12], v[12];
        load_link<RECON>(a.gauge, a.g.G, p, MU, e, u);

        load_spinor(a.x[1 - p], e_nb, psi);
        project<MU, -1>(psi, h);
        su3_mul(u, h, uh);
        if (!REALPH && wrap) phase_mul(uh, er, ei);
        load_spinor(a.y[p], e, psi);
        project<MU, -1>(psi, v);
        outer_acc(w, uh, v);

        load_spinor(a.y[1 - p], e_nb, psi);
        project<MU, +1>(psi, h);
        su3_mul(u, h, uh);
        if (!REALPH && wrap) phase_mul(uh, er, ei);
        load_spinor(a.x[p], e, psi);
        project<MU, +1>(psi, v);
        outer_acc(w, uh, v);
    }

    // F^a = 2 kappa Im tr(T^a W) = kappa Im tr(lambda^a W)
    const double k = (REALPH && wrap) ? a.kappa * a.g.ph_re[MU] : a.kappa;
    double2* out = reinterpret_cast<double2*>(a.force) +
                   ((size_t)(p * 4 + MU) * a.g.G + (e >> 5)) * (4 * 32) + (e & 31);
    out[0] = make_double2(k * (double)w.s[0], k * (double)w.r[0]);                          // lambda 1, 2
    out[32] = make_double2(k * ((double)w.d[0] - (double)w.d[1]), k * (double)w.s[1]);      // lambda 3, 4
    out[64] = make_double2(k * (double)w.r[1], k * (double)w.s[2]);                         // lambda 5, 6
    out[96] = make_double2(k * (double)w.r[2],                                              // lambda 7, 8
                           k * 0.57735026918962576451 * ((double)w.d[0] + (double)w.d[1] - 2.0 * (double)w.d[2]));
}

// grid = 2 G blocks of 128 threads: block b works on the 32 sites of group b / 2 of parity
// b mod 2; warp w takes direction mu = w.  The two parities are interleaved because every spinor
// site is read twice, as X(x) by its own block and as X(x+mu) by blocks of the other parity:
// sweeping one parity after the other put a whole field (805 MB of X, Y) between the two reads
// and cost a second DRAM pass (ncu: 3.35 GB of traffic against 2.55 GB algorithmic).
template <typename T, int RECON, bool REALPH, bool LF, int NB>
__global__ void __launch_bounds__(128, NB) force_kernel(const ForceArgs a) {
    const int G = a.g.G;
    const int p = (int)blockIdx.x & 1;
    const int e = ((int)blockIdx.x >> 1) * 32 + (threadIdx.x & 31);
    const int mu = threadIdx.x >> 5;
    if (e >= a.g.Vh) {   // pad sites of the last group: zero force
        double2* out = reinterpret_cast<double2*>(a.force) + ((size_t)(p * 4 + mu) * G + (e >> 5)) * (4 * 32) + (e & 31);
#pragma unroll
        for (int j = 0; j < 4; ++j) out[32 * j] = make_double2(0.0, 0.0);
        return;
    }
    const int N0h = a.g.N0h, N1 = a.g.N1, N2 = a.g.N2, N3 = a.g.N3;
    int x0h, x1, x2, x3;
    site_coords(a.g, e, x0h, x1, x2, x3);
    const int r = (x1 + x2 + x3 + p) & 1;
    const int s1 = N0h, s2 = N0h * N1, s3 = N0h * N1 * N2;
    if (mu == 0) {
        const bool wf = (r == 1) && (x0h == N0h - 1);
        force_link<T, RECON, 0, REALPH, LF>(a, p, e, wf ? e - (N0h - 1) : e + r, wf);
    } else if (mu == 1) {
        const bool wf = (x1 == N1 - 1);
        force_link<T, RECON, 1, REALPH, LF>(a, p, e, wf ? e - (N1 - 1) * s1 : e + s1, wf);
    } else if (mu == 2) {
        const bool wf = (x2 == N2 - 1);
        force_link<T, RECON, 2, REALPH, LF>(a, p, e, wf ? e - (N2 - 1) * s2 : e + s2, wf);
    } else {
        const bool wf = (x3 == N3 - 1);
        force_link<T, RECON, 3, REALPH, LF>(a, p, e, wf ? e - (N3 - 1) * s3 : e + s3, wf);
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
                                 const void* y_odd, void* force, double kappa, cudaStream_t st) {
    ForceArgs a;
    a.gauge = gauge;
    a.x[0] = x_even; a.x[1] = x_odd; a.y[0] = y_even; a.y[1] = y_odd;
    a.force = (double*)force;
    a.g = g; a.kappa = kappa;
    count_launch();
    ProfScope prof(6, st);
    const int grid = 2 * g.G;
    // The order of the loads and the CTAs per SM are per format (table at the top of the file).  The branch-free form of the
    // boundary phase is what ptxas schedules better in double/12 (438 against 482 us) and makes no difference elsewhere.
    const bool rp = g.real_ph;
#define LQCD_FORCE(TT, RR, LFV, NBV)                                                   \
    do {                                                                               \
        if (rp) force_kernel<TT, RR, true, LFV, NBV><<<grid, 128, 0, st>>>(a);         \
        else    force_kernel<TT, RR, false, LFV, NBV><<<grid, 128, 0, st>>>(a);        \
    } while (0)
    if (precision == 0) {
        if (recon == 12) LQCD_FORCE(double, 12, false, kForceMinBlocks);
        else             LQCD_FORCE(double, 18, true, kForceMinBlocksD18);
    } else {
        if (recon == 12) LQCD_FORCE(float, 12, true, kForceMinBlocksF12);
        else             LQCD_FORCE(float, 18, true, kForceMinBlocksF18);
    }
#undef LQCD_FORCE
    return cudaGetLastError();
}

cudaError_t launch_unpack_force(const Geometry& g, const void* force, void* canon, cudaStream_t st) {
    count_launch();
    ProfScope prof(4, st);
    unpack_force_kernel<<<(2 * g.Vh + 127) / 128, 128, 0, st>>>(g, (const double2*)force, (double2*)canon);
    return cudaGetLastError();
}

}  // namespace lqcd
