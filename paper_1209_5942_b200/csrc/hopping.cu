// hopping.cu -- the hopping term D_eo / D_oe of eq. 6 with fused
// diagonal-term epilogues, hand-written for sm_100a.
//
// One thread per output site.  Per site:
//   a1 site -> coordinates -> 8 neighbour indices and wrap flags (integer only)
//   a2 4 forward links U_mu(x) (own-parity array, own index: coalesced) and
//      4 backward links U_mu(x-mu) (other-parity array, neighbour's index);
//      every link of the lattice is read exactly once per application, so the
//      gauge loads are streamed (ld.global.cs: evict-first, no reuse expected)
//   a3 neighbour spinor -> spin projection to a half spinor (12 -> 6 complex);
//      neighbour spinors are reused by 8 output sites, so they go through the
//      read-only path with default caching (L1 for x/y neighbours, L2 for z/t)
//   a4 SU(3) x half spinor (U h forward, U^dag h backward)
//   a5 boundary phase on the hop that wraps, reconstruction to 4 spin rows, accumulate; where every phase is +-1
//      (REALPH) the phase is the sign s of acc = fma(s, chi, acc) and the thread has no branch at all
//   a6/a7 epilogue: out = c_chi * (acc + d_chi * aux), c, d complex per chirality:
//      covers -kappa (dslash_eo), M_oo^{-1} D_oe, and M_ee in - D_eo (.) in one store.
//   a9 (MODE 3) the last hopping launch of a CG iteration never stores q = A p: it
//      applies r -= alpha q in place and reduces |r|^2 (alpha = rho / pAp read from the
//      device scalars), which saves one field store, one field load and a launch.
//   BiCGStab (MODE 4, 5): a MODE 1 launch that also reduces |out|^2 and <w, out> (complex) for one or
//      two more fields w (rhat for sigma = <rhat, v>; s and rhat for <s, t>, |t|^2, <rhat, t>).  w(x) is brought
//      into shared memory by cp.async at the start of the thread (LDGSTS: no registers, in flight
//      with the first hop's loads) and read back in the epilogue, so the inner products cost one
//      field read instead of a vector kernel of their own (two field reads and a launch).
//
// Spin projection table (gamma basis of include/lqcd.h; reading G4),
// (1 + S gamma_mu) psi = (h0, h1, conj(c0) h0 or h1 ...):
//   h0 = psi_0 + c0 psi_j0,  h1 = psi_1 + c1 psi_j1,  j1 = 5 - j0,
//   row j0 of the result = conj(c0) h0, row j1 = conj(c1) h1.
//   S = -1:  mu=x: j0=3 c0=+i c1=+i | y: j0=3 c0=+1 c1=-1 | z: j0=2 c0=+i c1=-i | t: j0=2 c0=-1 c1=-1
//   S = +1:  all c negated.
// Forward hops of the operator use S = -1, backward hops S = +1; the adjoint
// stencil (DAG) swaps them.
#include "site_ops.cuh"

// CTAs of 128 threads per SM the register allocation aims at.  3 (168 registers) is best for
// double and for single/18 (measured: 2 and 4 are ~20% slower in double; 4, 5, 6 are 4-15% slower
// for single/18).  Single/12 moves the fewest DRAM bytes per thread and direction (60 B), so at
// 12 warps/SM it cannot keep enough requests in flight: 7 CTAs (72 registers) is 27% faster.
// Re-measured with the grouped layout (32^3 x 64, us per launch at 3 / 4 CTAs of 128, 8 CTAs of 64):
// double/18 252 / 288 / 287, double/12 213.5 / 207.5 / 208, single/18 123.7 / 122.2 / 120.5; at
// 16^3 x 32 (1.15 waves at 3 CTAs) the 128-register builds are 6% faster (17.5 vs 18.6 us), not
// enough to carry a second set of instantiations.  Only double/12 moves to 4 CTAs.
// single/12 re-measured at 5 / 6 / 7 / 8 CTAs (96 / 80 / 72 / 64 registers): 102.9 / 102.3 / 102.4 / 108.1 us per launch,
// CG iteration 574 / 562 / 561 / 602 us: flat between 6 and 7, 7 stays.
// double/12 is the one format the register file binds (acc 48 + link 36 + spinor 48 registers leave no room at 128 to
// fetch the next hop early, and the register file being per sub-partition there is no budget between 128 and 168: 96-,
// 64- and 160-thread CTAs with 5 / 7 / 3 per SM all compile to 128).  Tried in round 2: the lower half of the accumulator
// (spin 2, 3: 12 of the 24 reals) kept in shared memory, 6 LDS.128 + 6 STS.128 per hop, to free 24 registers: 226.9-228.4
// us at 4 CTAs, 222.3 at 3, 248.4 at 5 against 218.2 on the same box (results identical) -- not kept.
constexpr int kHopMinBlocks = 3;       // double/18, single/18
constexpr int kHopMinBlocksD12 = 4;    // double/12
constexpr int kHopMinBlocksF12 = 7;    // single/12

namespace lqcd {
namespace {


template <typename T, int RECON, int MU, int FWD, int DAG, bool SLAB, bool REALPH = false>
__device__ __forceinline__ void hop(T (&acc)[24], const HopArgs& a, int e, int e_nb, bool wrap) {
    constexpr int S = (FWD ? -1 : +1) * (DAG ? -1 : +1);
    T psi[24], u[18], h[12], chi[12];
    load_spinor(a.in, e_nb, psi);
    load_link<RECON>(a.gauge, SLAB ? a.g.Gg : a.g.G, FWD ? a.out_parity : 1 - a.out_parity, MU, FWD ? e : e_nb, u);
    project<MU, S>(psi, h);
    if (FWD) su3_mul(u, h, chi);
    else     su3_dag_mul(u, h, chi);
    if (REALPH) {   // phases +-1: the sign rides on the accumulation, no branch
        accumulate_scaled<MU, S>(acc, chi, wrap ? (T)a.g.ph_re[MU] : (T)1);
        return;
    }
    if (wrap) {  // boundary phase on the hop that wraps (forward: phase, backward: conj)
        const T pr = (T)a.g.ph_re[MU], pi = FWD ? (T)a.g.ph_im[MU] : -(T)a.g.ph_im[MU];
#pragma unroll
        for (int i = 0; i < 6; ++i) {
            const T re = chi[2 * i], im = chi[2 * i + 1];
            chi[2 * i] = fma_(-pi, im, pr * re);
            chi[2 * i + 1] = fma_(pi, re, pr * im);
        }
    }
    accumulate<MU, S>(acc, chi);
}

template <typename T, int RECON, int DAG, int MODE, bool SLAB, bool TILE = false, bool REALPH = false>
__global__ void __launch_bounds__(LQCD_HOP_MAX_THREADS, (RECON == 12) ? (sizeof(T) == 4 ? kHopMinBlocksF12 : kHopMinBlocksD12)
                                                                      : kHopMinBlocks)
hopping_kernel(const HopArgs a) {
    chain_prologue();
    if (a.scal != nullptr && a.scal->done) return;
    const int Vh = a.g.Vh;
    const int blk = a.reverse ? (int)(gridDim.x - 1 - blockIdx.x) : (int)blockIdx.x;
    // single lattice: site e of all Vh; slab mode: site i of the launch's SiteRange
    int i = blk * blockDim.x + threadIdx.x;
    if (TILE) {   // blk = tile (gy, z / 2, t / 2); warp w of the CTA: z = 2 (z / 2) + (w & 1), t = 2 (t / 2) + (w >> 1)
        const int w = threadIdx.x >> 5;
        const int q = blk / a.tile_gy, gy = blk - q * a.tile_gy;
        const int tt = q / a.tile_n2h, zt = q - tt * a.tile_n2h;
        i = 32 * (gy + a.tile_gy * ((2 * zt + (w & 1)) + a.g.N2 * (2 * tt + (w >> 1)))) + (threadIdx.x & 31);
    }
    const bool live = SLAB ? (i < a.rg.count) : (i < Vh);
    const int e = SLAB ? a.rg.base + i + (i >= a.rg.n1 ? a.rg.skip : 0) : i;
    double nrm = 0.0;
    // MODE 3: alpha = rho / <p, A p> and its inverse were left in the device scalars by
    // finalize(FIN_PAP), which also ends the solve (done = 1, caught above) on a breakdown.
    const double alpha = (MODE == 3) ? a.scal->alpha : 1.0;
    // MODE 4, 5: w(x) (and w2(x)) parked in shared memory, [field][component][thread], 16-byte elements
    constexpr int WCOMP = (sizeof(T) == 8) ? 12 : 6;
    constexpr int NW = (MODE == 5) ? 2 : (MODE == 4) ? 1 : 0;
    __shared__ __align__(16) unsigned char wsm_raw[NW > 0 ? NW * WCOMP * LQCD_HOP_MAX_THREADS * 16 : 16];
    double dre[NW > 0 ? NW : 1] = {}, dim_[NW > 0 ? NW : 1] = {};
    if (live) {
        if (NW > 0) {
#pragma unroll
            for (int f = 0; f < NW; ++f) {
                const char* src = reinterpret_cast<const char*>(f ? a.dotw2 : a.dotw) + ((size_t)(e >> 5) * (WCOMP * 32) + (e & 31)) * 16;
                const unsigned dst = (unsigned)__cvta_generic_to_shared(wsm_raw) + (f * WCOMP * LQCD_HOP_MAX_THREADS + threadIdx.x) * 16;
#pragma unroll
                for (int c = 0; c < WCOMP; ++c)
                    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;\n" ::"r"(dst + c * (LQCD_HOP_MAX_THREADS * 16)),
                                 "l"(src + c * 512) : "memory");
            }
            asm volatile("cp.async.commit_group;\n" ::: "memory");
        }
        // a1: e -> (x0h, x1, x2, x3); r = x0 mod 2 follows from the parity
        const int N0h = a.g.N0h, N1 = a.g.N1, N2 = a.g.N2, N3 = a.g.N3;
        int x0h, x1, x2, x3;
        site_coords(a.g, e, x0h, x1, x2, x3);
        const int r = (x1 + x2 + x3 + a.out_parity) & 1;
        const int s1 = N0h, s2 = N0h * N1, s3 = N0h * N1 * N2;

        // The accumulator starts at d_chi * aux(x) (MODE >= 1), so the M_ee * aux term of the
        // epilogue costs no registers and its loads are the first in flight instead of a
        // serialised DRAM round trip after the last hop: out = c_chi * (d_chi aux + bracket).
        T acc[24];
        if (MODE >= 1) {
            T x[24];
            load_spinor(a.aux, e, x);
            const T dur = (T)a.ep.du_re, dui = (T)a.ep.du_im, ddr = (T)a.ep.dd_re, ddi = (T)a.ep.dd_im;
#pragma unroll
            for (int c = 0; c < 12; ++c) {
                const T dr = (c < 6) ? dur : ddr, di = (c < 6) ? dui : ddi;
                acc[2 * c] = fma_(-di, x[2 * c + 1], dr * x[2 * c]);
                acc[2 * c + 1] = fma_(di, x[2 * c], dr * x[2 * c + 1]);
            }
            if (MODE == 3) {
                // r - alpha c (bracket + d aux) = (-alpha c) (bracket + d aux - r / (alpha c)):
                // the old residual joins the accumulator's initial value with s = -(1/alpha)(1/c),
                // 1/c = ep.s* prepared on the host
                load_spinor_rw(a.out, e, x);
                const double ia = -a.scal->inv_alpha;
                const T sur = (T)(ia * a.ep.su_re), sui = (T)(ia * a.ep.su_im);
                const T sdr = (T)(ia * a.ep.sd_re), sdi = (T)(ia * a.ep.sd_im);
#pragma unroll
                for (int c = 0; c < 12; ++c) {
                    const T sr = (c < 6) ? sur : sdr, si = (c < 6) ? sui : sdi;
                    acc[2 * c] = fma_(-si, x[2 * c + 1], fma_(sr, x[2 * c], acc[2 * c]));
                    acc[2 * c + 1] = fma_(si, x[2 * c], fma_(sr, x[2 * c + 1], acc[2 * c + 1]));
                }
            }
        } else {
#pragma unroll
            for (int i = 0; i < 24; ++i) acc[i] = 0;
        }

        {   // mu = 0: neighbour x0h' = x0h + r (forward), x0h + r - 1 (backward)
            const bool wf = (r == 1) && (x0h == N0h - 1);
            const bool wb = (r == 0) && (x0h == 0);
            hop<T, RECON, 0, 1, DAG, SLAB, REALPH>(acc, a, e, wf ? e - (N0h - 1) : e + r, wf);
            hop<T, RECON, 0, 0, DAG, SLAB, REALPH>(acc, a, e, wb ? e + (N0h - 1) : e + r - 1, wb);
        }
        {
            const bool wf = (x1 == N1 - 1), wb = (x1 == 0);
            hop<T, RECON, 1, 1, DAG, SLAB, REALPH>(acc, a, e, wf ? e - (N1 - 1) * s1 : e + s1, wf);
            hop<T, RECON, 1, 0, DAG, SLAB, REALPH>(acc, a, e, wb ? e + (N1 - 1) * s1 : e - s1, wb);
        }
        {
            const bool wf = (x2 == N2 - 1), wb = (x2 == 0);
            hop<T, RECON, 2, 1, DAG, SLAB, REALPH>(acc, a, e, wf ? e - (N2 - 1) * s2 : e + s2, wf);
            hop<T, RECON, 2, 0, DAG, SLAB, REALPH>(acc, a, e, wb ? e + (N2 - 1) * s2 : e - s2, wb);
        }
        {
            const bool wf = (x3 == N3 - 1), wb = (x3 == 0);
            if (SLAB) {   // across the rank's t boundary: the ghost slices (lqcd_internal.h Geometry)
                // forward ghost at Vh + s = e + s3 (no select needed); backward ghost at Vh + s3 + s = e + (N3 + 1) s3
                hop<T, RECON, 3, 1, DAG, SLAB, REALPH>(acc, a, e, e + s3, wf && a.g.tph_f);
                hop<T, RECON, 3, 0, DAG, SLAB, REALPH>(acc, a, e, wb ? e + (N3 + 1) * s3 : e - s3, wb && a.g.tph_b);
            } else {      // the periodic wrap (one shared constant (N3 - 1) s3: a second one costs 70 B of spills)
                hop<T, RECON, 3, 1, DAG, SLAB, REALPH>(acc, a, e, wf ? e - (N3 - 1) * s3 : e + s3, wf);
                hop<T, RECON, 3, 0, DAG, SLAB, REALPH>(acc, a, e, wb ? e + (N3 - 1) * s3 : e - s3, wb);
            }
        }

        // a6/a7: epilogue, complex coefficient per chirality
        T o[24];
        const double esc = (MODE == 3) ? -alpha : 1.0;
        const T cur = (T)(esc * a.ep.cu_re), cui = (T)(esc * a.ep.cu_im);
        const T cdr = (T)(esc * a.ep.cd_re), cdi = (T)(esc * a.ep.cd_im);
#pragma unroll
        for (int c = 0; c < 12; ++c) {
            const T cr = (c < 6) ? cur : cdr, ci = (c < 6) ? cui : cdi;
            o[2 * c] = fma_(-ci, acc[2 * c + 1], cr * acc[2 * c]);
            o[2 * c + 1] = fma_(ci, acc[2 * c], cr * acc[2 * c + 1]);
        }
        store_spinor(a.out, e, o);
        if (NW > 0) {  // <w, out> = sum conj(w) out, in double whatever T is
            asm volatile("cp.async.wait_all;\n" ::: "memory");
#pragma unroll
            for (int f = 0; f < NW; ++f) {
                if (sizeof(T) == 8) {
                    const double2* w = reinterpret_cast<const double2*>(wsm_raw) + f * WCOMP * LQCD_HOP_MAX_THREADS + threadIdx.x;
#pragma unroll
                    for (int c = 0; c < 12; ++c) {
                        const double2 v = w[c * LQCD_HOP_MAX_THREADS];
                        dre[f] = fma(v.x, (double)o[2 * c], fma(v.y, (double)o[2 * c + 1], dre[f]));
                        dim_[f] = fma(v.x, (double)o[2 * c + 1], fma(-v.y, (double)o[2 * c], dim_[f]));
                    }
                } else {
                    const float4* w = reinterpret_cast<const float4*>(wsm_raw) + f * WCOMP * LQCD_HOP_MAX_THREADS + threadIdx.x;
#pragma unroll
                    for (int k = 0; k < 6; ++k) {
                        const float4 v = w[k * LQCD_HOP_MAX_THREADS];
                        dre[f] += (double)v.x * (double)o[4 * k] + (double)v.y * (double)o[4 * k + 1] +
                                  (double)v.z * (double)o[4 * k + 2] + (double)v.w * (double)o[4 * k + 3];
                        dim_[f] += (double)v.x * (double)o[4 * k + 1] - (double)v.y * (double)o[4 * k] +
                                   (double)v.z * (double)o[4 * k + 3] - (double)v.w * (double)o[4 * k + 2];
                    }
                }
            }
        }
        if (MODE >= 2) {  // |out|^2 = |c_u|^2 |acc_upper|^2 + |c_d|^2 |acc_lower|^2
            double nu = 0.0, nd = 0.0;
#pragma unroll
            for (int i = 0; i < 12; ++i) {
                nu += (double)acc[i] * (double)acc[i];
                nd += (double)acc[12 + i] * (double)acc[12 + i];
            }
            nrm = (esc * esc) * ((a.ep.cu_re * a.ep.cu_re + a.ep.cu_im * a.ep.cu_im) * nu +
                                 (a.ep.cd_re * a.ep.cd_re + a.ep.cd_im * a.ep.cd_im) * nd);
        }
    }
    // pad sites of the last group hold zeros.  Slab mode has no pad sites (Vh is a multiple of 32) and
    // the condition below is never true there (n1 >= 0), but the branch stays: without it ptxas ends
    // the non-live threads with an early EXIT and schedules the whole kernel differently -- same
    // instruction count, 309 instead of 246 us per launch at 32^3 x 64 (measured).
    if (!live && (SLAB ? (a.rg.n1 < 0) : (e < a.g.G * 32))) {
        T z[24];
#pragma unroll
        for (int i = 0; i < 24; ++i) z[i] = 0;
        store_spinor(a.out, e, z);
    }
    if (MODE >= 2) {  // one partial per warp, plain store; summed by launch_finalize(FIN_PAP / FIN_RHO)
        nrm = warp_sum(nrm);
        if ((threadIdx.x & 31) == 0 && (!SLAB || live) && (NW == 0 || (e >> 5) < a.g.G)) a.red.partials[e >> 5] = nrm;
    }
    if (NW > 0) {  // partial set k of warp g at partials[k G + g]: k = 0 (above) |out|^2, then Re, Im <w, out> (, Re, Im <w2, out>)
#pragma unroll
        for (int f = 0; f < NW; ++f) {
            const double sr = warp_sum(dre[f]), si = warp_sum(dim_[f]);
            if ((threadIdx.x & 31) == 0 && (e >> 5) < a.g.G) {   // warps past the last group hold no partial
                a.red.partials[(size_t)(2 * f + 1) * a.g.G + (e >> 5)] = sr;
                a.red.partials[(size_t)(2 * f + 2) * a.g.G + (e >> 5)] = si;
            }
        }
    }
}

template <typename T, int RECON>
cudaError_t launch_tr(int dagger, int mode, const HopArgs& a, int block, cudaStream_t st) {
    const int grid = (a.rg.count + block - 1) / block;
    // REALPH: every boundary phase is +-1 (Geometry::real_ph), the sign rides on the accumulation and the kernel has no
    // branch per hop -- 4% faster at 32^3 x 64 in every format, bit-identical (profiles/r02_hopping_staged.md)
    const bool rp = a.g.real_ph && !a.general_phases;
    const bool ch = chained_launches(st);
#define LQCD_HOP_LAUNCH(D, M, SL, TL)                                                                                       \
    return rp ? launch_chained(ch, hopping_kernel<T, RECON, D, M, SL, TL, true>, grid, block, 0, st, a)                     \
              : launch_chained(ch, hopping_kernel<T, RECON, D, M, SL, TL, false>, grid, block, 0, st, a)
#define LQCD_HOP_CASE(D, M)                                                        \
    if (dagger == D && mode == M) {                                                \
        if (a.g.slab)           { LQCD_HOP_LAUNCH(D, M, true, false); }            \
        else if (a.tile_gy > 0) { LQCD_HOP_LAUNCH(D, M, false, true); }            \
        else                    { LQCD_HOP_LAUNCH(D, M, false, false); }           \
    }
    LQCD_HOP_CASE(0, 0) LQCD_HOP_CASE(0, 1) LQCD_HOP_CASE(0, 2)
    LQCD_HOP_CASE(1, 0) LQCD_HOP_CASE(1, 1) LQCD_HOP_CASE(1, 2) LQCD_HOP_CASE(1, 3)
#undef LQCD_HOP_CASE
    if (dagger == 0 && (mode == 4 || mode == 5) && !a.g.slab) {   // BiCGStab's fused inner products (single lattice only)
        if (mode == 4) { LQCD_HOP_LAUNCH(0, 4, false, false); }
        LQCD_HOP_LAUNCH(0, 5, false, false);
    }
#undef LQCD_HOP_LAUNCH
    return cudaErrorInvalidValue;
}

}  // namespace

// This file is compiled twice so that its two halves build in parallel (the kernel's instantiations are most of the
// library's compile time): as hopping.cu, with the double-precision kernels and the dispatcher, and through
// hopping_float.cu (LQCD_HOP_FLOAT_PART), with the single-precision kernels behind launch_hopping_float.  HopArgs lives in
// an unnamed namespace, so it crosses between the two as an untyped pointer to the same layout.
cudaError_t launch_hopping_float(int recon, int dagger, int mode, const void* hop_args, int block, cudaStream_t st);
#ifdef LQCD_HOP_FLOAT_PART
cudaError_t launch_hopping_float(int recon, int dagger, int mode, const void* hop_args, int block, cudaStream_t st) {
    const HopArgs& a = *static_cast<const HopArgs*>(hop_args);
    return recon == 12 ? launch_tr<float, 12>(dagger, mode, a, block, st)
                       : launch_tr<float, 18>(dagger, mode, a, block, st);
}
#else

// which kernel launch_hopping uses where a staged variant covers the launch (hopping_staged.cu); 0 = the plain kernel
static int g_hop_variant = 0;
void set_hopping_variant(int variant) { g_hop_variant = variant; }
int hopping_variant() { return g_hop_variant; }

// one partial per warp of live sites, indexed by e >> 5 whatever the launch's SiteRange and block size
int hopping_partials(int Vh, int block) {
    (void)block;
    return (Vh + 31) / 32;
}

cudaError_t launch_hopping(int precision, int recon, int dagger, int mode, const Geometry& g,
                           const Epilogue& ep, const void* gauge, const void* in, void* out,
                           const void* aux, int out_parity, int reverse, Reduction red,
                           CgScalars* scal, int block, cudaStream_t st, const SiteRange* range,
                           const void* dotw, const void* dotw2) {
    if (g_hop_variant >= 1 && g_hop_variant <= 5 && hopping_variant_covers(g_hop_variant, mode, g, range))
        return launch_hopping_variant(g_hop_variant, precision, recon, dagger, mode, g, ep, gauge, in, out, aux, out_parity,
                                      reverse, scal, block, st);
    HopArgs a;
    a.dotw = dotw; a.dotw2 = dotw2;
    if (range) a.rg = *range;
    else { a.rg.base = 0; a.rg.count = g.Vh; a.rg.n1 = g.Vh; a.rg.skip = 0; }
    if (a.rg.count <= 0) return cudaSuccess;
    a.reverse = reverse;
    a.gauge = gauge; a.in = in; a.out = out; a.aux = aux;
    a.g = g; a.ep = ep; a.out_parity = out_parity; a.red = red; a.scal = scal;
    a.tile_gy = a.tile_n2h = 0;
    a.general_phases = (g_hop_variant == 7) ? 1 : 0;
    if (block <= 0 || block > LQCD_HOP_MAX_THREADS || (block % 32) != 0) block = LQCD_HOP_MAX_THREADS;
    // variant 6: the 2 x 2 (z, t) tile order, where a z plane is a whole number of groups (modes 0-3, single lattice)
    if (g_hop_variant == 6 && !g.slab && range == nullptr && mode <= 3 && block == 128 && (g.N0h * g.N1) % 32 == 0) {
        a.tile_gy = (g.N0h * g.N1) / 32;
        a.tile_n2h = g.N2 / 2;
    }
    count_launch();
    ProfScope prof(mode == 3 ? 5 : (mode >= 4 ? 1 : mode), st);
    if (precision == 0) {
        return recon == 12 ? launch_tr<double, 12>(dagger, mode, a, block, st)
                           : launch_tr<double, 18>(dagger, mode, a, block, st);
    }
    return launch_hopping_float(recon, dagger, mode, &a, block, st);
}
#endif  // LQCD_HOP_FLOAT_PART

}  // namespace lqcd
