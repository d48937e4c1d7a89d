// lqcd_internal.h -- shared declarations of the CUDA path (not part of the ABI).
//
// Internal field layout (opaque to callers):
//   Vh = V/2 sites per parity, e = x0/2 + N0h (x1 + N1 (x2 + N2 x3)), N0h = N0/2.
//   Sites are grouped in 32s (one warp): G = ceil(Vh/32) groups, site e = (group g = e >> 5,
//   lane l = e & 31).  Inside a group the component index comes before the lane:
//   double spinor : double2 s[G][12][32]          component c = 3 alpha + a
//   float  spinor : float4  s[G][6][32]           element k holds components 2k, 2k+1
//   double gauge  : double2 g[2][4][G][9 or 6][32]  [parity of origin][mu][group][row-major entry][lane]
//   float  gauge 12: float4 g[2][4][G][3][32]
//   float  gauge 18: per (parity, mu, group) 576 floats: float4 planes 0..3 [32], then a float2 plane [32]
// A warp still touches 512 (double) contiguous, 512-byte aligned bytes per component -- 128-bit
// vectorised, fully coalesced, the same property the paper found for a 16-byte base type
// -- but the distance between the components of one site is now a compile-time
// constant (512 B), so the 12 + 9 loads of a hop take their offsets as instruction immediates
// from ONE computed address instead of one 64-bit address computation each (a plane-major
// [component][Vh] layout costs ~3.7 integer instructions per load).
// Pad sites (e >= Vh in the last group, only when Vh is not a multiple of 32) hold zeros in
// every spinor field the library writes.  The gauge field is split by the parity of the
// link's origin.
#pragma once

#include <cuda_runtime.h>
#include <stddef.h>

namespace lqcd {

// Division of a site index by a lattice extent without the ~20-instruction
// runtime integer division: for 2 <= d < 2^31, l = ceil(log2 d), mul = ceil(2^(31+l) / d) (< 2^32),
//   n / d = umulhi(n, mul) >> (l - 1)   exactly for every 0 <= n < 2^31
// (the rounding error n e / (d 2^(31+l)), e < d, is below 2^-l <= 1/d).  d = 1 is passed through.
struct FastDiv {
    unsigned d, mul, sh;
};
inline FastDiv make_fastdiv(unsigned d) {
    FastDiv f;
    f.d = d; f.mul = 0; f.sh = 0;
    if (d < 2) return f;
    unsigned l = 0;
    while ((1ull << l) < d) ++l;
    f.mul = (unsigned)(((1ull << (31 + l)) + d - 1) / d);
    f.sh = l - 1;
    return f;
}
#ifdef __CUDACC__
__device__ __forceinline__ int fd_div(int n, const FastDiv& f) {
    return f.d == 1 ? n : (int)(__umulhi((unsigned)n, f.mul) >> f.sh);
}
#endif

struct Geometry {
    int N0h, N1, N2, N3;  // N0h = N_x / 2
    int Vh;               // sites per parity
    int G;                // groups of 32 sites per parity = ceil(Vh / 32)
    FastDiv d0h, d1, d2;  // division by N0h, N1, N2
    double ph_re[4], ph_im[4];
    int real_ph;          // every phase is exactly +1 or -1 (periodic / antiperiodic): the hopping kernel's REALPH build
    // Slab mode (lqcd_slab_init): two ghost time slices sit behind the G groups of a field, the
    // forward ghost (slice t = N3 of the next rank) at site index Vh + s = e + s3 for a site of the
    // last slice, the backward ghost (slice t = -1 of the previous rank) at Vh + s3 + s (s = index
    // inside a slice, s3 = sites per slice and parity); the time boundary phase applies only on the
    // rank that owns the global boundary (tph_f on the last rank, tph_b on the first).
    int slab;             // 1 after lqcd_slab_init
    int tph_f, tph_b;
    int Gg;               // groups per (parity, mu) array of the gauge field: G, or G + ghost groups
};

// Index of the block that holds the links (parity of origin, mu) of group grp, in blocks of one group of links:
// g[parity][mu][group], one array per direction and parity.  (The other order, g[parity][group][mu] -- the four forward
// links of a group as one contiguous 18 KB block, four link streams per launch instead of eight -- was measured at
// 32^3 x 64: hopping double/18 255.9 against 250.5-251.3 us, everything else within 1%; not kept.)
#ifdef __CUDACC__
__host__ __device__
#endif
inline size_t gauge_block(int par, int mu, int G, int grp) { return (size_t)(par * 4 + mu) * G + grp; }

// Which output sites a hopping launch covers: site i of the launch is e = base + i (+ skip if
// i >= n1).  All sites: base 0, n1 = count = Vh.  Slab mode splits a launch into the interior
// (no ghost needed: overlaps the halo exchange) and the two boundary time slices.
struct SiteRange {
    int base, count, n1, skip;
};

#ifdef __CUDACC__
// a1: eo index e -> (x0h, x1, x2, x3), e = x0h + N0h (x1 + N1 (x2 + N2 x3))
__device__ __forceinline__ void site_coords(const Geometry& g, int e, int& x0h, int& x1, int& x2, int& x3) {
    int q = fd_div(e, g.d0h);
    x0h = e - q * g.N0h;
    int t = q;
    q = fd_div(t, g.d1);
    x1 = t - q * g.N1;
    t = q;
    x3 = fd_div(t, g.d2);
    x2 = t - x3 * g.N2;
}
#endif

// Coefficients of the fused epilogue, per chirality (u: alpha = 0,1; d: alpha = 2,3):
//   out = c_chi * (bracket + d_chi * aux)     bracket = the sum over 8 hops of eq. 6;
// the aux term (MODE >= 1) is what the accumulator is initialised with.
struct Epilogue {
    double cu_re, cu_im, cd_re, cd_im;
    double du_re, du_im, dd_re, dd_im;
    double su_re, su_im, sd_re, sd_im;   // 1 / c_chi (used by hopping MODE 3 only)
};

// Device scalars of the CG recurrence.
struct CgScalars {
    double rho;        // |r|^2
    double pAp;        // <p, A p> = |Mhat p|^2
    double beta;
    double alpha;      // rho / pAp of the current iteration (written by finalize(FIN_PAP))
    double inv_alpha;  // pAp / rho
    double bb;         // |b|^2
    double tol2bb;     // tol^2 |b|^2
    double resid_true; // |b - A x|^2
    int iters;
    int done;          // 1 once converged / broken down: later kernels are no-ops
    int status;        // LQCD_OK / LQCD_NOT_CONVERGED / LQCD_BREAKDOWN
    int upd;           // 1 if this iteration updated r, i.e. cg_update_xp has an x-update to apply
};

// Device scalars of BiCGStab on Mhat: the CG block carries what the shared plumbing reads
// (done, status, iters, bb, tol2bb, rho = |r|^2, resid_true); the complex recurrence scalars follow.
struct BiScalars {
    CgScalars cg;
    double rho_re, rho_im;      // <rhat, r>
    double alpha_re, alpha_im;
    double omega_re, omega_im;
    double beta_re, beta_im;
    double sigma_re, sigma_im;  // <rhat, v> of the current iteration (kept for rho' = (rho - alpha sigma) - omega <rhat, t>)
    int pend;                   // rho' or omega unusable: a breakdown unless this iteration's |r| already meets the tolerance
};

struct Reduction {
    double* partials;       // one per warp (hopping) or per block (vector kernels)
};

enum { FIN_NONE = 0, FIN_PAP = 1, FIN_BB = 2, FIN_RHO = 3, FIN_TRUE = 4 };
enum { FIN_BI_INIT = 0, FIN_BI_SIGMA = 1, FIN_BI_OMEGA = 2, FIN_BI_R = 3,
       // the same two steps fed by the partial sets of a hopping MODE 4 launch: (|out|^2, Re <w,out>, Im <w,out>)
       FIN_BI_SIGMA_HOP = 4,    // w = rhat, out = v: sigma = <rhat, v>
       FIN_BI_OMEGA_HOP = 5,    // w = s, out = t: <t, s> = conj <s, t>, |t|^2
       // the merged form (one pass for x, r and p): hopping MODE 5 partials (|t|^2, <s,t>, <rhat,t>) give omega AND
       // rho' = <rhat, r'> = <rhat, s> - omega <rhat, t>, <rhat, s> = rho - alpha sigma, hence beta before r' exists;
       FIN_BI_OMEGA_BETA = 6,
       FIN_BI_R2 = 7 };         // |r'|^2 of the merged pass: iteration count, convergence, deferred breakdown

// Thread-block size of the hopping kernel: LQCD_HOP_MAX_THREADS is its __launch_bounds__ limit,
// LQCD_DEFAULT_BLOCK what lqcd_init selects (lqcd_set_block_size overrides, up to the limit).
#ifndef LQCD_HOP_MAX_THREADS
#define LQCD_HOP_MAX_THREADS 128
#endif
#ifndef LQCD_DEFAULT_BLOCK
#define LQCD_DEFAULT_BLOCK LQCD_HOP_MAX_THREADS
#endif
// "Snake order": consecutive kernels of a chain traverse the sites in opposite directions
// (reverse = 0, 1, 0, 1, ...).  A field is 201 MB at 32^3 x 64 and L2 holds ~126 MB, so the
// part of its output a kernel wrote last is still in L2 when the next kernel starts; starting
// the next kernel at that end turns part of its compulsory DRAM reads into L2 hits.
// hopping.cu
// mode 0: out = c * bracket;  mode 1: out = c * (bracket + d * aux);  mode 2: mode 1 + |out|^2 partials;
// mode 3 (dagger = 1 only): out -= alpha * c * (bracket + d * aux) in place, alpha = scal->rho / scal->pAp, + |out|^2 partials
// mode 4 (dagger = 0, single lattice only): mode 2 + the partials of <dotw, out>; partial set k of warp w at
//         partials[k G + w]: k = 0 |out|^2, k = 1 Re <dotw, out>, k = 2 Im <dotw, out>
// mode 5: mode 4 + k = 3, 4: Re, Im <dotw2, out>
cudaError_t launch_hopping(int precision, int recon, int dagger, int mode, const Geometry& g,
                           const Epilogue& ep, const void* gauge, const void* in, void* out,
                           const void* aux, int out_parity, int reverse, Reduction red,
                           CgScalars* scal, int block, cudaStream_t st, const SiteRange* range = nullptr,
                           const void* dotw = nullptr, const void* dotw2 = nullptr);

// hopping_staged.cu: staged variants of the kernel (lqcd_set_hop_variant); they cover modes 0 and 1 on a single lattice
void set_hopping_variant(int variant);
int hopping_variant();
bool hopping_variant_covers(int variant, int mode, const Geometry& g, const SiteRange* range);
cudaError_t launch_hopping_variant(int variant, int precision, int recon, int dagger, int mode, const Geometry& g,
                                   const Epilogue& ep, const void* gauge, const void* in, void* out, const void* aux,
                                   int out_parity, int reverse, CgScalars* scal, int block, cudaStream_t st);

// vector_ops.cu  (n = number of reals in a half-spinor field incl. padding = 24 * 32 * G)
cudaError_t launch_cg_init(int precision, size_t n, const void* b, void* x, void* r, void* p,
                           double tol, Reduction red, CgScalars* scal, cudaStream_t st, double* sum_io = nullptr);
cudaError_t launch_cg_update_xp(int precision, size_t n, void* x, void* p, const void* r, int reverse,
                                CgScalars* scal, cudaStream_t st);
cudaError_t launch_true_resid(int precision, size_t n, const void* b, const void* ax, Reduction red,
                              CgScalars* scal, cudaStream_t st, double* sum_io = nullptr);
// out = a_chi * in, a_chi = (ur, ui) on the upper and (dr, di) on the lower chirality
cudaError_t launch_diag_scale(int precision, size_t n, const void* in, void* out, double ur, double ui,
                              double dr, double di, cudaStream_t st);
// mixed-precision solver helpers (double layout double2[12][Vh] <-> float layout float4[6][Vh])
cudaError_t launch_convert_d2f(size_t n, const void* src_d, void* dst_f, double scale, cudaStream_t st);
cudaError_t launch_axpy_f2d(size_t n, double a, const void* x_f, void* y_d, cudaStream_t st);  // y += a x
cudaError_t launch_residual(size_t n, const void* b, const void* ax, void* r, Reduction red,
                            CgScalars* scal, cudaStream_t st);  // r = b - ax (double), |r|^2 -> resid_true
// sums red.partials[0..n_partials) in a fixed order and applies the FIN_* action to *scal
cudaError_t launch_finalize(int fin, Reduction red, int n_partials, double tol, CgScalars* scal,
                            cudaStream_t st, double* sum_io = nullptr, int apply = 0);
// BiCGStab vector kernels (vector_ops.cu); partial sums use up to 3 * vector_grid(n) doubles
cudaError_t launch_bicg_init(int precision, size_t n, const void* b, void* x, void* r, void* p, double tol,
                             Reduction red, BiScalars* bs, cudaStream_t st);
cudaError_t launch_bicg_sigma(int precision, size_t n, const void* rhat, const void* v, int reverse,
                              Reduction red, BiScalars* bs, cudaStream_t st);
cudaError_t launch_bicg_s(int precision, size_t n, const void* r, const void* v, void* s, int reverse,
                          BiScalars* bs, cudaStream_t st);
cudaError_t launch_bicg_omega(int precision, size_t n, const void* t, const void* s, int reverse,
                              Reduction red, BiScalars* bs, cudaStream_t st);
cudaError_t launch_bicg_xr(int precision, size_t n, void* x, const void* p, const void* s, const void* t,
                           const void* rhat, void* r, int reverse, Reduction red, BiScalars* bs,
                           cudaStream_t st);
cudaError_t launch_bicg_xrp(int precision, size_t n, void* x, void* p, const void* s, const void* t, const void* v,
                            void* r, int reverse, Reduction red, BiScalars* bs, cudaStream_t st);
cudaError_t launch_bicg_finalize(int fin, Reduction red, int n_partials, BiScalars* bs, cudaStream_t st);
cudaError_t launch_bicg_p(int precision, size_t n, void* p, const void* r, const void* v, int reverse,
                          BiScalars* bs, cudaStream_t st);
int vector_grid(size_t n);
int hopping_partials(int Vh, int block);

// pack.cu
cudaError_t launch_pack_gauge(int precision, int recon, const Geometry& g, const void* canon,
                              void* internal, cudaStream_t st);
cudaError_t launch_pack_spinor(int precision, const Geometry& g, const void* canon, void* internal,
                               int parity, cudaStream_t st);
cudaError_t launch_unpack_spinor(int precision, const Geometry& g, const void* internal, void* canon,
                                 int parity, cudaStream_t st);

cudaError_t launch_unpack_gauge(int precision, int recon, const Geometry& g, const void* internal, void* canon,
                                cudaStream_t st);

// gauge_update.cu: one sub-sweep (all links U_mu(x), parity(x) = parity) of the heatbath (mode 0)
// or overrelaxation (mode 1) update, in place; the average plaquette as per-warp partial sums of
// Re tr P over the 6 V plaquettes (plaquette_partials(Vh) of them).
cudaError_t launch_gauge_update(int precision, int recon, int mode, const Geometry& g, void* gauge, int mu,
                                int parity, double beta, unsigned long long seed, unsigned long long tag,
                                cudaStream_t st);
cudaError_t launch_plaquette(int precision, int recon, const Geometry& g, const void* gauge, Reduction red,
                             cudaStream_t st);
int plaquette_partials(int Vh);
// the same with the partials in a file-scope device array (at most LQCD_PLAQUETTE_STATIC_MAX_PARTIALS of them: the caller
// checks) and the average written to out_dev; allocates nothing
cudaError_t launch_plaquette_static(int precision, int recon, const Geometry& g, const void* gauge, double* out_dev,
                                    cudaStream_t st);

// force.cu: F^a_mu(x) for every link from full-lattice X, Y given as half fields (the force is
// linear in kappa, so a common sign of the odd halves is passed as the sign of kappa).
// force: double2 f[2][4][G][4][32], element j of a link = (F^{2j+1}, F^{2j+2}); always double.
cudaError_t launch_fermion_force(int precision, int recon, const Geometry& g, const void* gauge,
                                 const void* x_even, const void* x_odd, const void* y_even,
                                 const void* y_odd, void* force, double kappa, cudaStream_t st);
cudaError_t launch_unpack_force(const Geometry& g, const void* force, void* canon, cudaStream_t st);

void count_launch(int n = 1);

// stream_probe.cu: the paper's buffer-copy micro-benchmark (Fig. 5) as the library's HBM probe
constexpr int kStreamProbeBlocks = 148 * 8;   // 8 CTAs of 256 threads per SM of a B200: every thread slot taken
cudaError_t launch_stream_probe(int elem, int mode, const void* src, void* dst, size_t bytes, cudaStream_t st);
cudaError_t launch_dfma_probe(double a, double b, int iters, double* out, cudaStream_t st);

// api.cu: optional per-launch event timing (lqcd_profile)
void prof_begin(int category, cudaStream_t st);
void prof_end(cudaStream_t st);
struct ProfScope {
    cudaStream_t st;
    ProfScope(int category, cudaStream_t s) : st(s) { prof_begin(category, s); }
    ~ProfScope() { prof_end(st); }
};

// Programmatic dependent launch (sm_90+) for the kernels of the CG iteration: launched with launch_chained, a kernel may
// be scheduled while the grid before it in the stream drains -- its CTAs take the SM slots the last wave of that grid
// frees, run up to chain_prologue() and wait there until the whole of that grid has completed and its writes are
// visible.  What it hides is the launch and ramp-up between two dependent kernels (7 boundaries per CG iteration), which
// is most of a CG iteration's fixed cost on small lattices.  chain_prologue() is the first
// statement of every kernel that is ever launched this way: launch_dependents lets the NEXT chained kernel be scheduled
// once every CTA of this grid has started; wait returns at once when the kernel was launched the ordinary way.
#ifdef __CUDACC__
__device__ __forceinline__ void chain_prologue() {
    asm volatile("griddepcontrol.launch_dependents;\n" ::: "memory");
    asm volatile("griddepcontrol.wait;\n" ::: "memory");
}
template <typename... KArgs, typename... Args>
inline cudaError_t launch_chained(bool chained, void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                                  Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = chained ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}
#endif
bool chained_launches(cudaStream_t st);    // api.cu: direct launches only; LQCD_PDL=0 in the environment turns them off

// Global sums are two-stage and fixed-order (deterministic for a given launch configuration):
// the producing kernel writes one partial per warp (hopping) or per block (vector kernels)
// with plain stores -- no fence, no atomic, no last-block election, which cost the hopping
// kernel 12% when every block had to drain its stores before signalling -- and a one-block
// finalisation kernel (vector_ops.cu: launch_finalize) adds them in index order and applies
// the scalar recurrence (FIN_*) on the device.
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

}  // namespace lqcd
