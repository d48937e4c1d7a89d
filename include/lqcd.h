/* lqcd.h -- C ABI of liblqcd.so: the even-odd preconditioned twisted-mass Wilson
 * fermion matrix of arxiv 1209.5942 and CG on Mhat^dag Mhat, on one NVIDIA B200.
 *
 * What is computed (eq. 6; readings G1-G11 in DESIGN.md):
 *
 *   (M psi)(x) = (1 + 2 i kappa mu gamma5) psi(x)
 *                - kappa sum_{mu=0..3} [ eta+_mu(x) (1 - gamma_mu) U_mu(x)        psi(x + mu)
 *                                      + eta-_mu(x) (1 + gamma_mu) U_mu(x - mu)^dag psi(x - mu) ]
 *
 * with coordinates mod N_mu, eta+_mu(x) = bc_phase_mu on the hop that wraps
 * (x_mu = N_mu - 1), eta-_mu(x) = conj(bc_phase_mu) at x_mu = 0, else 1.
 * mu = 0..3 = x,y,z,t.  Sites are split by parity p(x) = (x0+x1+x2+x3) mod 2:
 *   M = [[M_ee, D_eo], [D_oe, M_oo]],  M_ee = M_oo = 1 + 2 i kappa mu gamma5,
 *   Mhat = M_ee - D_eo M_oo^{-1} D_oe   on even sites (reading G3).
 * gamma basis (reading G4; chiral, gamma5 = diag(1,1,-1,-1)), rows top to bottom:
 *   gamma_x: (0,0,0,-i) (0,0,-i,0) (0,i,0,0) (i,0,0,0)
 *   gamma_y: (0,0,0,-1) (0,0,1,0)  (0,1,0,0) (-1,0,0,0)
 *   gamma_z: (0,0,-i,0) (0,0,0,i)  (i,0,0,0) (0,-i,0,0)
 *   gamma_t: (0,0,1,0)  (0,0,0,1)  (1,0,0,0) (0,1,0,0)
 *
 * Canonical (interchange) layout, always complex double, row-major, (re,im):
 *   gauge        U[lex(x)][mu][a][b]      144 B per link, 576 B per site
 *   half spinor  psi_p[e][alpha][a]       192 B per site, e = lex(x)/2 over
 *                                         the sites of parity p, lex(x) = x0 + N0 (x1 + N1 (x2 + N2 x3))
 * Internal layout: opaque structure-of-arrays on 128-bit elements (the thing
 * being tuned); sizes from lqcd_gauge_bytes() / lqcd_spinor_bytes(); convert
 * with lqcd_pack_* / lqcd_unpack_spinor.  In single precision the internal
 * fields are float (pack rounds to nearest, unpack widens).
 *
 * Pointers: every `*_dev` / gauge / in / out / b / x argument is a DEVICE
 * pointer, 16-byte aligned, allocated and freed by the caller; `*_host`
 * arguments (only in the lqcd_*_host calls) are HOST pointers.  The library
 * owns only its context and a lazily allocated CG / staging workspace, released
 * by lqcd_finalize().  `in` and `out` must not alias.  All device calls are
 * asynchronous on the stream given to lqcd_set_stream() (default: stream 0)
 * except lqcd_cg_mdagm, lqcd_cg_finish, lqcd_cg_stats and the *_host calls,
 * which synchronise that stream before returning.
 *
 * Every function returns an int status; no exception crosses the ABI.
 * The library is not thread safe (one context per process).
 */
#ifndef LQCD_H
#define LQCD_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LQCD_OK               0
#define LQCD_NOT_CONVERGED    1   /* cg only: maxit reached, x = last iterate        */
#define LQCD_NOT_INITIALISED (-1)
#define LQCD_BAD_DIMS        (-2) /* an extent is odd or < 2, or |bc_phase| != 1      */
#define LQCD_BAD_ARG         (-3) /* null pointer, parity not 0/1, non-finite scalar */
#define LQCD_CUDA_ERROR      (-4)
#define LQCD_BREAKDOWN       (-5) /* cg: <p, A p> <= 0 or not finite                  */

#define LQCD_DOUBLE 0
#define LQCD_SINGLE 1

/* Text of the last error on this process ("" if none). Never NULL. */
const char* lqcd_last_error(void);

/* Set the lattice extents N_x,N_y,N_z,N_t (all even, >= 2) and the boundary
 * phases e^{i pi theta_mu} as (re,im) pairs, mu = x,y,z,t (reading G5; the
 * paper never states its boundary conditions).  Resets format to double/18,
 * stream to 0.  No device work. */
int lqcd_init(const int dims[4], const double bc_phase[8]);
int lqcd_finalize(void);

/* cuda_stream is a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream). */
int lqcd_set_stream(void* cuda_stream);

/* precision: LQCD_DOUBLE or LQCD_SINGLE; recon: 18 (full link) or 12 (two rows
 * stored, third = conj(row0 x row1), reading G9).  Fields packed
 * under one format are only valid under that format. */
int lqcd_set_format(int precision, int recon);

size_t lqcd_gauge_bytes(void);   /* bytes of one internal gauge field (both parities, 4 mu) */
size_t lqcd_spinor_bytes(void);  /* bytes of one internal half-spinor field                 */

/* canonical (device) -> internal (device) and back; parity = parity of the sites held. */
int lqcd_pack_gauge(const void* canon_dev, void* internal_dev);
int lqcd_pack_spinor(const void* canon_dev, void* internal_dev, int parity);
int lqcd_unpack_spinor(const void* internal_dev, void* canon_dev, int parity);

/* Hopping block of eq. 6, including the factor -kappa:
 *   out_p = D_{p,1-p} in_{1-p},   parity = p = parity of the OUTPUT sites
 * (parity 0: out_e = D_eo in_o).  Internal layouts. */
int lqcd_dslash_eo(const void* gauge, const void* in, void* out, int parity, double kappa);

/* Even-odd preconditioned operator on even half fields (internal layout):
 *   dagger = 0: out = Mhat(mu) in;   dagger = 1: out = Mhat(mu)^dag in  (= gamma5 Mhat(-mu) gamma5 in).
 * Two hopping launches; the diagonal terms are fused into their epilogues.
 * Uses one half-spinor of library workspace. */
int lqcd_mtm(const void* gauge, const void* in, void* out, double kappa, double mu, int dagger);

/* The full operator of eq. 6 on both parities (internal layouts; two hopping launches with the
 * diagonal term in their epilogues):
 *   out_e = M_ee in_e + D_eo in_o,   out_o = M_oo in_o + D_oe in_e.   No buffer may alias another. */
int lqcd_mtm_full(const void* gauge, const void* in_even, const void* in_odd, void* out_even,
                  void* out_odd, double kappa, double mu);

/* Solve M psi = eta on the WHOLE lattice (eq. 8) through the even-odd system:
 *   rhs_e = eta_e - D_eo M_oo^{-1} eta_o;   CG on Mhat^dag Mhat psi_e = Mhat^dag rhs_e;
 *   psi_o = M_oo^{-1} (eta_o - D_oe psi_e).
 * tol is the CG tolerance on the normal equations (|Mhat^dag (rhs - Mhat psi_e)| <= tol |Mhat^dag rhs|);
 * the residual of the full system is larger by at most cond(Mhat).  psi_even / psi_odd are used as
 * scratch before they receive the solution and must not alias eta_*.  Returns the CG status;
 * lqcd_cg_stats() gives its iterations and residuals.  Synchronous. */
int lqcd_solve_full(const void* gauge, const void* eta_even, const void* eta_odd, void* psi_even,
                    void* psi_odd, double kappa, double mu, double tol, int maxit);

/* Solve Mhat^dag Mhat x = b on even sites by CG (reading G10):
 * x0 = 0 (input contents of x ignored), stop when |r| <= tol |b| (recursive
 * residual) or after maxit iterations.  Returns LQCD_OK, LQCD_NOT_CONVERGED or
 * LQCD_BREAKDOWN.  b, x in internal layout. */
int lqcd_cg_mdagm(const void* gauge, const void* b, void* x, double kappa, double mu,
                  double tol, int maxit);

/* The same solve in three steps (what lqcd_cg_mdagm does internally; bench.py
 * times lqcd_cg_iterate alone):
 *   lqcd_cg_setup    r = p = b, x = 0, rho = |b|^2                       (async)
 *   lqcd_cg_iterate  enqueue up to n iterations; iterations after convergence
 *                    are no-ops on the device                            (async)
 *   lqcd_cg_finish   synchronise, compute the true residual |b - A x|/|b|;
 *                    returns the solve status.
 * On a stream that can be captured (any but the legacy default stream) the solvers enqueue four
 * iterations at a time as a CUDA graph captured on first use and kept while gauge, x, format, block
 * size, kappa and mu stay the same (bit-identical to direct launches, ~13 us less device time per
 * iteration between the kernels); LQCD_CG_GRAPH=0 in the environment turns it off.  Launches that go straight into
 * a stream (the legacy default stream, the host-buffer calls; not while lqcd_profile records) chain the
 * hopping, finalisation and x/p kernels by programmatic dependent launch instead (sm_90+: a kernel is scheduled
 * while the grid before it drains and waits for it at its first instruction): 31 against 44 us per CG iteration at
 * 8^3 x 16, 100 against 113 at 16^3 x 32, 1298 against 1307 at 32^3 x 64, results bit-identical; LQCD_PDL=0 turns it
 * off. */
int lqcd_cg_setup(const void* gauge, const void* b, void* x, double kappa, double mu, double tol);
int lqcd_cg_iterate(int n);
int lqcd_cg_finish(void);

/* Solve Mhat x = b on even sites by BiCGStab, the second solver the paper names (
 * SURVEY.md section 8(f) row 2; reading G15 of DESIGN.md): shadow residual rhat = b, x0 = 0, one
 * iteration = two applications of Mhat; stops when |r| <= tol |b| (recursive residual) or after
 * maxit iterations.  Returns LQCD_OK, LQCD_NOT_CONVERGED or LQCD_BREAKDOWN (<rhat,v>, <rhat,r> or
 * omega zero or not finite); lqcd_cg_stats() gives iterations and the residuals of Mhat x = b.
 * <rhat,v>, <t,s>, |t|^2 and <rhat,t> are reduced inside the hopping launches that produce v and t, and
 * <rhat,r'> is taken as (rho - alpha <rhat,v>) - omega <rhat,t> (the same number to rounding), so that x, r
 * and p are updated in one pass; the four-iteration chunk goes through the graph cache described above.
 * b, x in internal layout; b is read throughout the solve.  Synchronous. */
int lqcd_bicgstab_mhat(const void* gauge, const void* b, void* x, double kappa, double mu, double tol,
                       int maxit);

/* Fermion force of the HMC (eq. 9-10: F = -dS/dU, a real 8-vector per link,
 * PAPER.md:106, :255; reading G16 of DESIGN.md).  Components are
 * taken along T^a = lambda^a / 2 (Gell-Mann matrices in the standard order) with the link varied
 * from the left, U_mu(x) -> exp(i w T^a) U_mu(x), F^a_mu(x) = -dS/dw at w = 0.
 *
 * lqcd_fermion_force: the outer-product kernel for two spinor fields X, Y on the WHOLE lattice,
 * given as even and odd half fields (internal layout, current format):
 *   F^a_mu(x) = 2 Re d/dw [Y^dag M(w) X] = 2 kappa Im [ Y(x)^dag T^a a(x) - b(x)^dag T^a X(x) ],
 *   a(x) = eta+_mu(x) (1 - gamma_mu) U_mu(x) X(x+mu),  b(x) = eta+_mu(x) (1 + gamma_mu) U_mu(x) Y(x+mu).
 * force: lqcd_force_bytes() bytes, internal layout, always double; lqcd_unpack_force converts to
 * the canonical double F[lex(x)][mu][8] (64 B per link, 256 B per site: Table 3).  Asynchronous.
 *
 * lqcd_force_tm: the whole force of S = phi^dag (Mhat^dag Mhat)^-1 phi, phi on even sites:
 * X_e = (Mhat^dag Mhat)^-1 phi by CG (tol, maxit as in lqcd_cg_mdagm), Y_e = Mhat X_e,
 * X_o = -M_oo^-1 D_oe X_e, Y_o = -(M_oo^-1)^dag (D_eo)^dag Y_e, then the kernel above.
 * Returns the CG status; synchronous; uses six half spinors of library workspace. */
size_t lqcd_force_bytes(void);
int lqcd_unpack_force(const void* force_internal_dev, void* canon_dev);
int lqcd_fermion_force(const void* gauge, const void* x_even, const void* x_odd, const void* y_even,
                       const void* y_odd, void* force, double kappa);
int lqcd_force_tm(const void* gauge, const void* phi, void* force, double kappa, double mu, double tol,
                  int maxit);

/* Pure-gauge heatbath and overrelaxation, the paper's second workload (Fig. 2;
 * Table 2; readings G17-G21 of DESIGN.md), for the
 * Wilson plaquette action S = beta sum_{x, mu<nu} (1 - Re tr P_mu_nu(x) / 3) (eq. 5 with c_1 = 0) on a
 * periodic gauge field.  Per link, with A the sum of its 6 staples and for the SU(2)
 * subgroups (0,1), (1,2), (0,2) in turn:  W = L A;  w = project(W);  v = update(w);  L = extend(v) L,
 *   LQCD_HEATBATH : v w = g drawn with density sqrt(1 - g0^2) exp((2 beta k / 3) g0) (Kennedy-Pendleton,
 *                   at most 32 attempts, else the subgroup is left unchanged), k^2 = det-like norm of w;
 *   LQCD_OVERRELAX: v w = w^dag (the action is unchanged; beta, seed, tag are ignored).
 * Random numbers: the counter-based generator of the input recipe, uniform(seed, stream = tag, counter),
 * counter = (((4 lex(x) + mu) 3 + subgroup) 33 + attempt) 4 + j; tag < 2^24 must differ from sweep to sweep.
 *
 * lqcd_gauge_update: one sub-sweep, in place: every link U_mu(x) with parity(x) = parity (these links
 *   are mutually independent).  gauge: internal layout of the current format.  Asynchronous.
 * lqcd_gauge_sweep : the 8 sub-sweeps mu = 0..3, parity 0 then 1.  Asynchronous.
 * lqcd_plaquette   : average of Re tr P / 3 over the 6 V plaquettes, written to a HOST double; synchronous.
 * lqcd_unpack_gauge: internal -> canonical U[lex(x)][mu][a][b] (complex double; 12-real storage
 *   rebuilds the third row).  Asynchronous.
 * LQCD_HEATBATH_WS=1 in the environment (read once) runs the heatbath with a warp-specialised kernel -- a second
 * warpgroup per CTA computes the field-independent part of the Kennedy-Pendleton draws -- with the same results;
 * it is slower than the default (profiles/r02_heatbath.md) and kept as the record of that experiment. */
#define LQCD_HEATBATH  0
#define LQCD_OVERRELAX 1
int lqcd_gauge_update(void* gauge, int mu, int parity, int mode, double beta, unsigned long long seed,
                      unsigned long long tag);
int lqcd_gauge_sweep(void* gauge, int mode, double beta, unsigned long long seed, unsigned long long tag);
int lqcd_plaquette(const void* gauge, double* plaquette_host);
/* lqcd_plaquette_static: the same average plaquette for callers that may not allocate (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc).  The call makes no cudaMalloc, cudaFree or allocating
 * library call: the per-warp partial sums, which lqcd_plaquette keeps in a buffer of the context, go to a file-scope
 * device array of LQCD_PLAQUETTE_STATIC_MAX_PARTIALS doubles (512 KiB, held by every GPU that loads the library until
 * exit), and the result goes to plaquette_dev, ONE double in DEVICE memory the caller owns.  Asynchronous on the
 * lqcd_set_stream stream; two launches.  Needs 8 * ceil(V/256) <= LQCD_PLAQUETTE_STATIC_MAX_PARTIALS, i.e. lattices
 * up to V = 2^21 sites (32^3 x 64); larger ones return LQCD_BAD_ARG with a message and launch nothing.  All calls share
 * the array, which keeps the last call's contents (nothing in it has to start at zero: every partial a call reads it
 * has written first); calls that overlap on the GPU -- two streams, two host threads -- race on it, so order them.
 * The first call on a device looks the array's device address up (no allocation); make it outside a capture.
 * Same gauge formats as lqcd_plaquette; not available after lqcd_slab_init.  The value agrees with lqcd_plaquette to
 * summation order (a few ulp). */
#define LQCD_PLAQUETTE_STATIC_MAX_PARTIALS 65536
int lqcd_plaquette_static(const void* gauge, double* plaquette_dev);
int lqcd_unpack_gauge(const void* internal_dev, void* canon_dev);

/* Mixed-precision solve of the same system (the paper's planned next step, PAPER.md:352;
 * SURVEY.md section 8(f) row 1): defect correction with the outer residual in double and the
 * inner CG in single precision,
 *   x = 0, r = b;  repeat { solve A e = r/|r| in single to inner_tol;  x += |r| e;  r = b - A x }
 * until |r| <= tol |b| (a TRUE residual, evaluated in double) or maxit inner iterations in total.
 * gauge_double / gauge_single: the same field packed under (LQCD_DOUBLE, recon_double) and
 * (LQCD_SINGLE, recon_single); b, x: double internal layout.  inner_tol in [0,1): 0 (recommended)
 * asks each inner solve for half the reduction still missing, floored at 1e-6 (what single
 * precision delivers).  Independent of lqcd_set_format.  Synchronous. */
int lqcd_cg_mdagm_mixed(const void* gauge_double, int recon_double, const void* gauge_single,
                        int recon_single, const void* b, void* x, double kappa, double mu, double tol,
                        int maxit, double inner_tol);
/* Outer (double-precision) corrections of the last lqcd_cg_mdagm_mixed call; 0 otherwise. */
int lqcd_cg_outer_iterations(void);

/* Results of the last solve: iterations done, recursive and true relative residual.
 * Any pointer may be NULL. */
int lqcd_cg_stats(int* iters, double* rel_resid_recursive, double* rel_resid_true);

/* Host-buffer entry points (canonical layout, HOST pointers; pinned memory is
 * faster but not required).  Each uploads its inputs, packs, computes, unpacks
 * and downloads the result, synchronously.  Device staging is library workspace. */
int lqcd_mtm_host(const void* gauge_canon_host, const void* in_canon_host, void* out_canon_host,
                  double kappa, double mu, int dagger);
int lqcd_cg_mdagm_host(const void* gauge_canon_host, const void* b_canon_host, void* x_canon_host,
                       double kappa, double mu, double tol, int maxit);

/* ---------------------------------------------------------------------------------------------
 * Slab decomposition of the time direction over several ranks, one GPU each (the paper lists
 * multi-GPU as future work).
 * Rank r of R owns the time slices [r N_t/R, (r+1) N_t/R) (N_t/R even, N_x N_y N_z / 2 a multiple
 * of 32) as a local lattice in the usual layouts.  Behind the sites of every half-spinor field sit
 * two ghost time slices: slice t = N_t/R of rank r+1 and slice t = -1 of rank r-1 (cyclically);
 * behind the time-like links the links U_t(x - t) of slice t = -1.  All are contiguous blocks of
 * the internal layout at the byte offsets the *_halo calls return, so a halo exchange is two
 * plain block copies per field (NCCL send/recv, peer-to-peer copies, or stores into peer memory).
 * The boundary phase of the time direction is applied on the ranks that own the global boundary.
 * The library computes and never communicates: the caller fills the ghosts of the field a call
 * reads (stated per call) and all-reduces the two scalars of a CG iteration in place on the
 * device.  Every hopping launch can be split (part = 1: interior time slices, which read no ghost
 * and can overlap the exchange; part = 2: the two boundary slices; part = 0: all sites).
 *
 * lqcd_select_context: up to 8 independent contexts per process (lattice, format, stream,
 * workspace, solver state); every call acts on the selected one.  Lets one process hold several
 * slabs (how the single-GPU tests check the decomposition); the default is context 0.
 * After lqcd_slab_init, lqcd_gauge_bytes / lqcd_spinor_bytes include the ghosts; lqcd_pack_* /
 * lqcd_unpack_* take the rank's LOCAL canonical fields; lqcd_dslash_eo covers all local sites
 * (ghosts of `in` must be current); the single-GPU solvers, force and gauge-update calls return
 * LQCD_BAD_ARG. */
int lqcd_select_context(int id);
int lqcd_slab_init(const int dims_global[4], const double bc_phase[8], int rank, int nranks);
/* Byte offsets inside an internal half-spinor field: send_lo / send_hi = this rank's first / last
 * time slice (go to the forward ghost of rank-1 / the backward ghost of rank+1), ghost_fwd /
 * ghost_bwd = where slice N_t/R of rank+1 / slice -1 of rank-1 are received; bytes per block. */
int lqcd_slab_spinor_halo(size_t* send_lo, size_t* send_hi, size_t* ghost_fwd, size_t* ghost_bwd, size_t* bytes);
/* The same for the time-like links of one origin parity (exchanged once, after lqcd_pack_gauge):
 * send_hi = this rank's last slice (goes to rank+1), ghost_bwd = where rank-1's is received. */
int lqcd_slab_gauge_halo(int parity, size_t* send_hi, size_t* ghost_bwd, size_t* bytes);
/* out_p = D_{p,1-p} in on the sites of `part` (reads the ghosts of `in` unless part = 1). */
int lqcd_slab_dslash(const void* gauge, const void* in, void* out, int parity, double kappa, int part);
/* Mhat / Mhat^dag in its two hopping launches:
 *   stage 1: tmp_odd = M_oo^-1 D_oe in         (ghosts of `in`)
 *   stage 2: out     = M_ee in - D_eo tmp_odd  (ghosts of `tmp_odd`)      even half fields in, out. */
int lqcd_slab_mhat_stage(const void* gauge, const void* in, void* tmp_odd, void* out, double kappa, double mu,
                         int dagger, int stage, int part);
/* CG on Mhat^dag Mhat across the ranks (reading G10), one stage at a time, all asynchronous:
 *   0  r = p = b, x = 0, own |b|^2 -> sum        [all-reduce sum]     1  rho = |b|^2
 *   2  t1 = M_oo^-1 D_oe p        (ghosts of p)   3  t2 = Mhat p, partial |t2|^2 (ghosts of t1)
 *   4  own <p, A p> -> sum        [all-reduce]    5  alpha
 *   6  t1 = (M_oo^-1)^dag (D_eo)^dag t2 (ghosts of t2)   7  r -= alpha Mhat^dag t2, partial |r|^2 (ghosts of t1)
 *   8  own |r|^2 -> sum           [all-reduce]    9  beta, convergence flag, x += alpha p, p = r + beta p
 *   11-14 the four launches of Mhat^dag Mhat x (ghosts of x, t1, t2, t1), 15 own |b - A x|^2 -> sum
 *   [all-reduce], 16 true residual.
 * Stages 2, 3, 6, 7, 11-14 take `part`.  lqcd_slab_cg_halo_field(stage) is the field whose ghosts
 * that stage reads (NULL: none); lqcd_slab_sum_ptr() the device double to all-reduce.  After
 * convergence the stages are no-ops on the device; lqcd_slab_cg_poll synchronises and reports the
 * flag; lqcd_slab_cg_end returns the status and fills lqcd_cg_stats. */
int lqcd_slab_cg_begin(const void* gauge, const void* b, void* x, double kappa, double mu, double tol);
int lqcd_slab_cg_stage(int stage, int part);
void* lqcd_slab_cg_halo_field(int stage);
void* lqcd_slab_sum_ptr(void);
int lqcd_slab_cg_poll(int* done, int* iters);
int lqcd_slab_cg_end(int with_true_resid);

/* The paper's buffer-copy micro-benchmark (Fig. 5: copy bandwidth by element type,
 * the experiment that fixed its structure-of-arrays format on a 16-byte element), kept as the
 * library's own HBM probe; timed by the caller (CUDA events on the library's stream).
 *   elem: LQCD_ELEM_FLOAT (4 B), LQCD_ELEM_DOUBLE (8 B), LQCD_ELEM_VEC16 (16 B = float4 = complex
 *         double; the storage element of every internal field): thread <-> array element;
 *         LQCD_ELEM_SU3_AOS (144 B), LQCD_ELEM_SPINOR_AOS (192 B): thread <-> whole struct, the
 *         array-of-structures access the paper started from; COPY only.
 *   mode: LQCD_STREAM_COPY   dst[i] = src[i]; reads `bytes`, writes `bytes`;
 *         LQCD_STREAM_READ   reads `bytes`; dst receives LQCD_STREAM_PROBE_BLOCKS 8-byte words whose
 *                            XOR is the XOR of all 8-byte words of src;
 *         LQCD_STREAM_MIX71  src = 7 planes of bytes/7 each, dst[i] = XOR over the planes of element i:
 *                            reads `bytes`, writes bytes/7 -- the read : write ratio of the hopping
 *                            term (1344 : 192 B per site).
 * src, dst: DEVICE pointers, 16-byte aligned, not overlapping; `bytes` (of src) a multiple of 16, of
 * the struct size for the AoS elements and of 112 in MIX71, else LQCD_BAD_ARG.  bytes = 0 is a no-op.
 * All arithmetic is bit-wise, so results are exact for any contents.  Asynchronous. */
#define LQCD_ELEM_FLOAT      0
#define LQCD_ELEM_DOUBLE     1
#define LQCD_ELEM_VEC16      2
#define LQCD_ELEM_SU3_AOS    3
#define LQCD_ELEM_SPINOR_AOS 4
#define LQCD_STREAM_COPY  0
#define LQCD_STREAM_READ  1
#define LQCD_STREAM_MIX71 2
#define LQCD_STREAM_PROBE_BLOCKS 1184
int lqcd_stream_probe(int elem, int mode, const void* src_dev, void* dst_dev, size_t bytes);

/* FP64 pipe probe, the secondary bound of the hopping term: LQCD_STREAM_PROBE_BLOCKS
 * CTAs of 256 threads; thread t runs 8 independent chains x <- fma(x, a, b) of `iters` links, chain c
 * starting at t + c, and stores the sum of its 8 results to out_dev[t] (LQCD_STREAM_PROBE_BLOCKS * 256
 * doubles, DEVICE).  16 * iters flop per thread; timed by the caller.  iters < 0, a or b not finite, null
 * pointer: LQCD_BAD_ARG.  Asynchronous. */
int lqcd_fp64_probe(double a, double b, int iters, double* out_dev);

/* Number of kernels this library has launched since lqcd_init (all streams). */
long long lqcd_launch_count(void);

/* Per-launch device timing.  lqcd_profile(1) starts recording a CUDA-event pair around every
 * kernel the library launches on its stream (and discards earlier records); lqcd_profile(0)
 * stops (the records stay); lqcd_profile(2) resumes without discarding or synchronising, so a caller can
 * sample some of its launches (an event pair costs ~2.5 us of device time per launch, 2.6% of a CG
 * iteration at 32^3 x 64 when every launch is recorded).  lqcd_profile_read synchronises the stream and returns the summed duration and the
 * launch count of one category: 0 hopping (plain epilogue), 1 hopping + M_ee*aux epilogue,
 * 2 hopping + M_ee*aux epilogue + fused norm, 3 CG vector kernels, 4 pack/unpack,
 * 5 hopping + M_ee*aux epilogue + fused CG residual update (r -= alpha q, |r|^2),
 * 6 fermion-force kernel, 7 gauge update (heatbath / overrelaxation sub-sweep), 8 plaquette. */
int lqcd_profile(int enable);
int lqcd_profile_read(int category, double* total_ms, int* launches);

/* Hopping-kernel thread-block size (tuning knob; 0 restores the default). */
int lqcd_set_block_size(int threads);

/* Which hopping kernel runs the launches with a plain or M_ee*aux epilogue on a single lattice (BASELINE.json
 * north_star: "neighbour spinors staged through shared memory or TMA ... every choice is evidenced by ncu
 * counters"; the counters are in profiles/r02_hopping_staged.md).  Process-wide, not per context.  Same result
 * to rounding order as the default; launches a variant does not cover (fused reductions, slab mode, and for variants
 * 1-5 lattices with a complex boundary phase) use variant 0.
 *   0      the default: one thread per site, every operand through LDG into registers
 *   1..3   "link ring": each thread prefetches the link of hop h + D (D = variant) into its own shared-memory
 *          slot with cp.async while it works on hop h
 *   4, 5   "bulk": lane 0 of every warp fetches the warp's forward links (one contiguous block per direction in the
 *          internal layout) with one cp.async.bulk per direction, completion on the warp's mbarrier; 4 = z and t
 *          links, 5 = all four directions
 *   6      "tile": the default kernel with another order of the sites: the four warps of a CTA take a 2 x 2 block in
 *          (z, t) of one 32-site group in (x, y) instead of four consecutive groups (16 instead of 21 groups of
 *          neighbour spinors per CTA); covers every launch on a single lattice whose z planes hold whole groups
 *   7      "general phases": where every phase of lqcd_init is exactly +-1 the default kernel applies it as the sign
 *          of the accumulation (a multiply-add in place of an add, no branch); variant 7 runs the general kernel
 *          (a complex multiplication behind a branch on every hop that wraps) on such lattices too, for comparison
 * Returns LQCD_BAD_ARG for other values. */
#define LQCD_HOP_VARIANT_MAX 7
int lqcd_set_hop_variant(int variant);

#ifdef __cplusplus
}
#endif
#endif /* LQCD_H */
